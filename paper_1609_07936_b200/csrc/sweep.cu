// sweep.cu — the persistent Monte Carlo sweep kernel.
//
// Mapping: one walker per warp; lane l owns tau-points j = l + 32 i, i < C, whose residual state
// lives in REGISTERS for the whole launch:
//     mt_j  = sum_k a_k exp(-omega_k tau_j)      (model in the pure-exponential basis, M_j = c_j mt_j)
//     G2_j  = 2 Wj (mt_j - fj)                   (Wj = (c_j/sigma_j)^2, fj = F_j/c_j)
// so that for a move (p, s, rho, delta_p, delta_s) (Eq. 17-22):
//     dt_j   = (rho-1) mt_j + delta_p E_pj + delta_s E_sj          E_kj = exp(-omega_k tau_j)
//     dchi2  = sum_j dt_j (Wj dt_j + G2_j)     [= sum_j d_j (d_j + 2 D_j) of SURVEY §8a row A4]
// The kernel rows are never read from a table in the inner loop: both grids are uniform (Eq. 2-3, 7), so
// E_{k,j+32} = E_kj exp(-omega_k 32 dtau), and v_i = delta_p E_p,i + delta_s E_s,i (i = tau-point index of the lane)
// obeys the two-term linear recurrence of its two geometric modes,
//     v_{i+1} = (r_p + r_s) v_i - (r_p r_s) v_{i-1},      r_k = exp(-omega_k 32 dtau),
// started from E0[k][l] (shared memory).  The tau loop costs 5 FP64 instructions per tau-point (DMUL + DFMA for v,
// then the three DFMAs of d, W d + G2, d (W d + G2)): the algorithmic count of SURVEY §8d.
//
// Proposals (Philox4x32-10 keyed by (seed; walker, sweep, move, 0), index draw, rho, Eq. 20-21, -T ln u) do not depend
// on the chain state within a sweep, so they are computed 32 moves at a time, one move per lane, and staged as records
// in shared memory.  Positivity (row A3) is tested for all moves of the batch AT ONCE, one move per lane, against the
// current spectrum: a ballot gives the mask of feasible moves and the serial chain visits only those.  Every accepted
// move changes the spectrum, so the lanes behind it are screened again; the values a lane holds from its LAST screen
// are exactly rho a_p + delta_p, rho a_s + delta_s of the state at its turn.  Eq. 19 (scale ALL coefficients by rho)
// is applied lazily: a = g * a~, g <- g rho on accept, folded into a~ at the end of every sweep.
//
// Template switches:  W2REG  2 Wj in registers as well (accepted update: 2 instead of 3 instructions per tau-point);
//   ACACHE  a lane keeps the two coefficients of ITS move in registers for the whole batch and an accepted move patches
//           them by shuffle (no global load behind an accepted move; pays when the spectra of the resident walkers
//           overflow L1: Stress);
//   WALK    index selection by a truncated Markov walk on the current spectrum (section 2.3): every lane walks its own
//           move at batch time, and the lanes behind an accepted move walk again (their candidates may have compared
//           against the two changed bins: only those whose walk READ one of them); the Philox words of the first two steps are staged behind the record.
#include "sweep_common.cuh"

// Diagnostic, off by default (no code): SAIL_DIAG_EXTRA_DFMA = N adds N FP64 instructions per evaluated move on two
// chains that nothing in the move depends on.  If the kernel had latency slack they would be free; measured, each costs
// 0.6-0.9 clk per SM per move, i.e. at least its own FP64-pipe time (profiles/r02_sweep_pipe_bound.md).
// Build with `python -m paper_1609_07936_b200.build --force --define SAIL_DIAG_EXTRA_DFMA=8`.
#ifndef SAIL_DIAG_EXTRA_DFMA
#define SAIL_DIAG_EXTRA_DFMA 0
#endif

namespace sail {

// state-independent half of a proposal (row A2): Philox -> uniform p, s (reading G11), rho, -T ln u, 1/rho
struct Draw { int p, s_raw; double alpha; };
__device__ __forceinline__ Draw draw_move(const SweepArgs &P, uint32_t walker, uint32_t sweep, uint32_t move, double y, double T,
                                          unsigned char *rec)
{
    uint32_t x[4];
    philox4x32_10(walker, sweep, move, 0u, P.seed_lo, P.seed_hi, x);
    const int p = (int)__umulhi(x[0], (uint32_t)P.n_omega);
    const int s_raw = (int)__umulhi(x[1], (uint32_t)(P.n_omega - 1));
    // rho in the method's operation order, no contraction: bit-identical to the definition
    const double rho = __dsub_rn(1.0, __dmul_rn(__dmul_rn(y, P.eta), __dsub_rn(__dmul_rn(2.0, u01(x[2])), 1.0)));
    const double thr = -T * log(u01(x[3]));
    *reinterpret_cast<double2 *>(rec + 64) = make_double2(thr, fast_recip(rho));
    return Draw{p, s_raw, __dsub_rn(rho, 1.0)};
}

// Section 2.3 (reading F4): Metropolis on the bin index with uniform candidates, j <- c if
// u a_j < a_c: L steps for p from its uniform start, then s starts from its uniform draw on the bins other than the
// final p and walks L steps on those.  Step l uses Philox counter (walker, sweep, move, 2 + l) = (candidate for p,
// u for p, candidate for s, u for s); the first two steps' words are staged at rec + 80.  The walk reads a RATIO of
// coefficients of the current spectrum, so the lazy scale cancels.
// The bins a walk READ (its two starts and every candidate; at most 2 L + 2): its outcome can change only if one of
// them changes.  Eight 16-bit slots in a 128-bit shift register (n_omega <= 8192 < 0xFFFF, the empty value); a longer
// walk sets `all` and counts as touching every bin.
struct WalkBins {
    unsigned long long lo, hi;
    int n;
    __device__ __forceinline__ void clear() { lo = hi = ~0ull; n = 0; }
    __device__ __forceinline__ void add(int bin) { hi = (hi << 16) | (lo >> 48); lo = (lo << 16) | (unsigned long long)(unsigned)bin; ++n; }
    __device__ __forceinline__ bool has(int bin) const
    {
        if (n > 8) return true;
        const unsigned long long k = (unsigned long long)(unsigned)bin * 0x0001000100010001ull, m = 0x8000800080008000ull, o = 0x0001000100010001ull;
        const unsigned long long x = lo ^ k, y = hi ^ k;                 // a zero 16-bit slot = a match
        return ((((x - o) & ~x) | ((y - o) & ~y)) & m) != 0ull;
    }
};

template <bool TRACK>
__device__ __forceinline__ void index_walk(const SweepArgs &P, uint32_t walker, uint32_t sweep, uint32_t move, int wl,
                                           const unsigned char *rec, const double *a_row, int &p, int s_raw, int &s, WalkBins &vis)
{
    auto words = [&](int l, uint32_t (&xw)[4]) {
        if (l < 2) {
            const uint4 q = *reinterpret_cast<const uint4 *>(rec + 80 + 16 * l);
            xw[0] = q.x; xw[1] = q.y; xw[2] = q.z; xw[3] = q.w;
        } else {
            philox4x32_10(walker, sweep, move, (uint32_t)(2 + l), P.seed_lo, P.seed_hi, xw);
        }
    };
    if (TRACK) { vis.clear(); if (wl > 0) vis.add(p); }
    for (int l = 0; l < wl; ++l) {
        uint32_t xw[4];
        words(l, xw);
        const int c = (int)__umulhi(xw[0], (uint32_t)P.n_omega);
        if (TRACK) vis.add(c);
        if (__dmul_rn(u01(xw[1]), ld_f64(a_row + p)) < ld_f64(a_row + c)) p = c;
    }
    s = s_raw + (s_raw >= p ? 1 : 0);
    if (TRACK && wl > 0) vis.add(s);
    for (int l = 0; l < wl; ++l) {
        uint32_t xw[4];
        words(l, xw);
        int c = (int)__umulhi(xw[2], (uint32_t)(P.n_omega - 1));
        c += (c >= p) ? 1 : 0;
        if (TRACK) vis.add(c);
        if (__dmul_rn(u01(xw[3]), ld_f64(a_row + s)) < ld_f64(a_row + c)) s = c;
    }
}

template <int C, int MAXW, bool FACT, bool TRACE, bool W2REG, bool ACACHE, bool WALK>
__global__ void __maxnreg__((65536 / (((MAXW + 3) & ~3) * 32)) & ~7) sweep_kernel(const SweepArgs P)
{
    constexpr int G = 32;
    constexpr int kRec = WALK ? kRecWalkBytes : kRecBytes;
    // WALK: track the bins a walk read (so that only affected lanes walk again) in the kernels that have the registers
    // for it; measured at L = 2: +10 % on a 1024-bin grid, -4 % at 256 bins in the 72-register form, which keeps re-walking
    constexpr bool TRACK = WALK && C > 4;
    // a schedule written on the device (sail_anneal_selfcool) says "halted" with a non-positive first temperature: the
    // whole launch is then a no-op.  Schedules from the host are validated > 0 by sail_anneal, so this never fires there.
    if (!(__ldg(P.T) > 0.0)) return;
    extern __shared__ __align__(16) unsigned char smem[];
    double *s_ratio = reinterpret_cast<double *>(smem);
    const int n_omega = P.n_omega;
    const int n_omega_pad = (n_omega + 1) & ~1;
    double *s_invd = s_ratio + n_omega_pad;
    double *s_E0 = s_invd + n_omega_pad;
    const int e0_elems = FACT ? (P.n_hi + P.n_lo) * G : n_omega * G;
    unsigned char *s_recs = reinterpret_cast<unsigned char *>(s_E0 + ((e0_elems + 1) & ~1));
    for (int i = threadIdx.x; i < n_omega; i += blockDim.x) { s_ratio[i] = P.ratio[i]; s_invd[i] = P.invd[i]; }
    for (int i = threadIdx.x; i < e0_elems; i += blockDim.x) s_E0[i] = P.E0[i];
    // records of lanes beyond a short last batch are read (and masked out) by the screen: keep p = s = 0 there
    for (int i = threadIdx.x; i < (int)(blockDim.x * (kRec / 4)); i += blockDim.x)
        reinterpret_cast<uint32_t *>(s_recs)[i] = 0u;
    __syncthreads();
    // WALK: the walk gathers the spectrum at random bins right after an accepted move has stored two of them; from
    // global memory every such gather waits for L2 (the stores drop the lines from L1), so each warp keeps a copy of its
    // walker's spectrum in shared memory when the copies of all resident warps fit
    double *s_spec = nullptr;
    if (WALK && P.spec_smem)
        s_spec = reinterpret_cast<double *>(s_recs + (size_t)(blockDim.x >> 5) * 32 * kRec) + (size_t)(threadIdx.x >> 5) * n_omega_pad;

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    unsigned char *my_rec_w = s_recs + ((size_t)warp * 32 + lane) * kRec;
    // 32-bit shared-window addresses, made opaque so that they stay in registers instead of being rematerialised
    uint32_t rbase = (uint32_t)__cvta_generic_to_shared(s_recs) + (uint32_t)(warp * 32 * kRec);
    uint32_t e0_lane = (uint32_t)__cvta_generic_to_shared(s_E0) + (uint32_t)(lane * 8);
    asm volatile("" : "+r"(rbase), "+r"(e0_lane));
    const uint32_t rec_own = rbase + (uint32_t)(lane * kRec);
    const uint32_t e0_lo = e0_lane + (uint32_t)(P.n_hi * G * 8);
    const int warps_per_cta = blockDim.x >> 5;
    const int fshift = P.fact_shift;
    const int fmask = (1 << fshift) - 1;
    const double half_dw = 0.5 * P.domega;
    // omega_k^m = omega_k + domega/2 (Eq. 14), from the caller's grid values
    auto wm = [&](int k) { return __dadd_rn(__ldg(P.omega + k), half_dw); };

    for (long long w = (long long)blockIdx.x * warps_per_cta + warp; w < P.W; w += (long long)gridDim.x * warps_per_cta) {
        // element offset of this walker's spectrum: the whole spectra array has < 2^32 elements (checked at launch)
        uint32_t wbase = (uint32_t)(w * n_omega);
        asm volatile("" : "+r"(wbase));
        double *const a_all = P.a;
        double mt[C], G2[C], Wt[C], d[C], W2[W2REG ? C : 1];
#pragma unroll
        for (int i = 0; i < C; ++i) {
            const int j = lane + G * i;
            const bool ok = j < P.n_tau;
            mt[i] = ok ? P.mt[(size_t)w * P.n_tau + j] : 0.0;
            Wt[i] = ok ? P.Wj[j] : 0.0;
            if (W2REG) W2[i] = Wt[i] + Wt[i];
            d[i] = 0.0;
        }
        const double *walk_src = a_all + wbase;           // where the index walk and (WALK) the screen read the spectrum
        if (WALK && s_spec) {
            for (int k = lane; k < n_omega; k += G) s_spec[k] = a_all[(size_t)wbase + k];
            walk_src = s_spec;
            __syncwarp();
        }
        const uint32_t wid = (uint32_t)(w + P.walker0);      // Philox counter word 0: the GLOBAL walker index
        double chi2 = P.chi2[w];
#if SAIL_DIAG_EXTRA_DFMA > 0
        double diag_a = 0.5, diag_b = 0.25;
#endif
        double g = 1.0, ginv = 1.0;
        bool tracing = false;
        if (TRACE) tracing = P.trace != nullptr && w >= P.trace_lo && w < P.trace_hi;

        for (int isw = 0; isw < P.n_sweeps; ++isw) {
            int acc_sweep = 0, eval_sweep = 0;
#pragma unroll
            for (int i = 0; i < C; ++i) {
                const int j = lane + G * i;
                const double f = (j < P.n_tau) ? P.fj[j] : 0.0;
                G2[i] = 2.0 * Wt[i] * (mt[i] - f);
            }
            const double y_sweep = P.y[w];
            const double T_sweep = P.T[isw];
            const uint32_t sweep_abs = (uint32_t)(P.sweep0 + isw);
            for (int m0 = 0; m0 < n_omega; m0 += G) {
                const int nb = min(G, n_omega - m0);
                // ---- proposals of the batch (row A2), one move per lane ------------------------------------
                Draw dr{0, 0, 0.0};
                int wl = 0;                                        // WALK: steps this lane's move walks
                WalkBins vis;                                      // WALK: the bins this lane's walk read
                vis.clear();
                if (lane < nb) {
                    dr = draw_move(P, wid, sweep_abs, (uint32_t)(m0 + lane), y_sweep, T_sweep, my_rec_w);
                    int p = dr.p, s = dr.s_raw + (dr.s_raw >= dr.p ? 1 : 0);
                    if (WALK) {
                        wl = P.walk_len;
                        if (P.walk_uniform > 0.0) {                // :158 uniform admixture: this move keeps its uniform indices
                            uint32_t xm[4];
                            philox4x32_10(wid, sweep_abs, (uint32_t)(m0 + lane), (uint32_t)(2 + P.walk_len), P.seed_lo, P.seed_hi, xm);
                            if (u01(xm[0]) < P.walk_uniform) wl = 0;
                        }
#pragma unroll
                        for (int l = 0; l < 2; ++l) {
                            uint32_t xw[4] = {0u, 0u, 0u, 0u};
                            if (l < wl) philox4x32_10(wid, sweep_abs, (uint32_t)(m0 + lane), (uint32_t)(2 + l), P.seed_lo, P.seed_hi, xw);
                            *reinterpret_cast<uint4 *>(my_rec_w + 80 + 16 * l) = make_uint4(xw[0], xw[1], xw[2], xw[3]);
                        }
                        index_walk<TRACK>(P, wid, sweep_abs, (uint32_t)(m0 + lane), wl, my_rec_w, walk_src, p, dr.s_raw, s, vis);
                    }
                    write_indexed(P, p, s, dr.alpha, s_ratio, s_invd, wm(s), wm(p), my_rec_w);
                }
                __syncwarp();
                const uint32_t valid = (nb == 32) ? 0xffffffffu : ((1u << nb) - 1u);

                // ---- positivity screen (row A3), one move per lane --------------------------
                double apn = 0.0, asn = 0.0;          // rho a_p + delta_p, rho a_s + delta_s of this lane's move
                double ca_p = 0.0, ca_s = 0.0;        // ACACHE: a~_p, a~_s of this lane's move
                if (ACACHE) {
                    const int4 q0 = lds_s32x4(rec_own);
                    ca_p = ldg_f64(elem_ptr(a_all, wbase + (uint32_t)q0.x));
                    ca_s = ldg_f64(elem_ptr(a_all, wbase + (uint32_t)q0.y));
                }
                auto screen = [&](uint32_t sel) -> uint32_t {
                    const int4 q0 = lds_s32x4(rec_own);
                    const double2 qd = lds_f64x2(rec_own + 16);
                    const double a_p = ACACHE ? ca_p : WALK ? ld_f64(walk_src + q0.x) : ldg_f64(elem_ptr(a_all, wbase + (uint32_t)q0.x));
                    const double a_s = ACACHE ? ca_s : WALK ? ld_f64(walk_src + q0.y) : ldg_f64(elem_ptr(a_all, wbase + (uint32_t)q0.y));
                    const double qa = __hiloint2double(q0.w, q0.z);
                    const double gn = fma(qa, g, g);
                    const double x_p = fma(gn, a_p, qd.x);
                    const double x_s = fma(gn, a_s, qd.y);
                    if (!TRACE || ((sel >> lane) & 1u)) { apn = x_p; asn = x_s; }
                    const bool feas = (__double2hiint(x_p) | __double2hiint(x_s)) >= 0;
                    return __ballot_sync(0xffffffffu, feas) & sel;
                };
                uint32_t mask = screen(valid);
                uint32_t ev_mask = 0u, tr_acc = 0u;   // moves evaluated / (TRACE) accepted in this batch
                double tr_dchi2 = 0.0;

                while (mask) {
                    const int m = __ffs((int)mask) - 1;
                    const uint32_t r = rbase + (uint32_t)(m * kRec);
                    const int4 r0 = lds_s32x4(r);
                    const double2 dd = lds_f64x2(r + 16);
                    const double2 dr2 = lds_f64x2(r + 32);
                    const double2 sc = lds_f64x2(r + 48);
                    const double2 th = lds_f64x2(r + 64);
                    const double alpha = __hiloint2double(r0.w, r0.z);
                    double e0p, e0s;
                    if (FACT) {
                        e0p = lds_f64(e0_lane + (uint32_t)((r0.x >> fshift) * (G * 8))) * lds_f64(e0_lo + (uint32_t)((r0.x & fmask) * (G * 8)));
                        e0s = lds_f64(e0_lane + (uint32_t)((r0.y >> fshift) * (G * 8))) * lds_f64(e0_lo + (uint32_t)((r0.y & fmask) * (G * 8)));
                    } else {
                        e0p = lds_f64(e0_lane + (uint32_t)(r0.x * (G * 8)));
                        e0s = lds_f64(e0_lane + (uint32_t)(r0.y * (G * 8)));
                    }
                    // ---- incremental Delta chi^2 over all tau (row A4, Eq. 22 + Eq. 9) -------------------
                    double vm = fma(dd.x, e0p, dd.y * e0s);        // v_0
                    double vc = fma(dr2.x, e0p, dr2.y * e0s);      // v_1
                    double acc_a = 0.0, acc_b = 0.0;
#pragma unroll
                    for (int i = 0; i < C; ++i) {
                        double vi;
                        if (i == 0) vi = vm;
                        else if (i == 1) vi = vc;
                        else { vi = fma(sc.x, vc, sc.y * vm); vm = vc; vc = vi; }
                        d[i] = fma(alpha, mt[i], vi);
                        const double t = fma(Wt[i], d[i], G2[i]);
                        if (i & 1) acc_b = fma(d[i], t, acc_b);
                        else       acc_a = fma(d[i], t, acc_a);
                    }
#if SAIL_DIAG_EXTRA_DFMA > 0
#pragma unroll
                    for (int q = 0; q < SAIL_DIAG_EXTRA_DFMA; ++q) {
                        if (q & 1) diag_b = fma(diag_b, alpha, th.x);
                        else       diag_a = fma(diag_a, alpha, th.x);
                    }
#endif
                    const double dchi2 = warp_sum_dmma((C > 1) ? acc_a + acc_b : acc_a);
                    ev_mask |= 1u << m;
                    if (TRACE) { if (lane == m) tr_dchi2 = dchi2; }
                    // ---- Metropolis (row A5, Eq. 10); identical in every lane: a uniform branch ----------
                    if (dchi2 < th.x) {
#pragma unroll
                        for (int i = 0; i < C; ++i) {
                            mt[i] += d[i];
                            if (W2REG) G2[i] = fma(W2[i], d[i], G2[i]);
                            else       G2[i] = fma(Wt[i], d[i] + d[i], G2[i]);
                        }
                        chi2 += dchi2;
                        g = fma(alpha, g, g);
                        ginv *= th.y;
                        const int mine = (lane == m) ? 1 : 0;
                        const double newp = apn * ginv, news = asn * ginv;
                        stg_f64_if(elem_ptr(a_all, wbase + (uint32_t)r0.x), newp, mine);
                        stg_f64_if(elem_ptr(a_all, wbase + (uint32_t)r0.y), news, mine);
                        if (WALK && s_spec && mine) { s_spec[r0.x] = newp; s_spec[r0.y] = news; }
                        acc_sweep++;
                        if (TRACE) tr_acc |= 1u << m;
                        const uint32_t behind = valid & ~((2u << m) - 1u);
                        if (ACACHE) {
                            const double bp = __shfl_sync(0xffffffffu, newp, m);
                            const double bs = __shfl_sync(0xffffffffu, news, m);
                            const int2 q = *reinterpret_cast<const int2 *>(my_rec_w);
                            if (q.x == r0.x) ca_p = bp;
                            if (q.x == r0.y) ca_p = bs;
                            if (q.y == r0.x) ca_s = bp;
                            if (q.y == r0.y) ca_s = bs;
                        } else {
                            __syncwarp();
                        }
                        if (WALK) {
                            // the accepted move changed bins p and s: a lane behind it walks again only if its walk
                            // READ one of the two (nothing else can change its indices); no lane, no work
                            const bool again = ((behind >> lane) & 1u) && wl > 0 && (!TRACK || vis.has(r0.x) || vis.has(r0.y));
                            if (__ballot_sync(0xffffffffu, again)) {
                                if (again) {
                                    const int2 q = *reinterpret_cast<const int2 *>(my_rec_w);
                                    int p = dr.p, s = q.y;
                                    index_walk<TRACK>(P, wid, sweep_abs, (uint32_t)(m0 + lane), wl, my_rec_w, walk_src, p, dr.s_raw, s, vis);
                                    if (p != q.x || s != q.y) write_indexed(P, p, s, dr.alpha, s_ratio, s_invd, wm(s), wm(p), my_rec_w);
                                }
                                __syncwarp();
                            }
                        }
                        // the spectrum changed: screen the moves behind this one again
                        mask = screen(behind);
                    } else {
                        mask &= mask - 1u;
                    }
                }
                eval_sweep += __popc(ev_mask);
                if (TRACE) {
                    if (lane < nb) {
                        const int4 q0 = lds_s32x4(rec_own);
                        const double2 qd = lds_f64x2(rec_own + 16);
                        const double2 qt = lds_f64x2(rec_own + 64);
                        const bool feas = (__double2hiint(apn) | __double2hiint(asn)) >= 0;
                        const int fl = (feas ? 1 : 0) | (((tr_acc >> lane) & 1u) ? 2 : 0) | (((ev_mask >> lane) & 1u) ? 4 : 0);
                        const size_t mv = ((size_t)(P.call_off + isw)) * n_omega + m0 + lane;
                        if (P.flags) P.flags[(size_t)w * P.call_sweeps * n_omega + mv] = (uint8_t)fl;
                        if (tracing) {
                            sail_trace_rec *tr = P.trace + ((size_t)(w - P.trace_lo) * P.call_sweeps * n_omega + mv);
                            tr->p = q0.x; tr->s = q0.y; tr->flags = fl; tr->move = m0 + lane;
                            tr->rho = 1.0 + __hiloint2double(q0.w, q0.z); tr->delta_p = qd.x; tr->delta_s = qd.y;
                            tr->dchi2 = tr_dchi2; tr->thr = qt.x; tr->ap_new = apn; tr->as_new = asn;
                        }
                    }
                }
                __syncwarp();
            }
            // ---- end of sweep: fold the lazy scale (Eq. 19), counters, y (row A6, Eq. 30) ----------------
            for (int k = lane; k < n_omega; k += G) {
                const double v = ((WALK && s_spec) ? s_spec[k] : a_all[(size_t)wbase + k]) * g;
                a_all[(size_t)wbase + k] = v;
                if (WALK && s_spec) s_spec[k] = v;
            }
            g = 1.0;
            ginv = 1.0;
            if (lane == 0) {
                P.n_acc[w] += (unsigned long long)acc_sweep;
                P.n_eval[w] += (unsigned long long)eval_sweep;
                P.y[w] = amp_factor(P, acc_sweep, y_sweep);
            }
            __syncwarp();
        }
#pragma unroll
        for (int i = 0; i < C; ++i) {
            const int j = lane + G * i;
            if (j < P.n_tau) P.mt[(size_t)w * P.n_tau + j] = mt[i];
        }
#if SAIL_DIAG_EXTRA_DFMA > 0
        if (diag_a + diag_b == 1.2345) chi2 += 1.0;           // never: keeps the two chains alive
#endif
        if (lane == 0) P.chi2[w] = chi2;
        __syncwarp();
    }
}

// ---- sweep tables: ratio[k] = exp(-omega_k 32 dtau); invd[k] = 1/(k domega); start values E0 ----------
__global__ void sweep_tables_kernel(int n_omega, int G, double domega, double tau0, double dtau,
                                    const double *omega, int fact, int shift, int n_hi, int n_lo,
                                    double *ratio, double *invd, double *E0)
{
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int stride = gridDim.x * blockDim.x;
    for (int k = tid; k < n_omega; k += stride) {
        ratio[k] = exp(-omega[k] * ((double)G * dtau));
        invd[k] = k ? 1.0 / ((double)k * domega) : 0.0;
    }
    if (!fact) {
        for (int i = tid; i < n_omega * G; i += stride) {
            const int k = i / G, l = i % G;
            E0[i] = exp(-omega[k] * (tau0 + l * dtau));
        }
    } else {
        for (int i = tid; i < (n_hi + n_lo) * G; i += stride) {
            const int r = i / G, l = i % G;
            const double t = tau0 + l * dtau;
            // high part carries omega_0; low part the remaining k_lo * domega
            E0[i] = (r < n_hi) ? exp(-omega[(size_t)r << shift] * t) : exp(-((double)(r - n_hi) * domega) * t);
        }
    }
}

// direct start table E0[k][lane] up to 64 KB, otherwise the product of two small tables H[k_hi][lane] L[k_lo][lane]
static void table_shape(int n_omega, bool *fact, int *shift, int *n_hi, int *n_lo)
{
    *fact = (size_t)n_omega * 32 * sizeof(double) > 64 * 1024;
    *shift = *n_hi = *n_lo = 0;
    if (*fact) {
        int bits = 0;
        while ((1 << bits) < n_omega) bits++;
        *shift = bits / 2;
        *n_lo = 1 << *shift;
        *n_hi = (n_omega + *n_lo - 1) >> *shift;
    }
}

int ensure_sweep_tables(sail_handle *h)
{
    if (h->tables_ready) return SAIL_OK;
    bool fact;
    int shift, n_hi, n_lo;
    table_shape(h->n_omega, &fact, &shift, &n_hi, &n_lo);
    h->tables_fact = fact;
    h->fact_shift = shift;
    sweep_tables_kernel<<<64, 256, 0, h->stream>>>(h->n_omega, 32, h->domega, h->tau0, h->dtau, h->tab.omega,
                                                   fact ? 1 : 0, shift, n_hi, n_lo, h->sw_ratio, h->sw_invd, h->sw_E0);
    SAIL_LAUNCH_OK(h, "sweep_tables_kernel");
    h->tables_ready = true;
    return SAIL_OK;
}

// shared memory of one CTA: ratio + invd tables, start table(s), one record per lane of every warp
static size_t sweep_smem_bytes(int n_omega, int warps, bool walk)
{
    bool fact;
    int shift, n_hi, n_lo;
    table_shape(n_omega, &fact, &shift, &n_hi, &n_lo);
    const int e0_elems = fact ? (n_hi + n_lo) * 32 : n_omega * 32;
    return (size_t)(2 * ((n_omega + 1) & ~1) + ((e0_elems + 1) & ~1)) * sizeof(double)
           + (size_t)warps * 32 * (walk ? kRecWalkBytes : kRecBytes);
}

// does the sweep kernel launch at this n_omega (tables + the records of at least four warps within 227 KB)?
bool sweep_fits(int n_omega) { return sweep_smem_bytes(n_omega, 4, true) <= 227 * 1024; }

// doubles of the start table(s) (workspace sizing)
size_t sweep_e0_doubles(int n_omega)
{
    bool fact;
    int shift, n_hi, n_lo;
    table_shape(n_omega, &fact, &shift, &n_hi, &n_lo);
    return fact ? (size_t)(n_hi + n_lo) * 32 : (size_t)n_omega * 32;
}

template <int C, int MAXW, bool FACT, bool TRACE, bool W2REG, bool ACACHE, bool WALK>
static int launch_variant(sail_handle *h, SweepArgs &args)
{
    int warps = (int)((args.W + h->num_sms - 1) / h->num_sms);
    if (warps > MAXW) warps = MAXW;
    if (warps < 1) warps = 1;
    // large omega grids: fewer warps per CTA until tables + records fit the 227 KB of one SM
    while (warps > 1 && sweep_smem_bytes(args.n_omega, warps, WALK) > 227 * 1024) --warps;
    size_t smem = sweep_smem_bytes(args.n_omega, warps, WALK);
    if (smem > 227 * 1024)
        return set_err(h, SAIL_ERR_ARG, "sweep tables need %zu bytes of shared memory (> 227 KB)", smem);
    const size_t spec_bytes = (size_t)warps * ((args.n_omega + 1) & ~1) * sizeof(double);
    args.spec_smem = (WALK && smem + spec_bytes <= 227 * 1024) ? 1 : 0;
    if (args.spec_smem) smem += spec_bytes;
    long long ctas = (args.W + warps - 1) / warps;
    if (ctas > h->num_sms) ctas = h->num_sms;
    void (*kern)(const SweepArgs) = sweep_kernel<C, MAXW, FACT, TRACE, W2REG, ACACHE, WALK>;
    SAIL_CUDA_OK(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<(unsigned)ctas, warps * 32, smem, h->stream>>>(args);
    SAIL_LAUNCH_OK(h, "sweep_kernel");
    return SAIL_OK;
}

template <int C, int MAXW, bool W2REG, bool ACACHE>
static int launch_c(sail_handle *h, SweepArgs &a, bool trace)
{
    const bool walk = a.walk_len > 0;
    // the walking kernels run as many warps per SM as the plain ones (fewer were tried and lost); when the spectra of the
    // resident warps fit beside tables + records they are copied to shared memory (launch_variant: spec_smem)
    constexpr int MAXW_WALK = MAXW;
#define SAIL_PICK(FA, TR)                                                                    \
    return walk ? launch_variant<C, MAXW_WALK, FA, TR, W2REG, false, true>(h, a)            \
                : launch_variant<C, MAXW, FA, TR, W2REG, ACACHE, false>(h, a);
    if (a.fact) { if (trace) { SAIL_PICK(true, true) } else { SAIL_PICK(true, false) } }
    if (trace) { SAIL_PICK(false, true) }
    SAIL_PICK(false, false)
#undef SAIL_PICK
}

int launch_sweeps(sail_handle *h, const double *d_T, int64_t n_sweeps, const sail_anneal_params *p,
                  int64_t sweeps_in_call, int64_t call_offset)
{
    constexpr int G = 32;
    if (p->walk_length < 0 || p->walk_length > 4096) return set_err(h, SAIL_ERR_ARG, "walk_length=%d outside [0, 4096]", p->walk_length);
    if (!(p->walk_uniform >= 0.0 && p->walk_uniform <= 1.0)) return set_err(h, SAIL_ERR_ARG, "walk_uniform must lie in [0, 1]");
    const int C = (h->n_tau + G - 1) / G;
    if (C > 16) return set_err(h, SAIL_ERR_ARG, "n_tau=%d needs more than 16 tau-points per lane", h->n_tau);
    int rc = ensure_sweep_tables(h);
    if (rc) return rc;
    if ((unsigned long long)h->W * (unsigned long long)h->n_omega >= (1ull << 32))
        return set_err(h, SAIL_ERR_ARG, "W * n_omega must be < 2^32 spectral coefficients");

    SweepArgs a{};
    a.n_omega = h->n_omega; a.n_tau = h->n_tau; a.W = h->W; a.walker0 = h->walker0;
    a.A = h->A; a.B = h->B; a.domega = h->domega; a.eta = p->eta;
    a.amp_p = p->amp_p; a.amp_m = p->amp_m; a.y_min = p->y_min; a.amp_mode = p->amp_mode;
    a.seed_lo = (uint32_t)(h->seed & 0xFFFFFFFFu); a.seed_hi = (uint32_t)(h->seed >> 32);
    a.Wj = h->tab.Wj; a.fj = h->tab.fj; a.ratio = h->sw_ratio; a.E0 = h->sw_E0; a.invd = h->sw_invd; a.omega = h->tab.omega;
    a.fact = h->tables_fact ? 1 : 0; a.fact_shift = h->fact_shift;
    if (h->tables_fact) { a.n_lo = 1 << h->fact_shift; a.n_hi = (h->n_omega + a.n_lo - 1) >> h->fact_shift; }
    a.a = h->st.a; a.mt = h->st.mt; a.chi2 = h->st.chi2; a.y = h->st.y;
    a.n_acc = h->st.n_acc; a.n_eval = h->st.n_eval;
    a.T = d_T; a.sweep0 = h->sweep; a.n_sweeps = (int)n_sweeps;
    a.walk_len = p->walk_length; a.walk_uniform = p->walk_uniform;
    a.trace_lo = p->trace_lo; a.trace_hi = p->trace_hi; a.trace = p->trace; a.flags = p->flags;
    a.call_sweeps = sweeps_in_call; a.call_off = call_offset;
    const bool trace = (p->trace != nullptr) || (p->flags != nullptr);

    // register budgets: 72 (C <= 4, 28 warps per SM), 128 (C <= 8, 16 warps), 168 (C <= 16, 12 warps)
    if (C <= 4) return launch_c<4, 28, false, false>(h, a, trace);
    if (C <= 7) return launch_c<7, 16, true, false>(h, a, trace);
    if (C <= 8) return launch_c<8, 16, true, false>(h, a, trace);
    return launch_c<16, 12, false, true>(h, a, trace);
}

} // namespace sail
