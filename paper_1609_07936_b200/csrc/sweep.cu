// sweep.cu — the persistent Monte Carlo sweep kernels with one walker per warp (
// PAPER.md:127-148, :205) and the dispatch of all sweep-kernel forms.
//
// Mapping: one walker per warp; lane l owns tau-points j = l + 32 i, i < C, whose residual state
// lives in REGISTERS for the whole launch:
//     mt_j  = sum_k a_k exp(-omega_k tau_j)      (model in the pure-exponential basis, M_j = c_j mt_j)
//     G2_j  = 2 Wj (mt_j - fj)                   (Wj = (c_j/sigma_j)^2, fj = F_j/c_j)
// so that for a move (p, s, rho, delta_p, delta_s) (Eq. 17-22):
//     dt_j   = (rho-1) mt_j + delta_p E_pj + delta_s E_sj          E_kj = exp(-omega_k tau_j)
//     dchi2  = sum_j dt_j (Wj dt_j + G2_j)     [= sum_j d_j (d_j + 2 D_j) of SURVEY §8a row A4]
// The kernel rows are never read from a table in the inner loop: both grids are uniform (Eq. 2-3, 7), so
// E_{k,j+32} = E_kj exp(-omega_k 32 dtau); each lane starts from E0[k][l] (shared memory) and advances by a
// recurrence along its tau-points.
//   sweep_kernel_mask (default): positivity screened for a 32-move batch at once (ballot), two-term recurrence for
//       delta_p E_p + delta_s E_s (5 FP64 per tau-point), warp sum on the DMMA path; see its own comment below;
//   sweep_kernel_warp: the plain form — every move visited in turn, one geometric recurrence per row (6 FP64 per
//       tau-point), shuffle butterfly; kept as the simple reference form of the same arithmetic.
// Proposals (Philox4x32-10 keyed by (seed; walker, sweep, move, 0), index draw, rho, Eq. 20-21, -T ln u) do not
// depend on the chain state within a sweep, so they are computed 32 moves at a time, one move per lane, and staged
// as records in shared memory.  Eq. 19 (scale ALL coefficients by rho) is applied lazily: a = g * a~, g <- g rho on
// accept, folded into a~ at the end of every sweep.  Walker slots W .. W_pad-1 (W_pad = W rounded up to 4) are
// scratch copies of the last walker (used by the grouped kernel of sweep_grp.cu); they are never reported.
#include "sweep_common.cuh"

namespace sail {

// ---- one proposal (row A2): Philox4x32-10 keyed by (seed; walker, sweep, move, 0) -> 64-byte record ------
//   [ 0] p, s (int32), alpha = rho - 1      [16] delta_p, delta_s (Eq. 20-21)
//   [32] thr = -T ln u_acc, 1/rho            [48] exp(-omega_p G dtau), exp(-omega_s G dtau)
__device__ __forceinline__ void propose(const SweepArgs &P, uint32_t walker, uint32_t sweep, uint32_t move, double y, double T,
                                        const double *s_ratio, const double *s_invd, const double *s_wm, unsigned char *rec)
{
    uint32_t x[4];
    philox4x32_10(walker, sweep, move, 0u, P.seed_lo, P.seed_hi, x);
    const int p = (int)__umulhi(x[0], (uint32_t)P.n_omega);
    int s = (int)__umulhi(x[1], (uint32_t)(P.n_omega - 1));
    s += (s >= p) ? 1 : 0;
    const double u_rho = ((double)x[2] + 0.5) * 2.3283064365386962890625e-10;
    const double u_acc = ((double)x[3] + 0.5) * 2.3283064365386962890625e-10;
    // rho in the method's operation order, no contraction: bit-identical to the definition
    const double rho = __dsub_rn(1.0, __dmul_rn(__dmul_rn(y, P.eta), __dsub_rn(__dmul_rn(2.0, u_rho), 1.0)));
    const double alpha = __dsub_rn(rho, 1.0);          // exact
    // Eq. 20-21 in the method's operation order; only the division by (p-s) domega is a multiplication by
    // the correctly rounded reciprocal (delta within 2 ulp of the division form)
    const double omr = __dsub_rn(1.0, rho);
    const int dps = p - s;
    const double inv = (dps > 0) ? s_invd[dps] : -s_invd[-dps];
    const double dp = __dmul_rn(__dmul_rn(omr, __dsub_rn(P.B, __dmul_rn(P.A, s_wm[s]))), inv);
    const double ds = -__dmul_rn(__dmul_rn(omr, __dsub_rn(P.B, __dmul_rn(P.A, s_wm[p]))), inv);
    const double thr = -T * log(u_acc);
    *reinterpret_cast<int4 *>(rec) = make_int4(p, s, __double2loint(alpha), __double2hiint(alpha));
    *reinterpret_cast<double2 *>(rec + 16) = make_double2(dp, ds);
    *reinterpret_cast<double2 *>(rec + 32) = make_double2(thr, fast_recip(rho));
    *reinterpret_cast<double2 *>(rec + 48) = make_double2(s_ratio[p], s_ratio[s]);
}

// ---- one walker per WARP, register-lean (<= 72 registers: 28 resident warps per SM = 7 per sub-partition) ------
// No software pipeline (the other six warps of the sub-partition hide
// the latencies), every decision is warp-uniform, so infeasible and rejected moves branch around the work.
template <int C, int MAXW, bool FACT, bool TRACE, bool WALK>
__global__ void __maxnreg__((65536 / (((MAXW + 3) & ~3) * 32)) & ~7) sweep_kernel_warp(const SweepArgs P)
{
    constexpr int G = 32;
    constexpr int kRecBytes = WALK ? 96 : sail::kRecBytes;   // WALK: + the Philox words of the first two walk steps
    extern __shared__ __align__(16) unsigned char smem[];
    double *s_ratio = reinterpret_cast<double *>(smem);
    const int n_omega = P.n_omega;
    const int n_omega_pad = (n_omega + 1) & ~1;
    double *s_invd = s_ratio + n_omega_pad;
    double *s_wm = s_invd + n_omega_pad;
    double *s_E0 = s_wm + n_omega_pad;
    const int e0_elems = FACT ? (P.n_hi + P.n_lo) * G : n_omega * G;
    unsigned char *s_recs = reinterpret_cast<unsigned char *>(s_E0 + ((e0_elems + 1) & ~1));
    for (int i = threadIdx.x; i < n_omega; i += blockDim.x) {
        s_ratio[i] = P.ratio[i]; s_invd[i] = P.invd[i]; s_wm[i] = __dadd_rn(P.omega[i], 0.5 * P.domega);
    }
    for (int i = threadIdx.x; i < e0_elems; i += blockDim.x) s_E0[i] = P.E0[i];
    __syncthreads();

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    unsigned char *my_rec_w = s_recs + ((size_t)warp * 32 + lane) * kRecBytes;
    // 32-bit shared-window addresses, made opaque so that they stay in registers instead of being
    // rematerialised (the generic->shared conversion costs an S2R + several ALU instructions per move)
    uint32_t rbase = (uint32_t)__cvta_generic_to_shared(s_recs) + (uint32_t)(warp * 32 * kRecBytes);
    uint32_t e0_lane = (uint32_t)__cvta_generic_to_shared(s_E0) + (uint32_t)(lane * 8);
    asm volatile("" : "+r"(rbase), "+r"(e0_lane));
    const uint32_t e0_lo = e0_lane + (uint32_t)(P.n_hi * G * 8);
    const int warps_per_cta = blockDim.x >> 5;
    const int fshift = P.fact_shift;
    const int fmask = (1 << fshift) - 1;
    const int lane0 = (lane == 0) ? 1 : 0;

    for (long long w = (long long)blockIdx.x * warps_per_cta + warp; w < P.n_groups; w += (long long)gridDim.x * warps_per_cta) {
        // element offset of this walker's spectrum: the whole spectra array has < 2^32 elements (checked at launch)
        uint32_t wbase = (uint32_t)(w * n_omega);
        asm volatile("" : "+r"(wbase));
        double *const a_all = P.a;
        double mt[C], G2[C], Wt[C], d[C];
#pragma unroll
        for (int i = 0; i < C; ++i) {
            const int j = lane + G * i;
            const bool ok = j < P.n_tau;
            mt[i] = ok ? P.mt[(size_t)w * P.n_tau + j] : 0.0;
            Wt[i] = ok ? P.Wj[j] : 0.0;
            d[i] = 0.0;
        }
        double chi2 = P.chi2[w];
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
            for (int m0 = 0; m0 < n_omega; m0 += G) {
                const int nb = min(G, n_omega - m0);
                if (lane < nb)
                    propose(P, (uint32_t)w, (uint32_t)(P.sweep0 + isw), (uint32_t)(m0 + lane), P.y[w], P.T[isw],
                            s_ratio, s_invd, s_wm, my_rec_w);
                if (WALK) {
                    // the random words of the walk do not depend on the state: the first two steps are drawn here, one
                    // move per lane, and staged behind the record
                    if (lane < nb) {
#pragma unroll
                        for (int l = 0; l < 2; ++l) {
                            uint32_t xw[4] = {0u, 0u, 0u, 0u};
                            if (l < P.walk_len)
                                philox4x32_10((uint32_t)w, (uint32_t)(P.sweep0 + isw), (uint32_t)(m0 + lane), (uint32_t)(2 + l), P.seed_lo, P.seed_hi, xw);
                            *reinterpret_cast<uint4 *>(my_rec_w + 64 + 16 * l) = make_uint4(xw[0], xw[1], xw[2], xw[3]);
                        }
                    }
                }
                __syncwarp();
                const uint32_t r_end = rbase + (uint32_t)(nb * kRecBytes);
                for (uint32_t r = rbase; r != r_end; r += kRecBytes) {
                    int4 r0 = lds_s32x4(r);
                    double2 dd = lds_f64x2(r + 16);
                    const double alpha = __hiloint2double(r0.w, r0.z);
                    double2 rr = lds_f64x2(r + 48);
                    const double2 th = lds_f64x2(r + 32);
                    if (WALK) {
                        // ---- index selection by a truncated Markov walk (section 2.3; reading F4):
                        // Metropolis on the bin index with uniform candidates, j <- c if u a_j < a_c, L steps for p,
                        // then L steps for s on the bins other than p.  The walk reads the CURRENT spectrum (a ratio:
                        // the lazy scale cancels), so it runs at the move's turn, redundantly in every lane, and the
                        // index-dependent half of the proposal (Eq. 20-21, the recurrence ratios) is redone here in the
                        // operation order of propose().
                        const uint32_t mv = (uint32_t)(m0 + (int)((r - rbase) / kRecBytes));
                        const uint32_t sw = (uint32_t)(P.sweep0 + isw);
                        int p = r0.x, s = r0.y;
                        const int sraw = s - (s > p ? 1 : 0);
                        // :158 uniform admixture: below walk_uniform the move keeps its uniform indices
                        int wl = P.walk_len;
                        if (P.walk_uniform > 0.0) {
                            uint32_t xm[4];
                            philox4x32_10((uint32_t)w, sw, mv, (uint32_t)(2 + P.walk_len), P.seed_lo, P.seed_hi, xm);
                            if (((double)xm[0] + 0.5) * 2.3283064365386962890625e-10 < P.walk_uniform) wl = 0;
                        }
                        auto walk_words = [&](int l, uint32_t (&xw)[4]) {
                            if (l < 2) {
                                const int4 q = lds_s32x4(r + 64 + 16 * l);
                                xw[0] = (uint32_t)q.x; xw[1] = (uint32_t)q.y; xw[2] = (uint32_t)q.z; xw[3] = (uint32_t)q.w;
                            } else {
                                philox4x32_10((uint32_t)w, sw, mv, (uint32_t)(2 + l), P.seed_lo, P.seed_hi, xw);
                            }
                        };
                        for (int l = 0; l < wl; ++l) {
                            uint32_t xw[4];
                            walk_words(l, xw);
                            const int c = (int)__umulhi(xw[0], (uint32_t)n_omega);
                            const double u = ((double)xw[1] + 0.5) * 2.3283064365386962890625e-10;
                            if (__dmul_rn(u, ldg_f64(elem_ptr(a_all, wbase + (uint32_t)p))) < ldg_f64(elem_ptr(a_all, wbase + (uint32_t)c))) p = c;
                        }
                        s = sraw + (sraw >= p ? 1 : 0);
                        for (int l = 0; l < wl; ++l) {
                            uint32_t xw[4];
                            walk_words(l, xw);
                            int c = (int)__umulhi(xw[2], (uint32_t)(n_omega - 1));
                            c += (c >= p) ? 1 : 0;
                            const double u = ((double)xw[3] + 0.5) * 2.3283064365386962890625e-10;
                            if (__dmul_rn(u, ldg_f64(elem_ptr(a_all, wbase + (uint32_t)s))) < ldg_f64(elem_ptr(a_all, wbase + (uint32_t)c))) s = c;
                        }
                        const double omr = -alpha;                       // 1 - rho, exact like alpha = rho - 1
                        const int dps = p - s;
                        const double inv = (dps > 0) ? s_invd[dps] : -s_invd[-dps];
                        dd.x = __dmul_rn(__dmul_rn(omr, __dsub_rn(P.B, __dmul_rn(P.A, s_wm[s]))), inv);
                        dd.y = -__dmul_rn(__dmul_rn(omr, __dsub_rn(P.B, __dmul_rn(P.A, s_wm[p]))), inv);
                        rr = make_double2(s_ratio[p], s_ratio[s]);
                        r0.x = p; r0.y = s;
                    }
                    double *const pp = elem_ptr(a_all, wbase + (uint32_t)r0.x);
                    double *const ps = elem_ptr(a_all, wbase + (uint32_t)r0.y);
                    const double a_p = ldg_f64(pp), a_s = ldg_f64(ps);
                    double ep, es;
                    if (FACT) {
                        ep = lds_f64(e0_lane + (uint32_t)((r0.x >> fshift) * (G * 8))) * lds_f64(e0_lo + (uint32_t)((r0.x & fmask) * (G * 8)));
                        es = lds_f64(e0_lane + (uint32_t)((r0.y >> fshift) * (G * 8))) * lds_f64(e0_lo + (uint32_t)((r0.y & fmask) * (G * 8)));
                    } else {
                        ep = lds_f64(e0_lane + (uint32_t)(r0.x * (G * 8)));
                        es = lds_f64(e0_lane + (uint32_t)(r0.y * (G * 8)));
                    }
                    // ---- positivity (row A3) ----------------------------------------------
                    const double gn = fma(alpha, g, g);
                    const double ap_new = fma(gn, a_p, dd.x);
                    const double as_new = fma(gn, a_s, dd.y);
                    const bool feas = (__double2hiint(ap_new) | __double2hiint(as_new)) >= 0;
                    int fl = 0;
                    double dchi2 = 0.0;
                    if (feas) {
                        // ---- incremental Delta chi^2 over all tau (row A4, Eq. 22 + Eq. 9) ---------------
                        ep *= dd.x;
                        es *= dd.y;
                        double acc_a = 0.0, acc_b = 0.0;
#pragma unroll
                        for (int i = 0; i < C; ++i) {
                            d[i] = fma(alpha, mt[i], ep + es);
                            const double t = fma(Wt[i], d[i], G2[i]);
                            if (i & 1) acc_b = fma(d[i], t, acc_b);
                            else       acc_a = fma(d[i], t, acc_a);
                            if (i + 1 < C) { ep *= rr.x; es *= rr.y; }
                        }
                        dchi2 = (C > 1) ? acc_a + acc_b : acc_a;
#pragma unroll
                        for (int off = 16; off > 0; off >>= 1) dchi2 += __shfl_xor_sync(0xffffffffu, dchi2, off);
                        fl = 5;
                        eval_sweep++;
                        // ---- Metropolis (row A5, Eq. 10); identical in every lane: a uniform branch ------
                        if (dchi2 < th.x) {
#pragma unroll
                            for (int i = 0; i < C; ++i) {
                                mt[i] += d[i];
                                G2[i] = fma(Wt[i], d[i] + d[i], G2[i]);
                            }
                            chi2 += dchi2;
                            g = gn;
                            ginv *= th.y;
                            stg_f64_if(pp, ap_new * ginv, lane0);
                            stg_f64_if(ps, as_new * ginv, lane0);
                            acc_sweep++;
                            fl = 7;
                            __syncwarp();
                        }
                    }
                    if (TRACE) {
                        if (lane == 0 && w < P.W) {
                            const int mm = (int)((r - rbase) / kRecBytes);
                            const size_t mv = ((size_t)(P.call_off + isw)) * n_omega + m0 + mm;
                            if (P.flags) P.flags[(size_t)w * P.call_sweeps * n_omega + mv] = (uint8_t)fl;
                            if (tracing) {
                                sail_trace_rec *tr = P.trace + ((size_t)(w - P.trace_lo) * P.call_sweeps * n_omega + mv);
                                tr->p = r0.x; tr->s = r0.y; tr->flags = fl; tr->move = m0 + mm;
                                tr->rho = 1.0 + alpha; tr->delta_p = dd.x; tr->delta_s = dd.y;
                                tr->dchi2 = dchi2; tr->thr = th.x; tr->ap_new = ap_new; tr->as_new = as_new;
                            }
                        }
                    }
                }
                __syncwarp();
            }
            // ---- end of sweep: fold the lazy scale (Eq. 19), counters, y (row A6, Eq. 30) ----------------
            for (int k = lane; k < n_omega; k += G) a_all[(size_t)wbase + k] *= g;
            g = 1.0;
            ginv = 1.0;
            if (lane == 0) {
                P.n_acc[w] += (unsigned long long)acc_sweep;
                P.n_eval[w] += (unsigned long long)eval_sweep;
                P.y[w] = amp_factor(P, acc_sweep, P.y[w]);
            }
            __syncwarp();
        }
#pragma unroll
        for (int i = 0; i < C; ++i) {
            const int j = lane + G * i;
            if (j < P.n_tau) P.mt[(size_t)w * P.n_tau + j] = mt[i];
        }
        if (lane == 0) P.chi2[w] = chi2;
        __syncwarp();
    }
}

// ---- one walker per WARP, feasibility-screened ("mask") form: the default ------------------------------------
// Differences from sweep_kernel_warp (same moves, same decisions):
//  * positivity (row A3) is tested for all moves of a 32-move batch AT ONCE, one move per lane, against the
//    current spectrum: a ballot gives the mask of feasible moves and the serial chain visits only those — an
//    infeasible move costs nothing.  Every accepted move changes the spectrum (all coefficients scale by rho,
//    two of them shift), so the lanes behind it are screened again; the values a lane holds from its LAST
//    screen are exactly rho a_p + delta_p, rho a_s + delta_s of the state at its turn.
//  * the kernel-row combination v_i = delta_p E_p,i + delta_s E_s,i (i = tau-point index of the lane) obeys
//    the two-term linear recurrence of its two geometric modes,
//        v_{i+1} = (r_p + r_s) v_i - (r_p r_s) v_{i-1},      r_k = exp(-omega_k 32 dtau),
//    so the tau loop costs 5 FP64 instructions per tau-point (DMUL + DFMA for v, then the three DFMAs of
//    d, W d + G2, d (W d + G2)): the algorithmic count of SURVEY §8d.  Rounding errors enter relative to |v_i|
//    and propagate through the bounded Green's function (r_p^{n+1} - r_s^{n+1})/(r_p - r_s) <= n + 1.
//  * with W2REG the constants 2 Wj live in registers as well: the accepted update is 2 instructions per
//    tau-point instead of 3.
template <int C, int MAXW, bool FACT, bool TRACE, bool W2REG, int DMMA>
__global__ void __maxnreg__((65536 / (((MAXW + 3) & ~3) * 32)) & ~7) sweep_kernel_mask(const SweepArgs P)
{
    constexpr int G = 32;
    extern __shared__ __align__(16) unsigned char smem[];
    double *s_ratio = reinterpret_cast<double *>(smem);
    const int n_omega = P.n_omega;
    const int n_omega_pad = (n_omega + 1) & ~1;
    double *s_invd = s_ratio + n_omega_pad;
    double *s_wm = s_invd + n_omega_pad;
    double *s_E0 = s_wm + n_omega_pad;
    const int e0_elems = FACT ? (P.n_hi + P.n_lo) * G : n_omega * G;
    unsigned char *s_recs = reinterpret_cast<unsigned char *>(s_E0 + ((e0_elems + 1) & ~1));
    for (int i = threadIdx.x; i < n_omega; i += blockDim.x) {
        s_ratio[i] = P.ratio[i]; s_invd[i] = P.invd[i]; s_wm[i] = __dadd_rn(P.omega[i], 0.5 * P.domega);
    }
    for (int i = threadIdx.x; i < e0_elems; i += blockDim.x) s_E0[i] = P.E0[i];
    // records of lanes beyond a short last batch are read (and masked out) by the screen: keep p = s = 0 there
    for (int i = threadIdx.x; i < (int)(blockDim.x * (kRecMaskBytes / 4)); i += blockDim.x)
        reinterpret_cast<uint32_t *>(s_recs)[i] = 0u;
    __syncthreads();

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    unsigned char *my_rec_w = s_recs + ((size_t)warp * 32 + lane) * kRecMaskBytes;
    uint32_t rbase = (uint32_t)__cvta_generic_to_shared(s_recs) + (uint32_t)(warp * 32 * kRecMaskBytes);
    uint32_t e0_lane = (uint32_t)__cvta_generic_to_shared(s_E0) + (uint32_t)(lane * 8);
    asm volatile("" : "+r"(rbase), "+r"(e0_lane));
    const uint32_t rec_own = rbase + (uint32_t)(lane * kRecMaskBytes);
    const uint32_t e0_lo = e0_lane + (uint32_t)(P.n_hi * G * 8);
    const int warps_per_cta = blockDim.x >> 5;
    const int fshift = P.fact_shift;
    const int fmask = (1 << fshift) - 1;

    for (long long w = (long long)blockIdx.x * warps_per_cta + warp; w < P.n_groups; w += (long long)gridDim.x * warps_per_cta) {
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
        double chi2 = P.chi2[w];
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
            for (int m0 = 0; m0 < n_omega; m0 += G) {
                const int nb = min(G, n_omega - m0);
                if (lane < nb)
                    propose_mask(P, (uint32_t)w, (uint32_t)(P.sweep0 + isw), (uint32_t)(m0 + lane), y_sweep, T_sweep,
                                 s_ratio, s_invd, s_wm, my_rec_w);
                __syncwarp();
                const uint32_t valid = (nb == 32) ? 0xffffffffu : ((1u << nb) - 1u);

                // ---- positivity screen (row A3), one move per lane --------------------------
                double apn = 0.0, asn = 0.0;          // rho a_p + delta_p, rho a_s + delta_s of this lane's move
                auto screen = [&](uint32_t sel) -> uint32_t {
                    const int4 q0 = lds_s32x4(rec_own);
                    const double2 qd = lds_f64x2(rec_own + 16);
                    const double a_p = ldg_f64(elem_ptr(a_all, wbase + (uint32_t)q0.x));
                    const double a_s = ldg_f64(elem_ptr(a_all, wbase + (uint32_t)q0.y));
                    const double qa = __hiloint2double(q0.w, q0.z);
                    const double gn = fma(qa, g, g);
                    const double x_p = fma(gn, a_p, qd.x);
                    const double x_s = fma(gn, a_s, qd.y);
                    if (!TRACE || ((sel >> lane) & 1u)) { apn = x_p; asn = x_s; }
                    const bool feas = (__double2hiint(x_p) | __double2hiint(x_s)) >= 0;
                    return __ballot_sync(0xffffffffu, feas) & sel;
                };
                uint32_t mask = screen(valid);
                uint32_t tr_eval = 0u, tr_acc = 0u;   // TRACE: moves evaluated / accepted in this batch
                double tr_dchi2 = 0.0;

                while (mask) {
                    const int m = __ffs((int)mask) - 1;
                    const uint32_t r = rbase + (uint32_t)(m * kRecMaskBytes);
                    const int4 r0 = lds_s32x4(r);
                    const double2 dd = lds_f64x2(r + 16);
                    const double2 dr = lds_f64x2(r + 32);
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
                    double vc = fma(dr.x, e0p, dr.y * e0s);        // v_1
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
                    double dchi2 = (C > 1) ? acc_a + acc_b : acc_a;
                    if (DMMA == 1) {
                        dchi2 = warp_sum_dmma(dchi2);
                    } else {
#pragma unroll
                        for (int off = 16; off > 0; off >>= 1) dchi2 += __shfl_xor_sync(0xffffffffu, dchi2, off);
                    }
                    eval_sweep++;
                    if (TRACE) { tr_eval |= 1u << m; if (lane == m) tr_dchi2 = dchi2; }
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
                        stg_f64_if(elem_ptr(a_all, wbase + (uint32_t)r0.x), apn * ginv, mine);
                        stg_f64_if(elem_ptr(a_all, wbase + (uint32_t)r0.y), asn * ginv, mine);
                        acc_sweep++;
                        if (TRACE) tr_acc |= 1u << m;
                        __syncwarp();
                        // the spectrum changed: screen the moves behind this one again
                        mask = screen(valid & ~((2u << m) - 1u));
                    } else {
                        mask &= mask - 1u;
                    }
                }
                if (TRACE) {
                    if (lane < nb && w < P.W) {
                        const int4 q0 = lds_s32x4(rec_own);
                        const double2 qd = lds_f64x2(rec_own + 16);
                        const double2 qt = lds_f64x2(rec_own + 64);
                        const bool feas = (__double2hiint(apn) | __double2hiint(asn)) >= 0;
                        const int fl = (feas ? 1 : 0) | (((tr_acc >> lane) & 1u) ? 2 : 0) | (((tr_eval >> lane) & 1u) ? 4 : 0);
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
            for (int k = lane; k < n_omega; k += G) a_all[(size_t)wbase + k] *= g;
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
        if (lane == 0) P.chi2[w] = chi2;
        __syncwarp();
    }
}

// ---- sweep tables: ratio[k] = exp(-omega_k G dtau); invd[k] = 1/(k domega); start values E0 ----------
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

// scratch walker slots W .. W_pad-1 := copies of walker W-1
__global__ void pad_walkers_kernel(int n_omega, int n_tau, long long W, long long W_pad, double *a, double *mt,
                                   double *chi2, double *y)
{
    for (long long r = W + blockIdx.x; r < W_pad; r += gridDim.x) {
        for (int k = threadIdx.x; k < n_omega; k += blockDim.x) a[(size_t)r * n_omega + k] = a[(size_t)(W - 1) * n_omega + k];
        for (int j = threadIdx.x; j < n_tau; j += blockDim.x) mt[(size_t)r * n_tau + j] = mt[(size_t)(W - 1) * n_tau + j];
        if (threadIdx.x == 0) { chi2[r] = chi2[W - 1]; y[r] = y[W - 1]; }
    }
}

int ensure_sweep_tables(sail_handle *h, int G)
{
    if (h->tables_G == G) return SAIL_OK;
    const bool fact = (size_t)h->n_omega * G * sizeof(double) > 64 * 1024;
    int shift = 0, n_hi = 0, n_lo = 0;
    if (fact) {
        int bits = 0;
        while ((1 << bits) < h->n_omega) bits++;
        shift = bits / 2;
        n_lo = 1 << shift;
        n_hi = (h->n_omega + n_lo - 1) >> shift;
    }
    h->tables_fact = fact;
    h->fact_shift = shift;
    sweep_tables_kernel<<<64, 256, 0, h->stream>>>(h->n_omega, G, h->domega, h->tau0, h->dtau, h->tab.omega,
                                                   fact ? 1 : 0, shift, n_hi, n_lo, h->sw_ratio, h->sw_invd, h->sw_E0);
    SAIL_LAUNCH_OK(h, "sweep_tables_kernel");
    h->tables_G = G;
    return SAIL_OK;
}

// ---- dispatch -----------------------------------------------------------------------------------------
// MODE 1: lean one walker per warp (sweep_kernel_warp), 4: the same with the index walk of section 2.3,
//      2: screened one walker per warp (sweep_kernel_mask),
//      3: the same with 2 Wj in registers
template <int C, int MAXW, bool FACT, bool TRACE, int MODE, int DMMA = 0>
static int launch_variant(sail_handle *h, SweepArgs &args)
{
    constexpr int G = 32;
    constexpr int rec_bytes = (MODE == 2 || MODE == 3) ? kRecMaskBytes : (MODE == 4) ? 96 : kRecBytes;
    args.n_groups = args.W;
    int warps = (int)((args.n_groups + h->num_sms - 1) / h->num_sms);
    if (warps > MAXW) warps = MAXW;
    if (warps < 1) warps = 1;
    long long ctas = (args.n_groups + warps - 1) / warps;
    if (ctas > h->num_sms) ctas = h->num_sms;
    const int e0_elems = args.fact ? (args.n_hi + args.n_lo) * G : args.n_omega * G;
    const size_t smem = (size_t)(3 * ((args.n_omega + 1) & ~1) + ((e0_elems + 1) & ~1)) * sizeof(double)
                        + (size_t)warps * 32 * rec_bytes;
    if (smem > 227 * 1024)
        return set_err(h, SAIL_ERR_ARG, "sweep tables need %zu bytes of shared memory (> 227 KB)", smem);
    void (*kern)(const SweepArgs);
    if constexpr (MODE == 3) kern = sweep_kernel_mask<C, MAXW, FACT, TRACE, true, DMMA>;
    else if constexpr (MODE == 2) kern = sweep_kernel_mask<C, MAXW, FACT, TRACE, false, DMMA>;
    else if constexpr (MODE == 4) kern = sweep_kernel_warp<C, MAXW, FACT, TRACE, true>;
    else kern = sweep_kernel_warp<C, MAXW, FACT, TRACE, false>;
    SAIL_CUDA_OK(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int resident = 0;
    SAIL_CUDA_OK(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&resident, kern, warps * 32, smem));
    if (resident < 1)
        return set_err(h, SAIL_ERR_CUDA, "sweep kernel (mode %d, C=%d, MAXW=%d) does not fit one SM at %d warps per CTA", MODE, C, MAXW, warps);
    kern<<<(unsigned)ctas, warps * 32, smem, h->stream>>>(args);
    SAIL_LAUNCH_OK(h, "sweep_kernel");
    return SAIL_OK;
}

// lanes_per_walker (a tuning knob, see include/sail.h): 0 / 32 = screened one-walker-per-warp kernel with the DMMA
// warp sum (default), 35 = the same with the other register trade-off, 37 = the same with the shuffle butterfly,
// 34 = the unscreened lean form,
// 8 / 16 = grouped screened kernel (several walkers per warp), 36 = its 32-lane instance
static int pick_lanes(int requested)
{
    if (requested == 8 || requested == 16) return requested;
    return 32;
}

int launch_sweeps(sail_handle *h, const double *d_T, int64_t n_sweeps, const sail_anneal_params *p,
                  int64_t sweeps_in_call, int64_t call_offset)
{
    const int req = p->lanes_per_walker;
    if (!(req == 0 || req == 8 || req == 16 || req == 32 || (req >= 34 && req <= 37)))
        return set_err(h, SAIL_ERR_ARG, "lanes_per_walker=%d is not one of 0, 8, 16, 32, 34..37", req);
    if (p->walk_length < 0 || p->walk_length > 4096) return set_err(h, SAIL_ERR_ARG, "walk_length=%d outside [0, 4096]", p->walk_length);
    if (!(p->walk_uniform >= 0.0 && p->walk_uniform <= 1.0)) return set_err(h, SAIL_ERR_ARG, "walk_uniform must lie in [0, 1]");
    if (p->walk_length > 0 && !(req == 0 || req == 32 || req == 34))
        return set_err(h, SAIL_ERR_ARG, "walk_length > 0 runs on the plain one-walker-per-warp kernel: lanes_per_walker must be 0, 32 or 34");
    const int G = pick_lanes(req);
    // (16 lanes per walker win the first sweeps of Branching, 0.281 against 0.269, but lose over the whole anneal,
    // 0.270 against 0.280: auto stays with one walker per warp)
    const int C = (h->n_tau + G - 1) / G;
    if (C > 16) return set_err(h, SAIL_ERR_ARG, "n_tau=%d needs more than 16 tau-points per lane at %d lanes", h->n_tau, G);
    int rc = ensure_sweep_tables(h, G);
    if (rc) return rc;
    const long long W_pad = (h->W + 3) & ~3LL;
    if ((unsigned long long)W_pad * (unsigned long long)h->n_omega >= (1ull << 32))
        return set_err(h, SAIL_ERR_ARG, "W * n_omega must be < 2^32 spectral coefficients");
    if (W_pad > h->W) {
        pad_walkers_kernel<<<(unsigned)(W_pad - h->W), 128, 0, h->stream>>>(h->n_omega, h->n_tau, h->W, W_pad, h->st.a,
                                                                          h->st.mt, h->st.chi2, h->st.y);
        SAIL_LAUNCH_OK(h, "pad_walkers_kernel");
    }

    SweepArgs a{};
    a.n_omega = h->n_omega; a.n_tau = h->n_tau; a.W = h->W;
    a.A = h->A; a.B = h->B; a.omega_mid0 = h->omega0 + 0.5 * h->domega; a.domega = h->domega; a.eta = p->eta;
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

    // grouped screened kernel (sweep_grp.cu): 8 / 16 lanes per walker, 36 = its one-walker-per-warp instance
    if (a.walk_len == 0 && (req == 8 || req == 16 || req == 36)) return launch_sweep_grp(h, a, G, C, trace, 0);

#define SAIL_VARIANT(CC, MW, MODE)                                                                                  \
    {                                                                                                                   \
        if (a.fact) return trace ? launch_variant<CC, MW, true, true, MODE>(h, a) : launch_variant<CC, MW, true, false, MODE>(h, a);   \
        return trace ? launch_variant<CC, MW, false, true, MODE>(h, a) : launch_variant<CC, MW, false, false, MODE>(h, a);             \
    }
#define SAIL_VARIANT_D(CC, MW, MODE)                                                                                \
    {                                                                                                                   \
        if (a.fact) return trace ? launch_variant<CC, MW, true, true, MODE, 1>(h, a) : launch_variant<CC, MW, true, false, MODE, 1>(h, a);   \
        return trace ? launch_variant<CC, MW, false, true, MODE, 1>(h, a) : launch_variant<CC, MW, false, false, MODE, 1>(h, a);             \
    }
    if (a.walk_len > 0) {                              // index selection by a truncated walk: the plain form only
        if (C <= 4) SAIL_VARIANT(4, 28, 4)
        if (C <= 8) SAIL_VARIANT(8, 16, 4)
        SAIL_VARIANT(16, 12, 4)
    }
    if (req == 0 || req == 32) {                       // screened, DMMA warp sum (default)
        if (C <= 4) SAIL_VARIANT_D(4, 28, 2)
        if (C <= 7) SAIL_VARIANT_D(7, 16, 3)
        if (C <= 8) SAIL_VARIANT_D(8, 16, 3)
        SAIL_VARIANT_D(16, 12, 2)
    }
    if (req == 35) {                                   // the same, the other register trade-off
        if (C <= 4) SAIL_VARIANT_D(4, 24, 3)
        if (C <= 7) SAIL_VARIANT_D(7, 16, 2)
        if (C <= 8) SAIL_VARIANT_D(8, 16, 2)
        SAIL_VARIANT_D(16, 8, 3)
    }
    if (req == 37) {                                   // screened, shuffle-butterfly warp sum
        if (C <= 4) SAIL_VARIANT(4, 28, 2)
        if (C <= 7) SAIL_VARIANT(7, 16, 3)
        if (C <= 8) SAIL_VARIANT(8, 16, 3)
        SAIL_VARIANT(16, 12, 2)
    }
    // req == 34: unscreened lean form
    if (C <= 4) SAIL_VARIANT(4, 28, 1)
    if (C <= 8) SAIL_VARIANT(8, 16, 1)
    SAIL_VARIANT(16, 12, 1)
#undef SAIL_VARIANT
#undef SAIL_VARIANT_D
}

} // namespace sail
