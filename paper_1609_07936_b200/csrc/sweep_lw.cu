// sweep_lw.cu — the "lane per walker" sweep kernel.
//
// The same moves, decisions and per-tau-point arithmetic as sweep_kernel_mask (sweep.cu), with the warp turned
// round: a CTA owns 32 walkers, LANE l of every warp belongs to walker l, and WARP s of the CTA owns the tau-slice
// j = s CS .. s CS + CS - 1 of all 32 residual vectors (registers).  Everything that is per-move scalar work in the
// one-walker-per-warp form — the record, the start values, the sum over tau, the Metropolis decision — is now
// done for 32 walkers by one instruction:
//   * proposals (row A2) are generated ahead, 8 moves per walker per round (warp s < 8 makes move gen + s of its
//     lane's walker), into a per-walker ring of LW_Q entries in shared memory; they depend on the chain only
//     through y, which is fixed within a sweep;
//   * positivity (row A3): warps 0..3 test the next four queued moves of every walker against its current spectrum;
//     the first feasible one is the walker's move of this step, the ones before it are rejected for good;
//   * Delta chi^2 (row A4): every warp runs the tau loop over its slice for all 32 walkers (5 FP64 per tau-point,
//     two-term recurrence for delta_p E_p + delta_s E_s along the slice, start values gathered from a
//     [slice][omega] table), partial sums meet in shared memory and are added in a fixed tree order;
//   * Metropolis (row A5) per lane; the residual update is selected per lane, not branched.
// Walkers of a CTA finish a sweep together (a walker that is through its N_omega moves idles until the others are).
#include "sweep_common.cuh"

namespace sail {

constexpr int LW_Q = 16;            // ring entries per walker (power of two)
constexpr int LW_GEN = 8;           // moves generated per walker per refill round (warps 0 .. LW_GEN-1)
constexpr int LW_SCR = 4;           // queued moves screened per walker per step (warps 0 .. LW_SCR-1)
constexpr int LW_MAXTAU = 256;      // S * CS <= 256
// ring fields (each [LW_Q][32] doubles): 0 (p, s) as int2, 1 alpha = rho - 1, 2 delta_p, 3 delta_s,
// 4 delta_p r_p, 5 delta_s r_s, 6 r_p + r_s, 7 -(r_p r_s), 8 thr = -T ln u, 9 1/rho       (r_k = exp(-omega_k dtau))
constexpr int LW_NF = 10;

struct LwArgs {
    SweepArgs a;
    const double *etab;             // [S][n_omega]: exp(-omega_k tau_{s CS})
    const double *ratio1;           // [n_omega]:    exp(-omega_k dtau)
    double Wj[LW_MAXTAU];           // (c_j / sigma_j)^2, zero beyond n_tau
    double W2j[LW_MAXTAU];          // 2 Wj
    double fj[LW_MAXTAU];
};

__global__ void lw_tables_kernel(int n_omega, int S, int CS, double tau0, double dtau, const double *omega,
                                 double *ratio1, double *invd, double domega, double *etab)
{
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int stride = gridDim.x * blockDim.x;
    for (int k = tid; k < n_omega; k += stride) {
        ratio1[k] = exp(-omega[k] * dtau);
        invd[k] = k ? 1.0 / ((double)k * domega) : 0.0;
    }
    for (int i = tid; i < S * n_omega; i += stride) {
        const int s = i / n_omega, k = i % n_omega;
        etab[i] = exp(-omega[k] * (tau0 + (double)(s * CS) * dtau));
    }
}

__device__ __forceinline__ uint32_t lw_ring(uint32_t ring, int field, int slot, int lane)
{
    return ring + (uint32_t)(((field * LW_Q + slot) * 32 + lane) * 8);
}
__device__ __forceinline__ void sts_f64(uint32_t addr, double v)
{
    asm volatile("st.shared.f64 [%0], %1;" :: "r"(addr), "d"(v) : "memory");
}
__device__ __forceinline__ double lds_f64m(uint32_t addr)          // with a memory clobber: ordered against barriers
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr) : "memory");
    return v;
}

// one proposal (row A2) of walker `walker`, written into ring slot `slot` of lane `lane`
__device__ __forceinline__ void lw_propose(const SweepArgs &P, uint32_t walker, uint32_t sweep, uint32_t move, double y, double T,
                                           const double *s_ratio, const double *s_invd, const double *s_wm,
                                           uint32_t ring, int slot, int lane)
{
    uint32_t x[4];
    philox4x32_10(walker, sweep, move, 0u, P.seed_lo, P.seed_hi, x);
    const int p = (int)__umulhi(x[0], (uint32_t)P.n_omega);
    int s = (int)__umulhi(x[1], (uint32_t)(P.n_omega - 1));
    s += (s >= p) ? 1 : 0;
    const double u_rho = ((double)x[2] + 0.5) * 2.3283064365386962890625e-10;
    const double u_acc = ((double)x[3] + 0.5) * 2.3283064365386962890625e-10;
    const double rho = __dsub_rn(1.0, __dmul_rn(__dmul_rn(y, P.eta), __dsub_rn(__dmul_rn(2.0, u_rho), 1.0)));
    const double alpha = __dsub_rn(rho, 1.0);
    const double omr = __dsub_rn(1.0, rho);
    const int dps = p - s;
    const double inv = (dps > 0) ? s_invd[dps] : -s_invd[-dps];
    const double dp = __dmul_rn(__dmul_rn(omr, __dsub_rn(P.B, __dmul_rn(P.A, s_wm[s]))), inv);
    const double ds = -__dmul_rn(__dmul_rn(omr, __dsub_rn(P.B, __dmul_rn(P.A, s_wm[p]))), inv);
    const double thr = -T * log(u_acc);
    const double rp = s_ratio[p], rs = s_ratio[s];
    sts_f64(lw_ring(ring, 0, slot, lane), __hiloint2double(s, p));
    sts_f64(lw_ring(ring, 1, slot, lane), alpha);
    sts_f64(lw_ring(ring, 2, slot, lane), dp);
    sts_f64(lw_ring(ring, 3, slot, lane), ds);
    sts_f64(lw_ring(ring, 4, slot, lane), dp * rp);
    sts_f64(lw_ring(ring, 5, slot, lane), ds * rs);
    sts_f64(lw_ring(ring, 6, slot, lane), rp + rs);
    sts_f64(lw_ring(ring, 7, slot, lane), -(rp * rs));
    sts_f64(lw_ring(ring, 8, slot, lane), thr);
    sts_f64(lw_ring(ring, 9, slot, lane), fast_recip(rho));
}

template <int S, int CS, bool TRACE>
__global__ void __launch_bounds__(S * 32, 1) sweep_kernel_lw(const __grid_constant__ LwArgs A)
{
    static_assert(S >= LW_GEN && S >= LW_SCR && (S & (S - 1)) == 0 && S * CS <= LW_MAXTAU, "slice layout");
    const SweepArgs &P = A.a;
    extern __shared__ __align__(16) unsigned char smem[];
    const int n_omega = P.n_omega;
    const int n_omega_pad = (n_omega + 1) & ~1;
    double *s_ratio = reinterpret_cast<double *>(smem);
    double *s_invd = s_ratio + n_omega_pad;
    double *s_wm = s_invd + n_omega_pad;
    double *s_etab = s_wm + n_omega_pad;                         // [S][n_omega]
    double *s_ring = s_etab + (size_t)S * n_omega;               // [LW_NF][LW_Q][32]
    double *s_part = s_ring + LW_NF * LW_Q * 32;                 // [S][32] partial sums of the step
    double *s_xbuf = s_part + S * 32;                            // [LW_SCR][2][32] screened new coefficients
    double *s_gbuf = s_xbuf + LW_SCR * 2 * 32;                   // [32] lazy scale of each walker at sweep end
    uint32_t *s_fb = reinterpret_cast<uint32_t *>(s_gbuf + 32);  // [32] four feasibility bytes per walker
    uint32_t *s_accf = s_fb + 32;                                // [32] Metropolis decision per walker
    for (int i = threadIdx.x; i < n_omega; i += blockDim.x) {
        s_ratio[i] = A.ratio1[i]; s_invd[i] = P.invd[i]; s_wm[i] = __dadd_rn(P.omega[i], 0.5 * P.domega);
    }
    for (int i = threadIdx.x; i < S * n_omega; i += blockDim.x) s_etab[i] = A.etab[i];
    for (int i = threadIdx.x; i < LW_NF * LW_Q * 32; i += blockDim.x) s_ring[i] = 0.0;
    __syncthreads();

    const int lane = threadIdx.x & 31;
    const int s = threadIdx.x >> 5;                              // warp = tau-slice
    const int j0 = s * CS;
    const uint32_t ring = (uint32_t)__cvta_generic_to_shared(s_ring);
    const uint32_t part = (uint32_t)__cvta_generic_to_shared(s_part);
    const uint32_t xbuf = (uint32_t)__cvta_generic_to_shared(s_xbuf);
    const uint32_t etab_s = (uint32_t)__cvta_generic_to_shared(s_etab) + (uint32_t)(s * n_omega * 8);
    constexpr unsigned FULL = 0xffffffffu;

    for (long long grp = blockIdx.x; grp < P.n_groups; grp += gridDim.x) {
        const long long w = grp * 32 + lane;
        const bool wvalid = w < P.W;
        const long long wc = wvalid ? w : P.W - 1;               // lanes beyond W address the last walker, never store
        const uint32_t wbase = (uint32_t)(wc * n_omega);
        double *const a_all = P.a;
        double mt[CS], G2[CS], d[CS];
#pragma unroll
        for (int i = 0; i < CS; ++i) {
            const int j = j0 + i;
            mt[i] = (j < P.n_tau) ? P.mt[(size_t)wc * P.n_tau + j] : 0.0;
            d[i] = 0.0;
        }
        double chi2 = P.chi2[wc];
        double y = P.y[wc];
        double g = 1.0, ginv = 1.0;
        unsigned long long acc_tot = 0ull, eval_tot = 0ull;
        bool tracing = false;
        if (TRACE) tracing = P.trace != nullptr && w >= P.trace_lo && w < P.trace_hi;
        auto trace_write = [&](int isw, int move, int p, int sidx, double alpha, double dp, double ds, double thr,
                               double xp, double xs, int fl, double dchi2) {
            const size_t mvi = ((size_t)(P.call_off + isw)) * n_omega + move;
            if (P.flags) P.flags[(size_t)w * P.call_sweeps * n_omega + mvi] = (uint8_t)fl;
            if (tracing) {
                sail_trace_rec *tr = P.trace + ((size_t)(w - P.trace_lo) * P.call_sweeps * n_omega + mvi);
                tr->p = p; tr->s = sidx; tr->flags = fl; tr->move = move;
                tr->rho = 1.0 + alpha; tr->delta_p = dp; tr->delta_s = ds;
                tr->dchi2 = dchi2; tr->thr = thr; tr->ap_new = xp; tr->as_new = xs;
            }
        };

        for (int isw = 0; isw < P.n_sweeps; ++isw) {
#pragma unroll
            for (int i = 0; i < CS; ++i) G2[i] = A.W2j[j0 + i] * (mt[i] - A.fj[j0 + i]);
            const double T_sweep = P.T[isw];
            const uint32_t sweep = (uint32_t)(P.sweep0 + isw);
            int cur = wvalid ? 0 : n_omega;                      // next move of this walker's sweep
            int gen = cur;                                       // moves proposed so far (ring holds [cur, gen))
            int acc_sweep = 0, eval_sweep = 0;

            while (true) {
                // ---- refill the ring (row A2): a round makes LW_GEN moves for every walker that has room --------
                const bool want = (gen - cur < LW_SCR) && (gen < n_omega);
                if (__any_sync(FULL, want)) {                    // identical in every warp of the CTA
                    const bool room = (gen - cur <= LW_Q - LW_GEN) && (gen < n_omega);
                    if (s < LW_GEN) {
                        const int n = gen + s;
                        if (room && n < n_omega)
                            lw_propose(P, (uint32_t)w, sweep, (uint32_t)n, y, T_sweep, s_ratio, s_invd, s_wm, ring, n & (LW_Q - 1), lane);
                    }
                    if (room) gen = min(gen + LW_GEN, n_omega);
                    __syncthreads();
                }
                const bool pend = cur < n_omega;
                if (!__any_sync(FULL, pend)) break;
                const int navail = min(LW_SCR, gen - cur);       // >= 1 for a pending walker

                // ---- positivity screen (row A3): warp s tests queued move cur + s ------------------
                int q_p = 0, q_s = 0;
                double q_alpha = 0.0, q_dp = 0.0, q_ds = 0.0, q_xp = 0.0, q_xs = 0.0;
                if (s < LW_SCR) {
                    const int slot = (cur + s) & (LW_Q - 1);
                    const double ps = lds_f64m(lw_ring(ring, 0, slot, lane));
                    q_p = __double2loint(ps); q_s = __double2hiint(ps);
                    q_alpha = lds_f64m(lw_ring(ring, 1, slot, lane));
                    q_dp = lds_f64m(lw_ring(ring, 2, slot, lane));
                    q_ds = lds_f64m(lw_ring(ring, 3, slot, lane));
                    const double a_p = ldg_f64(elem_ptr(a_all, wbase + (uint32_t)q_p));
                    const double a_s = ldg_f64(elem_ptr(a_all, wbase + (uint32_t)q_s));
                    const double gn = fma(q_alpha, g, g);
                    q_xp = fma(gn, a_p, q_dp);
                    q_xs = fma(gn, a_s, q_ds);
                    const bool feas = pend && s < navail && ((__double2hiint(q_xp) | __double2hiint(q_xs)) >= 0);
                    reinterpret_cast<volatile uint8_t *>(s_fb)[lane * 4 + s] = feas ? 1 : 0;
                    sts_f64(xbuf + (uint32_t)(((s * 2 + 0) * 32 + lane) * 8), q_xp);
                    sts_f64(xbuf + (uint32_t)(((s * 2 + 1) * 32 + lane) * 8), q_xs);
                }
                __syncthreads();                                 // B1: feasibility bytes and new coefficients

                // ---- the walker's move of this step: its first feasible queued move --------------------------------
                const uint32_t fw = reinterpret_cast<volatile uint32_t *>(s_fb)[lane];
                const bool act = fw != 0u;
                const int cidx = act ? ((__ffs((int)fw) - 1) >> 3) : navail;   // queued moves rejected before it
                if (TRACE) {
                    if (s < LW_SCR && pend && s < navail && s < cidx && wvalid)
                        trace_write(isw, cur + s, q_p, q_s, q_alpha, q_dp, q_ds,
                                    lds_f64m(lw_ring(ring, 8, (cur + s) & (LW_Q - 1), lane)), q_xp, q_xs, 0, 0.0);
                }
                const int mv = cur + (act ? cidx : 0);
                const int slot = mv & (LW_Q - 1);
                const double ps = lds_f64m(lw_ring(ring, 0, slot, lane));
                const int p = __double2loint(ps), sidx = __double2hiint(ps);
                const double alpha = lds_f64m(lw_ring(ring, 1, slot, lane));
                const double dp = lds_f64m(lw_ring(ring, 2, slot, lane));
                const double ds = lds_f64m(lw_ring(ring, 3, slot, lane));
                const double dpr = lds_f64m(lw_ring(ring, 4, slot, lane));
                const double dsr = lds_f64m(lw_ring(ring, 5, slot, lane));
                const double scx = lds_f64m(lw_ring(ring, 6, slot, lane));
                const double scy = lds_f64m(lw_ring(ring, 7, slot, lane));
                const double e0p = lds_f64m(etab_s + (uint32_t)(p * 8));
                const double e0s = lds_f64m(etab_s + (uint32_t)(sidx * 8));
                double thr = 0.0, rinv = 1.0, xpc = 0.0, xsc = 0.0;
                if (s < LW_SCR) {                                // the warps that decide and store
                    thr = lds_f64m(lw_ring(ring, 8, slot, lane));
                    rinv = lds_f64m(lw_ring(ring, 9, slot, lane));
                    const int cc = min(cidx, LW_SCR - 1);
                    xpc = lds_f64m(xbuf + (uint32_t)(((cc * 2 + 0) * 32 + lane) * 8));
                    xsc = lds_f64m(xbuf + (uint32_t)(((cc * 2 + 1) * 32 + lane) * 8));
                }
                // ---- incremental Delta chi^2 over this warp's tau-slice (row A4, Eq. 22 + Eq. 9) ---------------------
                double vm = fma(dp, e0p, ds * e0s);              // v at the first tau-point of the slice
                double vc = fma(dpr, e0p, dsr * e0s);            // ... and at the second
                double acc_a = 0.0, acc_b = 0.0;
#pragma unroll
                for (int i = 0; i < CS; ++i) {
                    double vi;
                    if (i == 0) vi = vm;
                    else if (i == 1) vi = vc;
                    else { vi = fma(scx, vc, scy * vm); vm = vc; vc = vi; }
                    d[i] = fma(alpha, mt[i], vi);
                    const double t = fma(A.Wj[j0 + i], d[i], G2[i]);
                    if (i & 1) acc_b = fma(d[i], t, acc_b);
                    else       acc_a = fma(d[i], t, acc_a);
                }
                sts_f64(part + (uint32_t)((s * 32 + lane) * 8), (CS > 1) ? acc_a + acc_b : acc_a);
                __syncthreads();                                 // B2: partial sums

                // ---- sum over the slices in a fixed tree order; Metropolis (row A5, Eq. 10) per walker ---------------
                bool acc = false;
                double dchi2 = 0.0;
                if (s < LW_SCR) {
                    double v[S];
#pragma unroll
                    for (int q = 0; q < S; ++q) v[q] = lds_f64m(part + (uint32_t)((q * 32 + lane) * 8));
#pragma unroll
                    for (int h = S / 2; h > 0; h >>= 1) {
#pragma unroll
                        for (int q = 0; q < h; ++q) v[q] += v[q + h];
                    }
                    dchi2 = v[0];
                    acc = act && (dchi2 < thr);
                    if (s == 0) reinterpret_cast<volatile uint32_t *>(s_accf)[lane] = acc ? 1u : 0u;
                }
                __syncthreads();                                 // B3: decisions
                if (s >= LW_SCR) acc = reinterpret_cast<volatile uint32_t *>(s_accf)[lane] != 0u;
                if (__any_sync(FULL, acc)) {
#pragma unroll
                    for (int i = 0; i < CS; ++i) {
                        const double dsel = acc ? d[i] : 0.0;
                        mt[i] += dsel;
                        G2[i] = fma(A.W2j[j0 + i], dsel, G2[i]);
                    }
                }
                if (s < LW_SCR && acc) {                         // every screening warp keeps its own view of a, g
                    g = fma(alpha, g, g);
                    ginv *= rinv;
                    if (wvalid) {
                        *elem_ptr(a_all, wbase + (uint32_t)p) = xpc * ginv;
                        *elem_ptr(a_all, wbase + (uint32_t)sidx) = xsc * ginv;
                    }
                }
                if (s == 0) {
                    if (acc) chi2 += dchi2;
                    if (TRACE) { if (act && wvalid) trace_write(isw, mv, p, sidx, alpha, dp, ds, thr, xpc, xsc, 5 | (acc ? 2 : 0), dchi2); }
                }
                acc_sweep += acc ? 1 : 0;
                eval_sweep += act ? 1 : 0;
                cur = act ? cur + cidx + 1 : cur + navail;
            }

            // ---- end of sweep: fold the lazy scale (Eq. 19) with coalesced rows, counters, y (row A6, Eq. 30) ----
            if (s == 0) s_gbuf[lane] = g;
            __syncthreads();
            for (int q = s; q < 32; q += S) {
                const long long ww = grp * 32 + q;
                if (ww < P.W) {
                    const double gq = s_gbuf[q];
                    for (int k = lane; k < n_omega; k += 32) a_all[(size_t)ww * n_omega + k] *= gq;
                }
            }
            g = 1.0;
            ginv = 1.0;
            y = amp_factor(P, acc_sweep, y);
            acc_tot += (unsigned long long)acc_sweep;
            eval_tot += (unsigned long long)eval_sweep;
            __syncthreads();
        }
        if (wvalid) {
#pragma unroll
            for (int i = 0; i < CS; ++i) {
                const int j = j0 + i;
                if (j < P.n_tau) P.mt[(size_t)w * P.n_tau + j] = mt[i];
            }
            if (s == 0) {
                P.chi2[w] = chi2;
                P.y[w] = y;
                P.n_acc[w] += acc_tot;
                P.n_eval[w] += eval_tot;
            }
        }
        __syncthreads();
    }
}

template <int S, int CS, bool TRACE>
static int launch_lw_variant(sail_handle *h, LwArgs &A)
{
    SweepArgs &a = A.a;
    const int key = -(S * 1000 + CS);                            // sweep tables of this slice layout
    if (h->tables_G != key) {
        lw_tables_kernel<<<64, 256, 0, h->stream>>>(h->n_omega, S, CS, h->tau0, h->dtau, h->tab.omega, h->sw_ratio, h->sw_invd,
                                                    h->domega, h->sw_E0);
        SAIL_LAUNCH_OK(h, "lw_tables_kernel");
        h->tables_G = key;
    }
    A.etab = h->sw_E0; A.ratio1 = h->sw_ratio;
    a.n_groups = (a.W + 31) / 32;
    const size_t smem = (size_t)(3 * ((a.n_omega + 1) & ~1) + S * a.n_omega + LW_NF * LW_Q * 32 + S * 32 + LW_SCR * 2 * 32 + 32) * sizeof(double)
                        + 64 * sizeof(uint32_t);
    if (smem > 227 * 1024)
        return set_err(h, SAIL_ERR_ARG, "lane-per-walker sweep kernel needs %zu bytes of shared memory (> 227 KB)", smem);
    void (*kern)(const LwArgs) = sweep_kernel_lw<S, CS, TRACE>;
    SAIL_CUDA_OK(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    long long ctas = a.n_groups < h->num_sms ? a.n_groups : h->num_sms;
    kern<<<(unsigned)ctas, S * 32, smem, h->stream>>>(A);
    SAIL_LAUNCH_OK(h, "sweep_kernel_lw");
    return SAIL_OK;
}

// lanes_per_walker == 1.  Host copies of Wj, fj travel as kernel parameters (constant bank): every warp reads the
// weights of its own tau-slice with a warp-uniform index.
int launch_sweep_lw(sail_handle *h, SweepArgs &a, bool trace, const double *h_Wj, const double *h_fj)
{
    if (a.n_tau > LW_MAXTAU)
        return set_err(h, SAIL_ERR_ARG, "lanes_per_walker=1 supports n_tau <= %d (n_tau=%d)", LW_MAXTAU, a.n_tau);
    if ((size_t)16 * a.n_omega > 16384)
        return set_err(h, SAIL_ERR_ARG, "lanes_per_walker=1 supports n_omega <= 1024 (n_omega=%d)", a.n_omega);
    static thread_local LwArgs A;
    A.a = a;
    for (int j = 0; j < LW_MAXTAU; ++j) {
        A.Wj[j] = j < a.n_tau ? h_Wj[j] : 0.0;
        A.W2j[j] = 2.0 * A.Wj[j];
        A.fj[j] = j < a.n_tau ? h_fj[j] : 0.0;
    }
    const int CS = (a.n_tau + 15) / 16;
#define SAIL_LW(SS, CC) return trace ? launch_lw_variant<SS, CC, true>(h, A) : launch_lw_variant<SS, CC, false>(h, A);
    if (CS <= 2) SAIL_LW(16, 2)
    if (CS <= 7) SAIL_LW(16, 7)
    if (CS <= 13) SAIL_LW(16, 13)
    SAIL_LW(16, 16)
#undef SAIL_LW
}

} // namespace sail
