// sweep.cu — the persistent Monte Carlo sweep kernel.
//
// Mapping: G lanes of a warp cooperate on one walker (32/G walkers per warp); lane l
// owns tau-points j = l + G*i, i < C, whose residual state lives in REGISTERS for the whole launch:
//     mt_j  = sum_k a_k exp(-omega_k tau_j)      (model in the pure-exponential basis, M_j = c_j mt_j)
//     G2_j  = 2 Wj (mt_j - fj)                   (Wj = (c_j/sigma_j)^2, fj = F_j/c_j)
// so that for a move (p, s, rho, delta_p, delta_s) (Eq. 17-22):
//     dt_j   = (rho-1) mt_j + delta_p E_pj + delta_s E_sj          E_kj = exp(-omega_k tau_j)
//     dchi2  = sum_j dt_j (Wj dt_j + G2_j)     [= sum_j d_j (d_j + 2 D_j) of SURVEY §8a row A4]
// The kernel rows are never read from a table in the inner loop: both grids are uniform (Eq. 2-3, 7),
// so E_{k,j+G} = E_kj * exp(-omega_k G dtau); each lane starts from E0[k][l] (shared memory) and
// advances by one DMUL per row per tau-point, with delta folded into the start value:
//     6 FP64-pipe instructions per tau-point (2 DMUL, 1 DADD, 3 DFMA), no memory traffic.
// Proposals (Philox4x32-10 keyed by (seed; walker, sweep, move, 0), index draw, rho, Eq. 20-21
// divisions, -T ln u) do not depend on the chain state within a sweep, so they are computed G moves
// at a time, one move per lane, and staged as 64-byte records in shared memory.
// Eq. 19 (scale ALL coefficients by rho) is applied lazily: a = g * a~, g <- g rho on accept, folded
// into a~ at the end of every sweep.
#include "sail_internal.cuh"

namespace sail {

struct SweepArgs {
    int n_omega, n_tau;
    long long W, n_groups;
    double A, B, domega, eta, amp_p, amp_m, y_min;
    int amp_mode;
    uint32_t seed_lo, seed_hi;
    const double *omega, *Wj, *fj, *ratio, *E0;
    int fact, fact_shift, n_hi, n_lo;
    double *a, *mt, *chi2, *y;
    unsigned long long *n_acc, *n_eval;
    const double *T;
    long long sweep0;
    int n_sweeps;
    long long trace_lo, trace_hi;
    sail_trace_rec *trace;
    uint8_t *flags;
    long long call_sweeps, call_off;   // sweeps in the whole sail_anneal call / offset of this launch
};

__device__ __forceinline__ double shfl_xor_f64(double v, int off)
{
    return __shfl_xor_sync(0xffffffffu, v, off);
}

template <int G, int C, int MAXW>
__global__ void __launch_bounds__(MAXW * 32, 1) sweep_kernel(const SweepArgs P)
{
    constexpr int NW = 32 / G;               // walkers per warp
    extern __shared__ __align__(16) unsigned char smem[];
    double *s_ratio = reinterpret_cast<double *>(smem);
    const int n_omega_pad = (P.n_omega + 1) & ~1;
    double *s_E0 = s_ratio + n_omega_pad;
    const int e0_elems = P.fact ? (P.n_hi + P.n_lo) * G : P.n_omega * G;
    unsigned char *s_recs = reinterpret_cast<unsigned char *>(s_E0 + ((e0_elems + 1) & ~1));

    for (int i = threadIdx.x; i < P.n_omega; i += blockDim.x) s_ratio[i] = P.ratio[i];
    for (int i = threadIdx.x; i < e0_elems; i += blockDim.x) s_E0[i] = P.E0[i];
    __syncthreads();

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int sub = lane % G;                // lane within the walker's group
    const int q = lane / G;                  // which walker of the warp
    unsigned char *my_recs = s_recs + (size_t)warp * 32 * kRecBytes;
    const int warps_per_cta = blockDim.x >> 5;
    const long long total_warps = (long long)gridDim.x * warps_per_cta;
    const int n_omega = P.n_omega;
    const double half_dw = 0.5 * P.domega;
    const int fmask = (1 << P.fact_shift) - 1;

    for (long long grp = (long long)blockIdx.x * warps_per_cta + warp; grp < P.n_groups; grp += total_warps) {
        const long long w_raw = grp * NW + q;
        const bool active = w_raw < P.W;
        const long long w = active ? w_raw : P.W - 1;
        double *a_w = P.a + (size_t)w * n_omega;

        // ---- load the walker's residual state into registers --------------------------------------
        double mt[C], G2[C], Wt[C], d[C], fv[C];
#pragma unroll
        for (int i = 0; i < C; ++i) {
            const int j = sub + G * i;
            const bool ok = j < P.n_tau;
            mt[i] = ok ? P.mt[(size_t)w * P.n_tau + j] : 0.0;
            Wt[i] = ok ? P.Wj[j] : 0.0;
            fv[i] = ok ? P.fj[j] : 0.0;
            d[i] = 0.0;
        }
        double chi2 = P.chi2[w];
        double y = P.y[w];
        double g = 1.0, ginv = 1.0;
        unsigned long long tot_acc = 0, tot_eval = 0;
        const bool tracing = P.trace != nullptr && active && w >= P.trace_lo && w < P.trace_hi;

        for (int isw = 0; isw < P.n_sweeps; ++isw) {
            const long long sweep = P.sweep0 + isw;
            const double T = P.T[isw];
            int acc_sweep = 0;
            // G2 is a pure function of mt at every sweep start, so splitting a run into several calls
            // (state round-trips through global memory) reproduces the single-call chain bit for bit
#pragma unroll
            for (int i = 0; i < C; ++i) G2[i] = 2.0 * Wt[i] * (mt[i] - fv[i]);

            for (int m0 = 0; m0 < n_omega; m0 += G) {
                const int nb = min(G, n_omega - m0);
                // ---- proposals for moves m0 .. m0+nb-1, one per lane (row A2) -----------------------
                if (sub < nb) {
                    const int m = m0 + sub;
                    uint32_t x[4];
                    philox4x32_10((uint32_t)w, (uint32_t)sweep, (uint32_t)m, 0u, P.seed_lo, P.seed_hi, x);
                    const int p = (int)__umulhi(x[0], (uint32_t)n_omega);
                    int s = (int)__umulhi(x[1], (uint32_t)(n_omega - 1));
                    s += (s >= p) ? 1 : 0;
                    const double u_rho = ((double)x[2] + 0.5) * 2.3283064365386962890625e-10;
                    const double u_acc = ((double)x[3] + 0.5) * 2.3283064365386962890625e-10;
                    // same operation order as the method's definition, no contraction (bit-stable draws)
                    const double rho = __dsub_rn(1.0, __dmul_rn(__dmul_rn(y, P.eta),
                                                                __dsub_rn(__dmul_rn(2.0, u_rho), 1.0)));
                    const double omr = __dsub_rn(1.0, rho);
                    const double wm_p = __dadd_rn(P.omega[p], half_dw);
                    const double wm_s = __dadd_rn(P.omega[s], half_dw);
                    const double dp = __ddiv_rn(__dmul_rn(omr, __dsub_rn(P.B, __dmul_rn(P.A, wm_s))),
                                                __dmul_rn((double)(p - s), P.domega));     // Eq. 20
                    const double ds = __ddiv_rn(__dmul_rn(omr, __dsub_rn(P.B, __dmul_rn(P.A, wm_p))),
                                                __dmul_rn((double)(s - p), P.domega));     // Eq. 21
                    const double thr = -T * log(u_acc);
                    const double alpha = __dsub_rn(rho, 1.0);
                    unsigned char *r = my_recs + (size_t)lane * kRecBytes;
                    *reinterpret_cast<int4 *>(r) = make_int4(p, s, __double2loint(alpha), __double2hiint(alpha));
                    *reinterpret_cast<double2 *>(r + 16) = make_double2(dp, ds);
                    *reinterpret_cast<double2 *>(r + 32) = make_double2(thr, 1.0 / rho);
                    *reinterpret_cast<double2 *>(r + 48) = make_double2(s_ratio[p], s_ratio[s]);
                }
                __syncwarp();

                // ---- software pipeline: record + spectrum values of the next move are fetched early --
                const unsigned char *rbase = my_recs + (size_t)(q * G) * kRecBytes;
                int4 r0 = *reinterpret_cast<const int4 *>(rbase);
                double ap_t = a_w[r0.x], as_t = a_w[r0.y];

                for (int mm = 0; mm < nb; ++mm) {
                    const unsigned char *r = rbase + (size_t)mm * kRecBytes;
                    const int p = r0.x, s = r0.y;
                    const double alpha = __hiloint2double(r0.w, r0.z);
                    const double2 dd = *reinterpret_cast<const double2 *>(r + 16);
                    const double2 th = *reinterpret_cast<const double2 *>(r + 32);
                    const double2 rr = *reinterpret_cast<const double2 *>(r + 48);
                    const double cap = ap_t, cas = as_t;
                    if (mm + 1 < nb) {
                        r0 = *reinterpret_cast<const int4 *>(r + kRecBytes);
                        ap_t = a_w[r0.x];
                        as_t = a_w[r0.y];
                    }
                    // ---- positivity (row A3) ------------------------------------------
                    const double gn = fma(alpha, g, g);                 // rho * g, exactly rounded
                    const double ap_new = fma(gn, cap, dd.x);           // rho a_p + delta_p
                    const double as_new = fma(gn, cas, dd.y);
                    const bool feas = active && (ap_new >= 0.0) && (as_new >= 0.0);
                    int fl = feas ? 1 : 0;
                    double dchi2 = 0.0;
                    if (__any_sync(0xffffffffu, feas)) {
                        // ---- incremental Delta chi^2 over all tau (row A4, Eq. 22 + Eq. 9) -----------
                        double e0p, e0s;
                        if (P.fact) {
                            e0p = s_E0[(p >> P.fact_shift) * G + sub] * s_E0[(P.n_hi + (p & fmask)) * G + sub];
                            e0s = s_E0[(s >> P.fact_shift) * G + sub] * s_E0[(P.n_hi + (s & fmask)) * G + sub];
                        } else {
                            e0p = s_E0[p * G + sub];
                            e0s = s_E0[s * G + sub];
                        }
                        double ep = dd.x * e0p, es = dd.y * e0s;
                        double acc_a = 0.0, acc_b = 0.0;
#pragma unroll
                        for (int i = 0; i < C; ++i) {
                            const double v = ep + es;
                            d[i] = fma(alpha, mt[i], v);
                            const double t = fma(Wt[i], d[i], G2[i]);
                            if (i & 1) acc_b = fma(d[i], t, acc_b);
                            else       acc_a = fma(d[i], t, acc_a);
                            if (i + 1 < C) { ep *= rr.x; es *= rr.y; }
                        }
                        dchi2 = acc_a + acc_b;
#pragma unroll
                        for (int off = G / 2; off > 0; off >>= 1) dchi2 += shfl_xor_f64(dchi2, off);
                        fl |= 4;
                        // ---- Metropolis (row A5, Eq. 10): accept iff dchi2/T + ln u < 0 --------------
                        const bool acc = feas && (dchi2 < th.x);
                        if (__any_sync(0xffffffffu, acc)) {
                            if (acc) {
#pragma unroll
                                for (int i = 0; i < C; ++i) {
                                    mt[i] += d[i];
                                    G2[i] = fma(Wt[i], d[i] + d[i], G2[i]);
                                }
                                chi2 += dchi2;
                                g = gn;
                                ginv *= th.y;
                                const double ap_store = ap_new * ginv, as_store = as_new * ginv;
                                if (sub == 0) { a_w[p] = ap_store; a_w[s] = as_store; }
                                // the next move's values were fetched before this store
                                if (r0.x == p) ap_t = ap_store; else if (r0.x == s) ap_t = as_store;
                                if (r0.y == p) as_t = ap_store; else if (r0.y == s) as_t = as_store;
                                acc_sweep++;
                                fl |= 2;
                            }
                            __syncwarp();
                        }
                    }
                    tot_eval += feas ? 1 : 0;
                    if (sub == 0 && active) {
                        if (P.flags)
                            P.flags[((size_t)w * P.call_sweeps + P.call_off + isw) * n_omega + m0 + mm] = (uint8_t)fl;
                        if (tracing) {
                            sail_trace_rec *tr = P.trace + (((size_t)(w - P.trace_lo) * P.call_sweeps + P.call_off + isw)
                                                            * n_omega + m0 + mm);
                            tr->p = p; tr->s = s; tr->flags = fl; tr->move = m0 + mm;
                            tr->rho = 1.0 + alpha; tr->delta_p = dd.x; tr->delta_s = dd.y;
                            tr->dchi2 = dchi2; tr->thr = th.x; tr->ap_new = ap_new; tr->as_new = as_new;
                        }
                    }
                }
                __syncwarp();
            }

            // ---- end of sweep: fold the lazy scale (Eq. 19) and update y (row A6, Eq. 30) ------------
            if (active) {
                for (int k = sub; k < n_omega; k += G) a_w[k] *= g;
            }
            g = 1.0;
            ginv = 1.0;
            tot_acc += acc_sweep;
            if (P.amp_mode == 1) {
                const double rate = (double)acc_sweep / (double)n_omega;
                if (rate >= P.amp_p) y = 1.0;
                else {
                    const double x = rate / P.amp_p;
                    const double yy = (P.amp_m == 2.0) ? x * x : pow(x, P.amp_m);
                    y = yy < P.y_min ? P.y_min : yy;
                }
            }
            __syncwarp();
        }

        // ---- store the state back ----------------------------------------------------------------
        if (active) {
#pragma unroll
            for (int i = 0; i < C; ++i) {
                const int j = sub + G * i;
                if (j < P.n_tau) P.mt[(size_t)w * P.n_tau + j] = mt[i];
            }
            if (sub == 0) {
                P.chi2[w] = chi2;
                P.y[w] = y;
                P.n_acc[w] += tot_acc;
                P.n_eval[w] += tot_eval;
            }
        }
        __syncwarp();
    }
}

// ---- sweep tables: ratio[k] = exp(-omega_k G dtau); start values E0 (direct or factored) -------------
__global__ void sweep_tables_kernel(int n_omega, int G, double omega0, double domega, double tau0, double dtau,
                                    const double *omega, int fact, int shift, int n_hi, int n_lo,
                                    double *ratio, double *E0)
{
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int stride = gridDim.x * blockDim.x;
    for (int k = tid; k < n_omega; k += stride) ratio[k] = exp(-omega[k] * ((double)G * dtau));
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
    sweep_tables_kernel<<<64, 256, 0, h->stream>>>(h->n_omega, G, h->omega0, h->domega, h->tau0, h->dtau,
                                                   h->tab.omega, fact ? 1 : 0, shift, n_hi, n_lo,
                                                   h->sw_ratio, h->sw_E0);
    SAIL_LAUNCH_OK(h, "sweep_tables_kernel");
    h->tables_G = G;
    return SAIL_OK;
}

// ---- dispatch -----------------------------------------------------------------------------------------
template <int G, int C, int MAXW>
static int launch_variant(sail_handle *h, SweepArgs &args)
{
    constexpr int NW = 32 / G;
    args.n_groups = (args.W + NW - 1) / NW;
    int warps = (int)((args.n_groups + h->num_sms - 1) / h->num_sms);
    if (warps > MAXW) warps = MAXW;
    if (warps < 1) warps = 1;
    long long ctas = (args.n_groups + warps - 1) / warps;
    if (ctas > h->num_sms) ctas = h->num_sms;
    const int e0_elems = args.fact ? (args.n_hi + args.n_lo) * G : args.n_omega * G;
    const size_t smem = (size_t)(((args.n_omega + 1) & ~1) + ((e0_elems + 1) & ~1)) * sizeof(double)
                        + (size_t)warps * 32 * kRecBytes;
    if (smem > 227 * 1024)
        return set_err(h, SAIL_ERR_ARG, "sweep tables need %zu bytes of shared memory (> 227 KB)", smem);
    auto kern = sweep_kernel<G, C, MAXW>;
    SAIL_CUDA_OK(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<(unsigned)ctas, warps * 32, smem, h->stream>>>(args);
    SAIL_LAUNCH_OK(h, "sweep_kernel");
    return SAIL_OK;
}

static int pick_lanes(const sail_handle *h, int requested)
{
    if (requested == 8 || requested == 16 || requested == 32) return requested;
    // auto: fewest lanes per walker that (a) keep <= 16 tau-points per lane and (b) still leave
    // enough warps to fill every SM sub-partition several times over
    for (int G = 8; G <= 32; G *= 2) {
        const int C = (h->n_tau + G - 1) / G;
        const long long warps = (h->W * G + 31) / 32;
        if (C <= 16 && warps >= (long long)h->num_sms * 24) return G;
    }
    return 32;
}

int launch_sweeps(sail_handle *h, const double *d_T, int64_t n_sweeps, const sail_anneal_params *p,
                  int64_t sweeps_in_call, int64_t call_offset)
{
    const int G = pick_lanes(h, p->lanes_per_walker);
    const int C = (h->n_tau + G - 1) / G;
    if (C > 16) return set_err(h, SAIL_ERR_ARG, "n_tau=%d needs more than 16 tau-points per lane at %d lanes", h->n_tau, G);
    int rc = ensure_sweep_tables(h, G);
    if (rc) return rc;

    SweepArgs a{};
    a.n_omega = h->n_omega; a.n_tau = h->n_tau; a.W = h->W;
    a.A = h->A; a.B = h->B; a.domega = h->domega; a.eta = p->eta;
    a.amp_p = p->amp_p; a.amp_m = p->amp_m; a.y_min = p->y_min; a.amp_mode = p->amp_mode;
    a.seed_lo = (uint32_t)(h->seed & 0xFFFFFFFFu); a.seed_hi = (uint32_t)(h->seed >> 32);
    a.omega = h->tab.omega; a.Wj = h->tab.Wj; a.fj = h->tab.fj; a.ratio = h->sw_ratio; a.E0 = h->sw_E0;
    a.fact = h->tables_fact ? 1 : 0; a.fact_shift = h->fact_shift;
    if (h->tables_fact) { a.n_lo = 1 << h->fact_shift; a.n_hi = (h->n_omega + a.n_lo - 1) >> h->fact_shift; }
    a.a = h->st.a; a.mt = h->st.mt; a.chi2 = h->st.chi2; a.y = h->st.y;
    a.n_acc = h->st.n_acc; a.n_eval = h->st.n_eval;
    a.T = d_T; a.sweep0 = h->sweep; a.n_sweeps = (int)n_sweeps;
    a.trace_lo = p->trace_lo; a.trace_hi = p->trace_hi; a.trace = p->trace; a.flags = p->flags;
    a.call_sweeps = sweeps_in_call; a.call_off = call_offset;

#define SAIL_VARIANT(GG, CC, MW) if (G == GG && C <= CC) return launch_variant<GG, CC, MW>(h, a);
    SAIL_VARIANT(32, 1, 28) SAIL_VARIANT(32, 2, 28) SAIL_VARIANT(32, 4, 28)
    SAIL_VARIANT(32, 7, 16) SAIL_VARIANT(32, 8, 16) SAIL_VARIANT(32, 16, 10)
    SAIL_VARIANT(16, 2, 28) SAIL_VARIANT(16, 4, 28) SAIL_VARIANT(16, 7, 16)
    SAIL_VARIANT(16, 8, 16) SAIL_VARIANT(16, 13, 10) SAIL_VARIANT(16, 16, 10)
    SAIL_VARIANT(8, 4, 28) SAIL_VARIANT(8, 8, 16) SAIL_VARIANT(8, 13, 10) SAIL_VARIANT(8, 16, 10)
#undef SAIL_VARIANT
    return set_err(h, SAIL_ERR_ARG, "no sweep kernel variant for lanes=%d, tau-points per lane=%d", G, C);
}

} // namespace sail
