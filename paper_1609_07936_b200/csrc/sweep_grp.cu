// sweep_grp.cu — the grouped screened sweep kernel.
//
// Same moves, same decisions and the same arithmetic per tau-point as sweep_kernel_mask (sweep.cu); what changes
// is how a warp is shared.  G lanes (8, 16 or 32) cooperate on one walker, so a warp carries NW = 32/G walkers
// whose Markov chains advance in LOCKSTEP, one feasible move of every walker per step:
//   * one FP64 / shared-memory / shuffle instruction serves NW walkers, the reduction has log2(G) stages, and
//     tau-grids that are not a multiple of 32 waste fewer lanes (N_tau = 100: 16 x 7 = 112 slots, not 128);
//   * a batch is G moves per walker, ONE PER LANE: the lane keeps its own move (p, s, rho - 1, delta_p, delta_s)
//     in registers and screens it for positivity (row A3) against the walker's current spectrum; one ballot
//     gives the warp-uniform mask of feasible pending moves of all walkers, from which every group takes its
//     lowest bit.  Only an accepted move changes a spectrum, so only then is the screen repeated;
//   * Metropolis decisions (row A5) are per group: the updates are predicated, not branched.
// A walker whose batch is exhausted idles until the slowest walker of the warp finishes its batch (the price
// of lockstep proposals: ~10 % of the steps at G = 16).
#include "sweep_common.cuh"

namespace sail {

template <int G> __device__ __forceinline__ uint32_t clear_lowest_per_group(uint32_t b)
{
    if (G == 32) return b & (b - 1u);
    uint32_t out = 0u;
#pragma unroll
    for (int q = 0; q < 32 / G; ++q) {
        const uint32_t m = b & (((G == 32) ? 0xffffffffu : ((1u << G) - 1u)) << (q * G));
        out |= m & (m - 1u);
    }
    return out;
}

template <int G, int C, int MAXW, bool FACT, bool TRACE, bool W2REG>
__global__ void __maxnreg__(((65536 / (((MAXW + 3) & ~3) * 32)) & ~7) > 255 ? 255 : ((65536 / (((MAXW + 3) & ~3) * 32)) & ~7))
sweep_kernel_grp(const SweepArgs P)
{
    constexpr int NW = 32 / G;
    constexpr uint32_t GM = (G == 32) ? 0xffffffffu : ((1u << G) - 1u);
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
    // a group with no feasible move left reads record G-1 of its batch (and ignores the result): keep it defined
    for (int i = threadIdx.x; i < (int)(blockDim.x * (kRecMaskBytes / 4)); i += blockDim.x)
        reinterpret_cast<uint32_t *>(s_recs)[i] = 0u;
    __syncthreads();

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int sub = lane & (G - 1);          // lane within the walker's group = tau offset = move slot of the batch
    const int q = lane / G;                  // which walker of the warp
    const int gshift = q * G;
    unsigned char *my_rec_w = s_recs + ((size_t)warp * 32 + lane) * kRecMaskBytes;
    uint32_t rbase = (uint32_t)__cvta_generic_to_shared(s_recs) + (uint32_t)((warp * 32 + q * G) * kRecMaskBytes);
    uint32_t e0_lane = (uint32_t)__cvta_generic_to_shared(s_E0) + (uint32_t)(sub * 8);
    asm volatile("" : "+r"(rbase), "+r"(e0_lane));
    const uint32_t e0_lo = e0_lane + (uint32_t)(P.n_hi * G * 8);
    const int warps_per_cta = blockDim.x >> 5;
    const int fshift = P.fact_shift;
    const int fmask = (1 << fshift) - 1;

    for (long long grp = (long long)blockIdx.x * warps_per_cta + warp; grp < P.n_groups; grp += (long long)gridDim.x * warps_per_cta) {
        const long long w = grp * NW + q;                          // < W_pad: always a valid slot
        uint32_t wbase = (uint32_t)(w * n_omega);
        asm volatile("" : "+r"(wbase));
        double *const a_all = P.a;
        double mt[C], G2[C], Wt[C], d[C], W2[W2REG ? C : 1];
#pragma unroll
        for (int i = 0; i < C; ++i) {
            const int j = sub + G * i;
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
                const int j = sub + G * i;
                const double f = (j < P.n_tau) ? P.fj[j] : 0.0;
                G2[i] = 2.0 * Wt[i] * (mt[i] - f);
            }
            const double y_sweep = P.y[w];
            const double T_sweep = P.T[isw];
            for (int m0 = 0; m0 < n_omega; m0 += G) {
                // ---- proposals (row A2): move m0 + sub of this lane's walker ------------------------------------
                const bool valid = m0 + sub < n_omega;
                MoveRegs mv{0, 0, 0.0, 0.0, 0.0};
                if (valid)
                    mv = propose_mask(P, (uint32_t)w, (uint32_t)(P.sweep0 + isw), (uint32_t)(m0 + sub), y_sweep, T_sweep,
                                      s_ratio, s_invd, s_wm, my_rec_w);
                __syncwarp();
                double *const my_pp = elem_ptr(a_all, wbase + (uint32_t)mv.p);
                double *const my_ps = elem_ptr(a_all, wbase + (uint32_t)mv.s);

                // ---- positivity screen (row A3) of this lane's move -----------------------------
                int mlast = -1;                       // last move of this walker's batch that had its turn
                double xp = 0.0, xs = 0.0;            // rho a_p + delta_p, rho a_s + delta_s at this lane's turn
                auto screen = [&]() -> uint32_t {
                    const double a_p = ldg_f64(my_pp), a_s = ldg_f64(my_ps);
                    const double gn = fma(mv.alpha, g, g);
                    const double x_p = fma(gn, a_p, mv.dp);
                    const double x_s = fma(gn, a_s, mv.ds);
                    const bool pend = valid && sub > mlast;
                    if (pend) { xp = x_p; xs = x_s; }
                    const bool feas = pend && ((__double2hiint(x_p) | __double2hiint(x_s)) >= 0);
                    return __ballot_sync(0xffffffffu, feas);
                };
                uint32_t ball = screen();             // warp-uniform: feasible pending moves of all NW walkers
                int tr_fl = 0;                        // TRACE: bit 1 accepted, bit 2 evaluated (this lane's move)
                double tr_dchi2 = 0.0;

                while (ball) {
                    const uint32_t gm = (ball >> gshift) & GM;
                    const bool active = gm != 0u;
                    const int m = (__ffs((int)gm) - 1) & (G - 1);
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
                    // ---- incremental Delta chi^2 over all tau (row A4, Eq. 22 + Eq. 9) ---------------------------
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
                    dchi2 = group_sum_dmma<G>(dchi2);         // sum over this walker's G lanes, no shuffles
                    // ---- Metropolis (row A5, Eq. 10), per walker ---------------------------------------------------
                    const bool acc = active && (dchi2 < th.x);
                    const int ia = acc ? 1 : 0;
                    eval_sweep += active ? 1 : 0;
                    if (TRACE) { if (active && sub == m) { tr_fl = 4 | (ia << 1); tr_dchi2 = dchi2; } }
                    mlast = active ? m : mlast;
                    if (__ballot_sync(0xffffffffu, acc)) {
                        // a real branch: the accepting groups run the update once, together; the others wait
                        if (acc) {
#pragma unroll
                            for (int i = 0; i < C; ++i) {
                                mt[i] += d[i];
                                if (W2REG) G2[i] = fma(W2[i], d[i], G2[i]);
                                else       G2[i] = fma(Wt[i], d[i] + d[i], G2[i]);
                            }
                            chi2 += dchi2;
                            g = fma(alpha, g, g);
                            ginv *= th.y;
                            // the lane that owns the accepted move holds its new coefficients from its last screen
                            if (sub == m) { *my_pp = xp * ginv; *my_ps = xs * ginv; }
                            acc_sweep++;
                        }
                        __syncwarp();
                        ball = screen();              // a spectrum changed: screen the pending moves again
                    } else {
                        ball = clear_lowest_per_group<G>(ball);
                    }
                }
                if (TRACE) {
                    if (valid && w < P.W) {
                        const uint32_t rq = rbase + (uint32_t)(sub * kRecMaskBytes);
                        const double2 qt = lds_f64x2(rq + 64);
                        const bool feas = (__double2hiint(xp) | __double2hiint(xs)) >= 0;
                        const int fl = (feas ? 1 : 0) | tr_fl;
                        const size_t mvi = ((size_t)(P.call_off + isw)) * n_omega + m0 + sub;
                        if (P.flags) P.flags[(size_t)w * P.call_sweeps * n_omega + mvi] = (uint8_t)fl;
                        if (tracing) {
                            sail_trace_rec *tr = P.trace + ((size_t)(w - P.trace_lo) * P.call_sweeps * n_omega + mvi);
                            tr->p = mv.p; tr->s = mv.s; tr->flags = fl; tr->move = m0 + sub;
                            tr->rho = 1.0 + mv.alpha; tr->delta_p = mv.dp; tr->delta_s = mv.ds;
                            tr->dchi2 = tr_dchi2; tr->thr = qt.x; tr->ap_new = xp; tr->as_new = xs;
                        }
                    }
                }
                __syncwarp();
            }
            // ---- end of sweep: fold the lazy scale (Eq. 19), counters, y (row A6, Eq. 30) ----------------
            for (int k = sub; k < n_omega; k += G) a_all[(size_t)wbase + k] *= g;
            g = 1.0;
            ginv = 1.0;
            if (sub == 0) {
                P.n_acc[w] += (unsigned long long)acc_sweep;
                P.n_eval[w] += (unsigned long long)eval_sweep;
                P.y[w] = amp_factor(P, acc_sweep, y_sweep);
            }
            __syncwarp();
        }
#pragma unroll
        for (int i = 0; i < C; ++i) {
            const int j = sub + G * i;
            if (j < P.n_tau) P.mt[(size_t)w * P.n_tau + j] = mt[i];
        }
        if (sub == 0) P.chi2[w] = chi2;
        __syncwarp();
    }
}

template <int G, int C, int MAXW, bool FACT, bool TRACE, bool W2REG>
static int launch_grp_variant(sail_handle *h, SweepArgs &args)
{
    constexpr int NW = 32 / G;
    args.n_groups = (args.W + NW - 1) / NW;
    int warps = (int)((args.n_groups + h->num_sms - 1) / h->num_sms);
    if (warps > MAXW) warps = MAXW;
    if (warps < 1) warps = 1;
    long long ctas = (args.n_groups + warps - 1) / warps;
    if (ctas > h->num_sms) ctas = h->num_sms;
    const int e0_elems = args.fact ? (args.n_hi + args.n_lo) * G : args.n_omega * G;
    const size_t smem = (size_t)(3 * ((args.n_omega + 1) & ~1) + ((e0_elems + 1) & ~1)) * sizeof(double)
                        + (size_t)warps * 32 * kRecMaskBytes;
    if (smem > 227 * 1024)
        return set_err(h, SAIL_ERR_ARG, "sweep tables need %zu bytes of shared memory (> 227 KB)", smem);
    void (*kern)(const SweepArgs) = sweep_kernel_grp<G, C, MAXW, FACT, TRACE, W2REG>;
    SAIL_CUDA_OK(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int resident = 0;
    SAIL_CUDA_OK(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&resident, kern, warps * 32, smem));
    if (resident < 1)
        return set_err(h, SAIL_ERR_CUDA, "grouped sweep kernel (G=%d, C=%d, MAXW=%d) does not fit one SM at %d warps per CTA", G, C, MAXW, warps);
    kern<<<(unsigned)ctas, warps * 32, smem, h->stream>>>(args);
    SAIL_LAUNCH_OK(h, "sweep_kernel_grp");
    return SAIL_OK;
}

int launch_sweep_grp(sail_handle *h, SweepArgs &a, int G, int C, bool trace, int flavour)
{
    (void)flavour;
#define SAIL_GRP(GG, CC, MW, W2)                                                                                        \
    {                                                                                                                   \
        if (a.fact) return trace ? launch_grp_variant<GG, CC, MW, true, true, W2>(h, a) : launch_grp_variant<GG, CC, MW, true, false, W2>(h, a);   \
        return trace ? launch_grp_variant<GG, CC, MW, false, true, W2>(h, a) : launch_grp_variant<GG, CC, MW, false, false, W2>(h, a);             \
    }
    if (G == 32) {
        if (C <= 4) SAIL_GRP(32, 4, 24, true)
        if (C <= 8) SAIL_GRP(32, 8, 16, true)
        SAIL_GRP(32, 16, 12, false)
    }
    if (G == 16) {
        if (C <= 2) SAIL_GRP(16, 2, 16, true)
        if (C <= 7) SAIL_GRP(16, 7, 16, true)
        if (C <= 13) SAIL_GRP(16, 13, 12, false)
        if (C <= 16) SAIL_GRP(16, 16, 8, true)
        return set_err(h, SAIL_ERR_ARG, "n_tau needs %d tau-points per lane at 16 lanes per walker (max 16)", C);
    }
    if (C <= 4) SAIL_GRP(8, 4, 16, true)
    if (C <= 13) SAIL_GRP(8, 13, 12, false)
    return set_err(h, SAIL_ERR_ARG, "n_tau needs %d tau-points per lane at 8 lanes per walker (max 13)", C);
#undef SAIL_GRP
}

} // namespace sail
