// smooth.cu — the smoothing step (Eq. 27-29; readings S1, S2 in DESIGN.md §2).
//   Eq. 27: a_j <- s a_{j-1} + (1 - 2s) a_j + s a_{j+1}     Eq. 28-29: reflecting end bins
// applied to all bins simultaneously (S1), followed by the renormalisation of the second sum rule (S2): a linear
// tilt a_k (1 + kappa (w^m_k - wbar)) about the new mean frequency, kappa = (B - B') / sum a_k (w^m_k - wbar)^2,
// clamped so that no coefficient turns negative.
// One WARP per walker row, no block barrier on the path: lane 0 streams whole rows global -> shared with the bulk-copy
// engine (cp.async.bulk + one mbarrier per warp), the lanes read the three taps from shared memory (bin k = lane +
// 32 i: conflict free) and keep the smoothed row in registers, so the stage is refilled with the warp's next row while
// A', B' and the second moment are reduced by shuffles (one round) and the tilted row is stored coalesced.  16 N_omega bytes of HBM traffic
// per walker.  The model and the residue are then refreshed by the dense forward kernel (row A7).
#include "sail_internal.cuh"

namespace sail {

constexpr int kSmoothWarps = 12;

// three sums over the warp at once (the butterflies interleave: one latency instead of three)
__device__ __forceinline__ void warp_sum3(double &x, double &y, double &z)
{
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        x += __shfl_xor_sync(0xffffffffu, x, off);
        y += __shfl_xor_sync(0xffffffffu, y, off);
        z += __shfl_xor_sync(0xffffffffu, z, off);
    }
}

template <int PER>   // bins per lane: n_omega <= 32 PER
__global__ void __launch_bounds__(kSmoothWarps * 32) smooth_kernel(int n_omega, long long W, double s, double B, double c0, double domega,
                                                                   const double *__restrict__ omega, double *__restrict__ a,
                                                                   const double *__restrict__ halt)
{
    if (halt && *halt != 0.0) return;      // sail_anneal_selfcool after its rule failed: the rest of the call is a no-op
    extern __shared__ __align__(128) unsigned char smem[];     // wm[n_pad] - c0 | per warp: one stage of n_pad doubles
    __shared__ __align__(8) unsigned long long bars[kSmoothWarps];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int n_pad = (n_omega + 1) & ~1;
    double *s_wm = reinterpret_cast<double *>(smem);
    double *row = s_wm + n_pad + (size_t)warp * n_pad;
    const double c = 1.0 - 2.0 * s, e = 1.0 - s, half = 0.5 * domega;
    const bool bulk = (n_omega & 1) == 0;                      // rows are multiples of 16 bytes: bulk copies
    // frequencies are kept RELATIVE to c0 = B / A, the mean frequency the two sum rules pin (Eq. 23): the smoothed row's
    // own mean differs from it by O(s domega), so the one-pass second moment below does not cancel however narrow the
    // spectrum is or wherever it sits on the grid (about 0 it lost (wbar / width)^2 eps)
    for (int k = threadIdx.x; k < n_omega; k += blockDim.x) s_wm[k] = (omega[k] + half) - c0;
    const uint32_t bar = (uint32_t)__cvta_generic_to_shared(&bars[warp]);
    if (lane == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(bar) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const long long stride = (long long)gridDim.x * kSmoothWarps;
    auto fetch = [&](long long w) {                            // lane 0: row w -> this warp's stage
        const uint32_t dst = (uint32_t)__cvta_generic_to_shared(row);
        const uint32_t bytes = (uint32_t)n_omega * 8u;
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     :: "r"(dst), "l"(a + (size_t)w * n_omega), "r"(bytes), "r"(bar) : "memory");
    };
    long long w = (long long)blockIdx.x * kSmoothWarps + warp;
    if (bulk && lane == 0 && w < W) fetch(w);
    int it = 0;
    for (; w < W; w += stride, ++it) {
        double *aw = a + (size_t)w * n_omega;
        if (bulk) {
            const uint32_t parity = (uint32_t)(it & 1);
            asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
                         "@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}" :: "r"(bar), "r"(parity) : "memory");
        } else {
            for (int k = lane; k < n_omega; k += 32) row[k] = aw[k];
            __syncwarp();
        }
        double nv[PER];
        double sA = 0.0, sB = 0.0, sC = 0.0;
#pragma unroll
        for (int i = 0; i < PER; ++i) {
            const int k = lane + 32 * i;
            nv[i] = 0.0;
            if (k < n_omega) {
                // the definition's operation order, two roundings per product, no contraction
                if (n_omega == 1) nv[i] = row[0];
                else if (k == 0) nv[i] = __dadd_rn(__dmul_rn(e, row[0]), __dmul_rn(s, row[1]));
                else if (k == n_omega - 1) nv[i] = __dadd_rn(__dmul_rn(e, row[k]), __dmul_rn(s, row[k - 1]));
                else nv[i] = __dadd_rn(__dadd_rn(__dmul_rn(s, row[k - 1]), __dmul_rn(c, row[k])), __dmul_rn(s, row[k + 1]));
                const double wk = s_wm[k];
                sA += nv[i];
                sB = fma(nv[i], wk, sB);
                sC = fma(nv[i] * wk, wk, sC);
            }
        }
        __syncwarp();
        // the whole row now lives in registers: the stage is free, the next row streams in behind the reductions
        if (bulk && lane == 0 && w + stride < W) fetch(w + stride);
        warp_sum3(sA, sB, sC);
        // with u_k = w_k - c0:  sB = B' - c0 A',  wbar - c0 = sB / A',  B - B' = (B - c0 A') - sB
        const double A1 = sA, U1 = sB;
        const double wbar = U1 / A1;                           // the row's mean frequency, relative to c0
        // sum a_k (u_k - wbar)^2 = sum a_k u_k^2 - wbar sum a_k u_k  (one reduction round instead of two)
        const double V = fma(-wbar, U1, sC);
        double kappa = (V > 0.0) ? (fma(-c0, A1, B) - U1) / V : 0.0;
        // positivity (reading S2): the tilt factor is linear in k, smallest at an end bin
        const double d_lo = s_wm[0] - wbar, d_hi = s_wm[n_omega - 1] - wbar;
        // (product and sum rounded separately, here and in the store below: a fused 1 + kappa d at the clamped end bin would
        // see the rounding error of -1 / d and could come out at -1e-16, a negative coefficient; fl(fl(-1/d) d) >= -1)
        if (__dadd_rn(1.0, __dmul_rn(kappa, d_lo)) < 0.0) kappa = -1.0 / d_lo;
        if (__dadd_rn(1.0, __dmul_rn(kappa, d_hi)) < 0.0) kappa = -1.0 / d_hi;
#pragma unroll
        for (int i = 0; i < PER; ++i) {
            const int k = lane + 32 * i;
            if (k < n_omega) aw[k] = nv[i] * __dadd_rn(1.0, __dmul_rn(kappa, s_wm[k] - wbar));
        }
    }
}

int launch_smooth(sail_handle *h, double s)
{
    if (h->n_omega > 2048) return set_err(h, SAIL_ERR_ARG, "sail_smooth supports n_omega <= 2048");
    const long long W = h->W;
    const int n_pad = (h->n_omega + 1) & ~1;
    const size_t smem = (size_t)(1 + kSmoothWarps) * n_pad * sizeof(double);
    void (*kern)(int, long long, double, double, double, double, const double *, double *, const double *);
    const int per = (h->n_omega + 31) / 32;
    if (per <= 8) kern = smooth_kernel<8>;
    else if (per <= 16) kern = smooth_kernel<16>;
    else if (per <= 32) kern = smooth_kernel<32>;
    else kern = smooth_kernel<64>;
    SAIL_CUDA_OK(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 0;
    SAIL_CUDA_OK(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kSmoothWarps * 32, smem));
    if (per_sm < 1) return set_err(h, SAIL_ERR_CUDA, "smooth_kernel does not fit an SM");
    long long blocks = (W + kSmoothWarps - 1) / kSmoothWarps;
    if (blocks > (long long)h->num_sms * per_sm) blocks = (long long)h->num_sms * per_sm;
    kern<<<(unsigned)blocks, kSmoothWarps * 32, smem, h->stream>>>(h->n_omega, W, s, h->B, h->B / h->A, h->domega, h->tab.omega, h->st.a, h->halt);
    SAIL_LAUNCH_OK(h, "smooth_kernel");
    return launch_forward(h, 0, W);
}

} // namespace sail
