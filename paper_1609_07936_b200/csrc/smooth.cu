// smooth.cu — the smoothing step (Eq. 27-29; readings S1, S2 in DESIGN.md §2).
//   Eq. 27: a_j <- s a_{j-1} + (1 - 2s) a_j + s a_{j+1}     Eq. 28-29: reflecting end bins
// applied to all bins simultaneously (S1), followed by the renormalisation of the second sum rule (S2): a linear
// tilt a_k (1 + kappa (w^m_k - wbar)) about the new mean frequency, kappa = (B - B') / sum a_k (w^m_k - wbar)^2.
// One 128-thread CTA per walker row: the row is read once (cp.async into a double-buffered shared-memory stage that
// serves the neighbour taps; the next row streams in while this one is reduced), three
// block sums (A', B', then the variance), written once: 16 N_omega bytes of HBM traffic per walker.  The model and
// the residue are then refreshed by the dense forward kernel (row A7).
#include "sail_internal.cuh"

namespace sail {

// two block sums with one barrier pair; red has 2 x nwarps slots and alternates between two halves (phase), so the
// slots of one call are not overwritten before every thread has read them
__device__ __forceinline__ void block_sum2(double &u, double &v, double *red, int nwarps, int phase)
{
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        u += __shfl_xor_sync(0xffffffffu, u, off);
        v += __shfl_xor_sync(0xffffffffu, v, off);
    }
    double *r = red + phase * 2 * nwarps;
    if ((threadIdx.x & 31) == 0) { r[2 * (threadIdx.x >> 5)] = u; r[2 * (threadIdx.x >> 5) + 1] = v; }
    __syncthreads();
    double tu = 0.0, tv = 0.0;
    for (int w = 0; w < nwarps; ++w) { tu += r[2 * w]; tv += r[2 * w + 1]; }   // same order in every thread
    u = tu; v = tv;
}

constexpr int kSmoothThreads = 128;
constexpr int kSmoothPerThread = 16;                   // 128 threads x 16 = rows of up to 2048 bins

__global__ void __launch_bounds__(kSmoothThreads) smooth_kernel(int n_omega, long long W, double s, double B, double domega,
                                                     const double *__restrict__ omega, double *__restrict__ a)
{
    extern __shared__ __align__(16) double rows[];     // [2][n_omega rounded up to even]: old spectra, double-buffered
    __shared__ double red[4 * (kSmoothThreads / 32)];
    const double c = 1.0 - 2.0 * s, e = 1.0 - s, half = 0.5 * domega;
    const int nwarps = blockDim.x >> 5;
    const int n_pad = (n_omega + 1) & ~1;
    const bool vec = (n_omega & 1) == 0;               // rows are 16-byte aligned: cp.async of pairs
    // the next row of this CTA streams into the other buffer (cp.async) while the current one is reduced
    auto prefetch = [&](long long w, int buf) {
        if (vec && w < W) {
            const uint32_t dst = (uint32_t)__cvta_generic_to_shared(rows + buf * n_pad);
            const double *src = a + (size_t)w * n_omega;
            for (int k2 = threadIdx.x; k2 < n_omega / 2; k2 += blockDim.x)
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(dst + (uint32_t)k2 * 16u), "l"(src + 2 * k2) : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    prefetch(blockIdx.x, 0);
    int it = 0;
    for (long long w = blockIdx.x; w < W; w += gridDim.x, ++it) {
        double *aw = a + (size_t)w * n_omega;
        double *row = rows + (it & 1) * n_pad;
        prefetch(w + gridDim.x, (it & 1) ^ 1);         // its previous contents were last read before the barriers of row it-1
        asm volatile("cp.async.wait_group 1;" ::: "memory");
        if (!vec)
            for (int k = threadIdx.x; k < n_omega; k += blockDim.x) row[k] = aw[k];
        __syncthreads();
        double nv[kSmoothPerThread];
        double sA = 0.0, sB = 0.0;
#pragma unroll
        for (int u = 0; u < kSmoothPerThread; ++u) {
            const int k = threadIdx.x + u * kSmoothThreads;
            nv[u] = 0.0;
            if (k < n_omega) {
                // the definition's operation order, two roundings per product, no contraction
                if (n_omega == 1) nv[u] = row[0];
                else if (k == 0) nv[u] = __dadd_rn(__dmul_rn(e, row[0]), __dmul_rn(s, row[1]));
                else if (k == n_omega - 1) nv[u] = __dadd_rn(__dmul_rn(e, row[k]), __dmul_rn(s, row[k - 1]));
                else nv[u] = __dadd_rn(__dadd_rn(__dmul_rn(s, row[k - 1]), __dmul_rn(c, row[k])), __dmul_rn(s, row[k + 1]));
                sA += nv[u];
                sB = fma(nv[u], omega[k] + half, sB);
            }
        }
        block_sum2(sA, sB, red, nwarps, 0);
        const double A1 = sA, B1 = sB;
        const double wbar = B1 / A1;
        double sV = 0.0;
#pragma unroll
        for (int u = 0; u < kSmoothPerThread; ++u) {
            const int k = threadIdx.x + u * kSmoothThreads;
            if (k < n_omega) { const double dw = (omega[k] + half) - wbar; sV = fma(nv[u] * dw, dw, sV); }
        }
        double dummy = 0.0;
        block_sum2(sV, dummy, red, nwarps, 1);
        const double V = sV;
        const double kappa = (V > 0.0) ? (B - B1) / V : 0.0;
#pragma unroll
        for (int u = 0; u < kSmoothPerThread; ++u) {
            const int k = threadIdx.x + u * kSmoothThreads;
            if (k < n_omega) aw[k] = nv[u] * (1.0 + kappa * ((omega[k] + half) - wbar));
        }
    }
}

int launch_smooth(sail_handle *h, double s)
{
    if (h->n_omega > kSmoothThreads * kSmoothPerThread)
        return set_err(h, SAIL_ERR_ARG, "sail_smooth supports n_omega <= %d", kSmoothThreads * kSmoothPerThread);
    const long long W = h->W;
    const int blocks = (int)(W < (long long)h->num_sms * 12 ? W : (long long)h->num_sms * 12);
    smooth_kernel<<<blocks, kSmoothThreads, (size_t)2 * ((h->n_omega + 1) & ~1) * sizeof(double), h->stream>>>(h->n_omega, W, s, h->B, h->domega,
                                                                                 h->tab.omega, h->st.a);
    SAIL_LAUNCH_OK(h, "smooth_kernel");
    return launch_forward(h, 0, W);
}

} // namespace sail
