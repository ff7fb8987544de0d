// forward.cu — problem tables (Eq. 5-8), the dense forward transform M = a K (Eq. 7) used by
// init, resync and state injection, and the residue chi^2 (Eq. 9).
#include "sail_internal.cuh"

namespace sail {

// c_j (Eq. 8 with expm1), Wj = (c_j/sigma_j)^2, fj = F_j/c_j, E[k][j] = exp(-omega_k tau_j)
__global__ void problem_tables_kernel(int n_omega, int n_tau, const double *omega, const double *tau,
                                      const double *F, const double *sigma, double domega,
                                      double *c, double *Wj, double *fj, double *E)
{
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int stride = gridDim.x * blockDim.x;
    const double two_pi = 6.283185307179586476925286766559;
    for (int j = tid; j < n_tau; j += stride) {
        const double t = tau[j];
        const double cj = (t == 0.0) ? domega / two_pi : -expm1(-domega * t) / (two_pi * t);
        const double sg = sigma ? sigma[j] : 1.0;
        const double r = cj / sg;
        c[j] = cj;
        Wj[j] = r * r;
        fj[j] = F[j] / cj;
    }
    const long long total = (long long)n_omega * n_tau;
    for (long long i = tid; i < total; i += stride) {
        const int k = (int)(i / n_tau), j = (int)(i % n_tau);
        E[i] = exp(-omega[k] * tau[j]);
    }
}

// ---- dense fp64 contraction: mt[w][j] = sum_k a[w][k] E[k][j] ----------------------------------------
// 64x64 output tile per CTA, 16x16 threads, 4x4 register micro-tile, K-step 16 through shared memory.
constexpr int FT = 64, FK = 16;

__global__ void __launch_bounds__(256) forward_kernel(int n_omega, int n_tau, long long w0, long long n,
                                                      const double *__restrict__ a, const double *__restrict__ E,
                                                      double *__restrict__ mt)
{
    __shared__ double As[FK][FT + 1];
    __shared__ double Bs[FK][FT];
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    const long long row0 = (long long)blockIdx.y * FT;   // walker offset within [w0, w0+n)
    const int col0 = blockIdx.x * FT;
    double acc[4][4] = {};
    for (int k0 = 0; k0 < n_omega; k0 += FK) {
        // A tile: 64 walkers x 16 k
        for (int i = threadIdx.x; i < FT * FK; i += 256) {
            const int r = i / FK, kk = i % FK;
            const long long wr = row0 + r;
            As[kk][r] = (wr < n && k0 + kk < n_omega) ? a[(size_t)(w0 + wr) * n_omega + k0 + kk] : 0.0;
        }
        for (int i = threadIdx.x; i < FK * FT; i += 256) {
            const int kk = i / FT, cc = i % FT;
            Bs[kk][cc] = (k0 + kk < n_omega && col0 + cc < n_tau) ? E[(size_t)(k0 + kk) * n_tau + col0 + cc] : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < FK; ++kk) {
            double av[4], bv[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) av[i] = As[kk][ty + 16 * i];
#pragma unroll
            for (int jx = 0; jx < 4; ++jx) bv[jx] = Bs[kk][tx + 16 * jx];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int jx = 0; jx < 4; ++jx) acc[i][jx] = fma(av[i], bv[jx], acc[i][jx]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const long long wr = row0 + ty + 16 * i;
        if (wr >= n) continue;
#pragma unroll
        for (int jx = 0; jx < 4; ++jx) {
            const int cc = col0 + tx + 16 * jx;
            if (cc < n_tau) mt[(size_t)(w0 + wr) * n_tau + cc] = acc[i][jx];
        }
    }
}

// chi^2[w] = sum_j Wj (mt_j - fj)^2 — one warp per walker
__global__ void chi2_kernel(int n_tau, long long w0, long long n, const double *__restrict__ mt,
                            const double *__restrict__ Wj, const double *__restrict__ fj, double *__restrict__ chi2)
{
    const long long wi = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (wi >= n) return;
    const int lane = threadIdx.x & 31;
    const double *row = mt + (size_t)(w0 + wi) * n_tau;
    double s = 0.0;
    for (int j = lane; j < n_tau; j += 32) {
        const double D = row[j] - fj[j];
        s = fma(Wj[j] * D, D, s);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    if (lane == 0) chi2[w0 + wi] = s;
}

int launch_forward(sail_handle *h, int64_t w0, int64_t n)
{
    if (n <= 0) return SAIL_OK;
    dim3 grid((h->n_tau + FT - 1) / FT, (unsigned)((n + FT - 1) / FT));
    forward_kernel<<<grid, 256, 0, h->stream>>>(h->n_omega, h->n_tau, w0, n, h->st.a, h->tab.E, h->st.mt);
    SAIL_LAUNCH_OK(h, "forward_kernel");
    const int wpb = 8;
    chi2_kernel<<<(unsigned)((n + wpb - 1) / wpb), wpb * 32, 0, h->stream>>>(h->n_tau, w0, n, h->st.mt,
                                                                            h->tab.Wj, h->tab.fj, h->st.chi2);
    SAIL_LAUNCH_OK(h, "chi2_kernel");
    return SAIL_OK;
}

__global__ void scale_model_kernel(long long total, int n_tau, const double *__restrict__ mt,
                                   const double *__restrict__ c, double *__restrict__ dst)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total;
         i += (long long)gridDim.x * blockDim.x)
        dst[i] = c[i % n_tau] * mt[i];
}

int launch_scale_model(sail_handle *h, double *dst)
{
    const long long total = h->W * h->n_tau;
    const int blocks = (int)((total + 255) / 256 < 4096 ? (total + 255) / 256 : 4096);
    scale_model_kernel<<<blocks, 256, 0, h->stream>>>(total, h->n_tau, h->st.mt, h->tab.c, dst);
    SAIL_LAUNCH_OK(h, "scale_model_kernel");
    return SAIL_OK;
}

int launch_problem_tables(sail_handle *h, const double *d_F, const double *d_sigma, double *c, double *Wj,
                          double *fj, double *E)
{
    problem_tables_kernel<<<256, 256, 0, h->stream>>>(h->n_omega, h->n_tau, h->tab.omega, h->tab.tau, d_F, d_sigma,
                                                      h->domega, c, Wj, fj, E);
    SAIL_LAUNCH_OK(h, "problem_tables_kernel");
    return SAIL_OK;
}

} // namespace sail
