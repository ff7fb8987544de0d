// forward.cu — problem tables (Eq. 5-8), the dense forward transform M = a K (Eq. 7) used by
// init, resync and state injection, and the residue chi^2 (Eq. 9).
#include "sail_internal.cuh"

namespace sail {

// c_j (Eq. 8 with expm1), Wj = (c_j/sigma_j)^2, fj = F_j/c_j, E[k][j] = exp(-omega_k tau_j)
__global__ void problem_tables_kernel(int n_omega, int n_tau, const double *omega, const double *tau,
                                      const double *F, const double *sigma, double domega,
                                      double *c, double *Wj, double *fj, double *E, double *ET)
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
        const double e = exp(-omega[k] * tau[j]);
        E[i] = e;
        ET[(size_t)j * n_omega + k] = e;
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

// ---- the same contraction on the DMMA path (mma.sync m8n8k4 f64) ------------------------------------------------
// On B200 a DMMA m8n8k4 occupies the FP64 pipe exactly like the 8 DFMAs it replaces (sail_microbench), so it buys
// no flops; what it buys is issue slots: one instruction per 256 fused multiply-adds, with operands taken straight
// from two registers per lane, leaves the scheduler free to feed the pipe, which the 4x4 register-tiled DFMA form
// (one LDS per 2 DFMA) cannot.  CTA tile 128 walkers x 64 tau, 8 warps of 32 x 32 (4 x 4 DMMA tiles, 32 fp64
// accumulators per lane), K-step 16 through a 3-stage cp.async ring.  Both operands are k-contiguous in memory
// (a[w][k], ET[j][k]) and are staged as [k-group of 4][row][4], which makes every fragment load of a half-warp
// 16 consecutive doubles (conflict-free).  Needs n_omega % 4 == 0 (16-byte cp.async of k-pairs).
constexpr int DM = 128, DN = 64, DK = 16, DST = 3;

__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src, bool valid)
{
    const int sz = valid ? 16 : 0;                     // src-size 0: the 16 bytes are zero-filled
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" :: "r"(dst), "l"(src), "r"(sz) : "memory");
}

__global__ void __launch_bounds__(256, 2) forward_dmma_kernel(int n_omega, int n_tau, long long w0, long long n,
                                                              const double *__restrict__ a, const double *__restrict__ ET,
                                                              double *__restrict__ mt)
{
    extern __shared__ __align__(16) double fsm[];
    double *As = fsm;                                  // [DST][4][DM][4]
    double *Bs = fsm + DST * 4 * DM * 4;               // [DST][4][DN][4]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = (warp & 3) * 32, wn = (warp >> 2) * 32;
    const long long row0 = (long long)blockIdx.y * DM;
    const int col0 = blockIdx.x * DN;
    const uint32_t as_u = (uint32_t)__cvta_generic_to_shared(As), bs_u = (uint32_t)__cvta_generic_to_shared(Bs);

    auto load_stage = [&](int st, int k0) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {                  // A: 128 rows x 8 pairs of doubles
            const int c = tid + 256 * i, r = c >> 3, part = c & 7, k = k0 + part * 2;
            const long long wr = row0 + r;
            const bool ok = wr < n && k < n_omega;
            const double *src = a + (size_t)(w0 + (ok ? wr : 0)) * n_omega + (ok ? k : 0);
            cp_async16(as_u + (uint32_t)((((st * 4 + (part >> 1)) * DM + r) * 4 + (part & 1) * 2) * 8), src, ok);
        }
#pragma unroll
        for (int i = 0; i < 2; ++i) {                  // B: 64 tau-columns x 8 pairs
            const int c = tid + 256 * i, r = c >> 3, part = c & 7, k = k0 + part * 2;
            const bool ok = col0 + r < n_tau && k < n_omega;
            const double *src = ET + (size_t)(ok ? col0 + r : 0) * n_omega + (ok ? k : 0);
            cp_async16(bs_u + (uint32_t)((((st * 4 + (part >> 1)) * DN + r) * 4 + (part & 1) * 2) * 8), src, ok);
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    double acc[4][4][2] = {};
    const int nk = (n_omega + DK - 1) / DK;
    for (int s = 0; s < DST - 1; ++s) {
        if (s < nk) load_stage(s, s * DK);
        else asm volatile("cp.async.commit_group;" ::: "memory");
    }
    for (int kt = 0; kt < nk; ++kt) {
        asm volatile("cp.async.wait_group %0;" :: "n"(DST - 2) : "memory");
        __syncthreads();                               // stage kt has landed; stage kt-1 is free for the next load
        if (kt + DST - 1 < nk) load_stage((kt + DST - 1) % DST, (kt + DST - 1) * DK);
        else asm volatile("cp.async.commit_group;" ::: "memory");
        const int st = kt % DST;
        const double *Ast = As + (size_t)st * 4 * DM * 4, *Bst = Bs + (size_t)st * 4 * DN * 4;
#pragma unroll
        for (int kg = 0; kg < 4; ++kg) {
            double af[4], bf[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) af[i] = Ast[((kg * DM) + wm + 8 * i + (lane >> 2)) * 4 + (lane & 3)];
#pragma unroll
            for (int j = 0; j < 4; ++j) bf[j] = Bst[((kg * DN) + wn + 8 * j + (lane >> 2)) * 4 + (lane & 3)];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                                 : "+d"(acc[i][j][0]), "+d"(acc[i][j][1]) : "d"(af[i]), "d"(bf[j]));
        }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const long long wr = row0 + wm + 8 * i + (lane >> 2);
        if (wr >= n) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int cc = col0 + wn + 8 * j + 2 * (lane & 3);
            double *dst = mt + (size_t)(w0 + wr) * n_tau + cc;
            if (cc < n_tau) dst[0] = acc[i][j][0];
            if (cc + 1 < n_tau) dst[1] = acc[i][j][1];
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
    if ((h->n_omega & 3) == 0) {
        const size_t smem = (size_t)DST * 4 * (DM + DN) * 4 * sizeof(double);
        SAIL_CUDA_OK(h, cudaFuncSetAttribute(forward_dmma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        dim3 grid((h->n_tau + DN - 1) / DN, (unsigned)((n + DM - 1) / DM));
        forward_dmma_kernel<<<grid, 256, smem, h->stream>>>(h->n_omega, h->n_tau, w0, n, h->st.a, h->tab.ET, h->st.mt);
        SAIL_LAUNCH_OK(h, "forward_dmma_kernel");
    } else {
        dim3 grid((h->n_tau + FT - 1) / FT, (unsigned)((n + FT - 1) / FT));
        forward_kernel<<<grid, 256, 0, h->stream>>>(h->n_omega, h->n_tau, w0, n, h->st.a, h->tab.E, h->st.mt);
        SAIL_LAUNCH_OK(h, "forward_kernel");
    }
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
                                                      h->domega, c, Wj, fj, E, h->tab.ET);
    SAIL_LAUNCH_OK(h, "problem_tables_kernel");
    return SAIL_OK;
}

} // namespace sail
