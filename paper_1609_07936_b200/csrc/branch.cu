// branch.cu — imprinted branching (Eq. 24-26; readings B1-B5 in
// DESIGN.md §2): fixed-point weights -> integer prefix sum -> comb multipliers (sum m = W exactly) ->
// donor map by binary search -> coalesced 128-bit imprint copy of (spectrum, model) + residue.
#include "sail_internal.cuh"
#include <math.h>
#include <string.h>

namespace sail {

constexpr int kScanThreads = 256;
constexpr int kScanItems = 4;
constexpr int kScanTile = kScanThreads * kScanItems;   // 1024 elements per CTA

// Order-preserving key of a double: the running residue chi2_0 + sum dchi2 can dip below zero near an exact fit, so
// the plain bit pattern (valid for values >= 0 only) is not enough.  Negative values have all bits flipped, the others
// only the sign bit: unsigned comparison of keys orders like the values (-0 < +0, NaN above +inf).
__device__ __forceinline__ unsigned long long ordered_key(double v)
{
    const unsigned long long b = (unsigned long long)__double_as_longlong(v);
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __forceinline__ double key_value(unsigned long long k)
{
    return __longlong_as_double((long long)((k >> 63) ? (k & 0x7fffffffffffffffull) : ~k));
}

__global__ void chi2_min_kernel(long long W, const double *__restrict__ chi2, unsigned long long *scalars)
{
    unsigned long long m = ~0ull;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < W; i += (long long)gridDim.x * blockDim.x) {
        const unsigned long long b = ordered_key(chi2[i]);
        m = b < m ? b : m;
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        const unsigned long long o = __shfl_xor_sync(0xffffffffu, m, off);
        m = o < m ? o : m;
    }
    if ((threadIdx.x & 31) == 0) atomicMin(scalars + 0, m);
}

// B1 + B3: e_i = exp(-(chi2_i - chi2_min)/T), E_i = floor(e_i 2^40)
__global__ void weights_kernel(long long W, const double *__restrict__ chi2, double T,
                               const unsigned long long *scalars, unsigned long long *ehat)
{
    const double cmin = key_value(scalars[0]);
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < W; i += (long long)gridDim.x * blockDim.x) {
        // chi2_i >= chi2_min makes the exponent <= 0 and the weight <= 2^40; a NaN residue gets weight 0
        const double e = exp(-(chi2[i] - cmin) / T);
        ehat[i] = (e == e) ? (unsigned long long)floor(fmin(e, 1.0) * 1099511627776.0) : 0ull;
    }
}

// ---- three-phase inclusive scan of u64 arrays (blockIdx.y selects the array) -----------------------
struct ScanArrays { unsigned long long *arr[2]; unsigned long long *sums[2]; };

__global__ void __launch_bounds__(kScanThreads) scan_tiles_kernel(long long n, ScanArrays S)
{
    __shared__ unsigned long long warp_tot[kScanThreads / 32];
    unsigned long long *x = S.arr[blockIdx.y];
    const long long base = (long long)blockIdx.x * kScanTile + (long long)threadIdx.x * kScanItems;
    unsigned long long v[kScanItems], run = 0;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        v[i] = (base + i < n) ? x[base + i] : 0ull;
        run += v[i];
        v[i] = run;
    }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    unsigned long long inc = run;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const unsigned long long o = __shfl_up_sync(0xffffffffu, inc, off);
        if (lane >= off) inc += o;
    }
    if (lane == 31) warp_tot[wid] = inc;
    __syncthreads();
    unsigned long long prefix = inc - run;
    for (int w2 = 0; w2 < wid; ++w2) prefix += warp_tot[w2];
#pragma unroll
    for (int i = 0; i < kScanItems; ++i)
        if (base + i < n) x[base + i] = v[i] + prefix;
    if (threadIdx.x == kScanThreads - 1) S.sums[blockIdx.y][blockIdx.x] = prefix + run;
}

__global__ void scan_sums_kernel(int n_tiles, ScanArrays S)
{
    // few tiles (W/1024): one thread per array is enough and keeps the result exact and ordered
    if (threadIdx.x == 0) {
        unsigned long long *s = S.sums[blockIdx.x];
        unsigned long long run = 0;
        for (int i = 0; i < n_tiles; ++i) { const unsigned long long t = s[i]; s[i] = run; run += t; }
    }
}

__global__ void __launch_bounds__(kScanThreads) scan_add_kernel(long long n, ScanArrays S)
{
    unsigned long long *x = S.arr[blockIdx.y];
    const unsigned long long off = S.sums[blockIdx.y][blockIdx.x];
    const long long base = (long long)blockIdx.x * kScanTile + (long long)threadIdx.x * kScanItems;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i)
        if (base + i < n) x[base + i] += off;
}

static int scan_inclusive(sail_handle *h, long long n, int n_arrays, unsigned long long *a0, unsigned long long *a1)
{
    const int tiles = (int)((n + kScanTile - 1) / kScanTile);
    ScanArrays S;
    S.arr[0] = a0; S.arr[1] = a1;
    S.sums[0] = h->br.block_sums; S.sums[1] = h->br.block_sums + tiles;
    scan_tiles_kernel<<<dim3(tiles, n_arrays), kScanThreads, 0, h->stream>>>(n, S);
    SAIL_LAUNCH_OK(h, "scan_tiles_kernel");
    if (tiles > 1) {
        scan_sums_kernel<<<n_arrays, 32, 0, h->stream>>>(tiles, S);
        SAIL_LAUNCH_OK(h, "scan_sums_kernel");
        scan_add_kernel<<<dim3(tiles, n_arrays), kScanThreads, 0, h->stream>>>(n, S);
        SAIL_LAUNCH_OK(h, "scan_add_kernel");
    }
    return SAIL_OK;
}

// B2: comb multipliers m_i = floor((C_i W + Xi)/S) - floor((C_{i-1} W + Xi)/S), Xi = (x0 S) >> 32
__global__ void multipliers_kernel(long long W, const unsigned long long *__restrict__ Cinc, uint32_t seed_lo,
                                   uint32_t seed_hi, uint32_t sweep, int32_t *mult, unsigned long long *is_rec,
                                   unsigned long long *extras, unsigned long long *scalars)
{
    const unsigned long long S = Cinc[W - 1];
    uint32_t x[4];
    philox4x32_10(0u, sweep, 0u, 1u, seed_lo, seed_hi, x);
    const unsigned __int128 Xi = ((unsigned __int128)x[0] * S) >> 32;
    int mmax = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < W; i += (long long)gridDim.x * blockDim.x) {
        const unsigned long long cprev = i ? Cinc[i - 1] : 0ull;
        const unsigned long long hi = (unsigned long long)(((unsigned __int128)Cinc[i] * (unsigned long long)W + Xi) / S);
        const unsigned long long lo = (unsigned long long)(((unsigned __int128)cprev * (unsigned long long)W + Xi) / S);
        const int m = (int)(hi - lo);
        mult[i] = m;
        is_rec[i] = (m == 0) ? 1ull : 0ull;
        extras[i] = (m > 1) ? (unsigned long long)(m - 1) : 0ull;
        mmax = m > mmax ? m : mmax;
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        const int o = __shfl_xor_sync(0xffffffffu, mmax, off);
        mmax = o > mmax ? o : mmax;
    }
    if ((threadIdx.x & 31) == 0) atomicMax(scalars + 3, (unsigned long long)mmax);
    if (blockIdx.x == 0 && threadIdx.x == 0) scalars[1] = S;
}

// B4: recipient of rank r takes the donor with X_i <= r < X_i + x_i (binary search on the inclusive scan)
__global__ void donor_map_kernel(long long W, const int32_t *__restrict__ mult, const unsigned long long *__restrict__ rec_inc,
                                 const unsigned long long *__restrict__ ext_inc, int64_t *donor_of, int64_t *rec_list,
                                 unsigned long long *scalars)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < W; i += (long long)gridDim.x * blockDim.x) {
        long long donor = -1;
        if (mult[i] == 0) {
            const unsigned long long r = rec_inc[i] - 1;
            long long lo = 0, hi = W - 1;            // first index with ext_inc > r
            while (lo < hi) {
                const long long mid = (lo + hi) >> 1;
                if (ext_inc[mid] > r) hi = mid; else lo = mid + 1;
            }
            donor = lo;
            rec_list[r] = i;
        }
        donor_of[i] = donor;
        if (i == W - 1) scalars[2] = rec_inc[i];
    }
}

// Eq. 26: a(l1) <- t a(l2) + (1-t) a(l1) for spectrum and model (linearity); chi^2 of the
// recipient from its new model.  One CTA per recipient, 128-bit accesses when rows are 16-byte aligned.
// One CTA per recipient: a and mt of the recipient become t * donor + (1 - t) * self (two roundings per product
// and one per sum, exactly the definition), chi^2 is recomputed from the new model.  COPY (t == 1): t * z + 0 * x
// is z bit for bit, so the recipient is not read at all (two streams instead of three).  All loads of a CTA's
// pass are issued before its first store (8 x 16 B per thread in flight).
template <bool COPY>
__global__ void __launch_bounds__(256) imprint_kernel(int n_omega, int n_tau, double t, const int64_t *__restrict__ rec_list,
                                                      const int64_t *__restrict__ donor_of, const unsigned long long *scalars,
                                                      double *a, double *mt, double *chi2,
                                                      const double *__restrict__ Wj, const double *__restrict__ fj)
{
    __shared__ double red[8];
    const long long n_rec = (long long)scalars[2];
    const double omt = 1.0 - t;
    auto mix = [&](double z, double x) { return COPY ? z : __dadd_rn(__dmul_rn(t, z), __dmul_rn(omt, x)); };
    for (long long r = blockIdx.x; r < n_rec; r += gridDim.x) {
        const long long i = rec_list[r], dn = donor_of[i];
        double *ai = a + (size_t)i * n_omega;
        const double *ad = a + (size_t)dn * n_omega;
        double *mi = mt + (size_t)i * n_tau;
        const double *md = mt + (size_t)dn * n_tau;
        if ((n_omega & 1) == 0) {
            double2 *ai2 = reinterpret_cast<double2 *>(ai);
            const double2 *ad2 = reinterpret_cast<const double2 *>(ad);
            const int n2 = n_omega / 2;
            constexpr int U = COPY ? 8 : 4;          // 8 x 16 B per thread in flight either way
            for (int k0 = threadIdx.x; k0 < n2; k0 += U * 256) {
                double2 x[U], z[U];
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const int k = k0 + u * 256;
                    if (k < n2) { z[u] = ad2[k]; if (!COPY) x[u] = ai2[k]; }
                }
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const int k = k0 + u * 256;
                    if (k < n2) ai2[k] = make_double2(mix(z[u].x, COPY ? 0.0 : x[u].x), mix(z[u].y, COPY ? 0.0 : x[u].y));
                }
            }
        } else {
            for (int k = threadIdx.x; k < n_omega; k += blockDim.x) ai[k] = mix(ad[k], COPY ? 0.0 : ai[k]);
        }
        double s = 0.0;
        for (int j = threadIdx.x; j < n_tau; j += blockDim.x) {
            const double v = mix(md[j], COPY ? 0.0 : mi[j]);
            mi[j] = v;
            const double D = v - fj[j];
            s = fma(Wj[j] * D, D, s);
        }
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
        __syncthreads();
        if (threadIdx.x == 0) {
            double tot = 0.0;
            for (int w2 = 0; w2 < (int)(blockDim.x >> 5); ++w2) tot += red[w2];
            chi2[i] = tot;
        }
        __syncthreads();
    }
}

// ---- the same imprint through the bulk-copy engine (TMA, cp.async.bulk + mbarrier) ---------------------------------
// One elected thread streams whole walker rows (spectrum 8 N_omega bytes + model 8 N_tau bytes) global -> shared
// -> global through an NST-stage ring: the donor rows (and, for t < 1, the recipient's own rows) of recipient it+NST-1
// are in flight while recipient it is combined, its residue summed, and its rows stored.  Bytes in flight per CTA
// are whole rows (20-40 KB on Stress) instead of 8 x 16 B per thread.  Needs rows that are multiples of 16 bytes.
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\t"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
                 "@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}" :: "r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void bulk_s2g(void *dst, uint32_t src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" :: "l"(dst), "r"(src), "r"(bytes) : "memory");
}

template <bool COPY, int NST>
__global__ void __launch_bounds__(128) imprint_tma_kernel(int n_omega, int n_tau, double t, const int64_t *__restrict__ rec_list,
                                                          const int64_t *__restrict__ donor_of, const unsigned long long *scalars,
                                                          double *a, double *mt, double *chi2,
                                                          const double *__restrict__ Wj, const double *__restrict__ fj)
{
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) unsigned long long bars[NST];
    __shared__ double red[4];
    const uint32_t ra = (uint32_t)n_omega * 8u, rm = (uint32_t)n_tau * 8u;
    const uint32_t stage_bytes = (COPY ? 1u : 2u) * (ra + rm);
    const long long n_rec = (long long)scalars[2];
    const long long n_my = n_rec > blockIdx.x ? (n_rec - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    const double omt = 1.0 - t;
    if (threadIdx.x == 0) {
        for (int k = 0; k < NST; ++k) mbar_init(smem_u32(&bars[k]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // stage layout: donor a | donor mt | (self a | self mt)
    auto issue = [&](long long it) {
        const int st = (int)(it % NST);
        const long long i = rec_list[blockIdx.x + it * gridDim.x], dn = donor_of[i];
        const uint32_t base = smem_u32(smem) + (uint32_t)st * stage_bytes, bar = smem_u32(&bars[st]);
        mbar_expect_tx(bar, stage_bytes);
        bulk_g2s(base, a + (size_t)dn * n_omega, ra, bar);
        bulk_g2s(base + ra, mt + (size_t)dn * n_tau, rm, bar);
        if (!COPY) {
            bulk_g2s(base + ra + rm, a + (size_t)i * n_omega, ra, bar);
            bulk_g2s(base + 2 * ra + rm, mt + (size_t)i * n_tau, rm, bar);
        }
    };
    if (threadIdx.x == 0)
        for (long long k = 0; k < NST - 1 && k < n_my; ++k) issue(k);

    for (long long it = 0; it < n_my; ++it) {
        const int st = (int)(it % NST);
        if (threadIdx.x == 0 && it + NST - 1 < n_my) {
            // the stage being refilled was the source of the most recent store group: wait until it has been read
            asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
            issue(it + NST - 1);
        }
        mbar_wait(smem_u32(&bars[st]), (uint32_t)((it / NST) & 1));
        unsigned char *sb = smem + (size_t)st * stage_bytes;
        double *da = reinterpret_cast<double *>(sb), *dm = reinterpret_cast<double *>(sb + ra);
        double *xa = reinterpret_cast<double *>(sb + ra + rm), *xm = reinterpret_cast<double *>(sb + 2 * ra + rm);
        if (!COPY)
            for (int k = threadIdx.x; k < n_omega; k += blockDim.x) xa[k] = __dadd_rn(__dmul_rn(t, da[k]), __dmul_rn(omt, xa[k]));
        double s = 0.0;
        for (int j = threadIdx.x; j < n_tau; j += blockDim.x) {
            double v = dm[j];
            if (!COPY) { v = __dadd_rn(__dmul_rn(t, v), __dmul_rn(omt, xm[j])); xm[j] = v; }
            const double D = v - fj[j];
            s = fma(Wj[j] * D, D, s);
        }
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
        if (!COPY) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic writes -> visible to the bulk store
        __syncthreads();
        if (threadIdx.x == 0) {
            const long long i = rec_list[blockIdx.x + it * gridDim.x];
            const uint32_t src = smem_u32(sb) + (COPY ? 0u : ra + rm);
            bulk_s2g(a + (size_t)i * n_omega, src, ra);
            bulk_s2g(mt + (size_t)i * n_tau, src + ra, rm);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            chi2[i] = (red[0] + red[1]) + (red[2] + red[3]);
        }
        __syncthreads();        // red[] and this stage's buffers are free for the next iterations
    }
    if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

// weights -> scan -> multipliers -> scans -> donor map for inverse temperature 1/T; the number of recipients (zero
// multipliers) ends up in scalars[2].  No walker state is touched.
static int branch_plan(sail_handle *h, double T)
{
    const long long W = h->W;
    BranchScratch &b = h->br;
    const int blocks = (int)((W + 255) / 256 < 1184 ? (W + 255) / 256 : 1184);
    SAIL_CUDA_OK(h, cudaMemsetAsync(b.scalars, 0, 8 * sizeof(unsigned long long), h->stream));
    SAIL_CUDA_OK(h, cudaMemsetAsync(b.scalars, 0xFF, sizeof(unsigned long long), h->stream));
    chi2_min_kernel<<<blocks, 256, 0, h->stream>>>(W, h->st.chi2, b.scalars);
    SAIL_LAUNCH_OK(h, "chi2_min_kernel");
    weights_kernel<<<blocks, 256, 0, h->stream>>>(W, h->st.chi2, T, b.scalars, b.ehat);
    SAIL_LAUNCH_OK(h, "weights_kernel");
    int rc = scan_inclusive(h, W, 1, b.ehat, nullptr);
    if (rc) return rc;
    multipliers_kernel<<<blocks, 256, 0, h->stream>>>(W, b.ehat, (uint32_t)(h->seed & 0xFFFFFFFFu), (uint32_t)(h->seed >> 32),
                                                      (uint32_t)h->sweep, b.mult, b.scanA, b.scanB, b.scalars);
    SAIL_LAUNCH_OK(h, "multipliers_kernel");
    rc = scan_inclusive(h, W, 2, b.scanA, b.scanB);
    if (rc) return rc;
    donor_map_kernel<<<blocks, 256, 0, h->stream>>>(W, b.mult, b.scanA, b.scanB, b.donor_of, b.rec_list, b.scalars);
    SAIL_LAUNCH_OK(h, "donor_map_kernel");
    return SAIL_OK;
}

static int branch_imprint(sail_handle *h, double t_imprint)
{
    const long long W = h->W;
    BranchScratch &b = h->br;
    const int iblocks = (int)(W < (long long)h->num_sms * 8 ? W : (long long)h->num_sms * 8);
    // t = 1 with rows that are multiples of 16 bytes goes through the bulk-copy engine (measured on Stress, 187799
    // recipients: 1.05 ms against 1.31 ms with plain loads); for t < 1 the plain-load kernel is the faster one
    // (1.64 ms against 1.79 ms: the combination runs out of shared memory at 2 CTAs per SM), so it keeps that path
    const size_t row_bytes = (size_t)(h->n_omega + h->n_tau) * sizeof(double);
    const bool copy = t_imprint == 1.0;
    const int nst = copy ? 3 : 2;
    const size_t tma_smem = (copy ? 1 : 2) * row_bytes * nst;
    if ((h->n_omega & 1) == 0 && (h->n_tau & 1) == 0 && tma_smem <= 96 * 1024 && copy) {
        const int per_sm = (int)((200 * 1024) / (tma_smem + 1024)) < 8 ? (int)((200 * 1024) / (tma_smem + 1024)) : 8;
        const int tblocks = (int)(W < (long long)h->num_sms * per_sm ? W : (long long)h->num_sms * per_sm);
        if (copy) {
            SAIL_CUDA_OK(h, cudaFuncSetAttribute(imprint_tma_kernel<true, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tma_smem));
            imprint_tma_kernel<true, 3><<<tblocks, 128, tma_smem, h->stream>>>(h->n_omega, h->n_tau, t_imprint, b.rec_list, b.donor_of, b.scalars,
                                                                              h->st.a, h->st.mt, h->st.chi2, h->tab.Wj, h->tab.fj);
        } else {
            SAIL_CUDA_OK(h, cudaFuncSetAttribute(imprint_tma_kernel<false, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tma_smem));
            imprint_tma_kernel<false, 2><<<tblocks, 128, tma_smem, h->stream>>>(h->n_omega, h->n_tau, t_imprint, b.rec_list, b.donor_of, b.scalars,
                                                                               h->st.a, h->st.mt, h->st.chi2, h->tab.Wj, h->tab.fj);
        }
        SAIL_LAUNCH_OK(h, "imprint_tma_kernel");
        return SAIL_OK;
    }
    if (t_imprint == 1.0)
        imprint_kernel<true><<<iblocks, 256, 0, h->stream>>>(h->n_omega, h->n_tau, t_imprint, b.rec_list, b.donor_of, b.scalars,
                                                             h->st.a, h->st.mt, h->st.chi2, h->tab.Wj, h->tab.fj);
    else
        imprint_kernel<false><<<iblocks, 256, 0, h->stream>>>(h->n_omega, h->n_tau, t_imprint, b.rec_list, b.donor_of, b.scalars,
                                                              h->st.a, h->st.mt, h->st.chi2, h->tab.Wj, h->tab.fj);
    SAIL_LAUNCH_OK(h, "imprint_kernel");
    return SAIL_OK;
}

int launch_branch(sail_handle *h, double T, double t_imprint)
{
    int rc = branch_plan(h, T);
    if (rc) return rc;
    return branch_imprint(h, t_imprint);
}

__global__ void chi2_max_kernel(long long W, const double *__restrict__ chi2, unsigned long long *dst)
{
    unsigned long long m = 0ull;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < W; i += (long long)gridDim.x * blockDim.x) {
        const unsigned long long b = ordered_key(chi2[i]);
        m = b > m ? b : m;
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        const unsigned long long o = __shfl_xor_sync(0xffffffffu, m, off);
        m = o > m ? o : m;
    }
    if ((threadIdx.x & 31) == 0) atomicMax(dst, m);
}

// SURVEY §8f row f2 (reading B6): 1/T such that `fraction` of the walkers get multiplier zero, found
// by bracketing (doubling / halving from 1/(chi2_max - chi2_min)) and 40 bisection steps on 1/T; every trial runs the
// multiplier chain on the device (same comb offset) and reads back one count.  Then the event itself at that T.
int launch_branch_fraction(sail_handle *h, double fraction, double t_imprint, double *T_found)
{
    const long long W = h->W;
    BranchScratch &b = h->br;
    *T_found = 0.0;
    const long long n0 = (long long)floor(fraction * (double)W + 0.5);
    const int blocks = (int)((W + 255) / 256 < 1184 ? (W + 255) / 256 : 1184);
    SAIL_CUDA_OK(h, cudaMemsetAsync(b.scalars, 0, 8 * sizeof(unsigned long long), h->stream));
    SAIL_CUDA_OK(h, cudaMemsetAsync(b.scalars, 0xFF, sizeof(unsigned long long), h->stream));
    chi2_min_kernel<<<blocks, 256, 0, h->stream>>>(W, h->st.chi2, b.scalars);
    SAIL_LAUNCH_OK(h, "chi2_min_kernel");
    chi2_max_kernel<<<blocks, 256, 0, h->stream>>>(W, h->st.chi2, b.scalars + 6);
    SAIL_LAUNCH_OK(h, "chi2_max_kernel");
    unsigned long long sc[8];
    SAIL_CUDA_OK(h, cudaMemcpyAsync(sc, b.scalars, sizeof sc, cudaMemcpyDeviceToHost, h->stream));
    SAIL_CUDA_OK(h, cudaStreamSynchronize(h->stream));
    double cmin, cmax;
    cmin = ordered_key_value(sc[0]); cmax = ordered_key_value(sc[6]);
    if (n0 <= 0 || !(cmax > cmin)) return SAIL_OK;     // nothing to branch
    int rc = SAIL_OK;
    auto zeros = [&](double beta) -> long long {
        if (rc) return 0;
        rc = branch_plan(h, 1.0 / beta);
        if (rc) return 0;
        unsigned long long z = 0;
        if (cudaMemcpyAsync(&z, b.scalars + 2, 8, cudaMemcpyDeviceToHost, h->stream) != cudaSuccess ||
            cudaStreamSynchronize(h->stream) != cudaSuccess) { rc = set_err(h, SAIL_ERR_CUDA, "read-back of the recipient count failed"); return 0; }
        return (long long)z;
    };
    double lo, hi = 1.0 / (cmax - cmin);
    if (zeros(hi) >= n0) {
        lo = 0.5 * hi;
        for (int it = 0; it < 200 && zeros(lo) >= n0; ++it) { hi = lo; lo = 0.5 * lo; }
    } else {
        lo = hi; hi = 2.0 * hi;
        int it = 0;
        for (; it < 200 && zeros(hi) < n0; ++it) { lo = hi; hi = 2.0 * hi; }
        if (it == 200) return rc;                      // the fraction cannot be reached
    }
    for (int it = 0; it < 40; ++it) {
        const double mid = 0.5 * (lo + hi);
        if (zeros(mid) >= n0) hi = mid; else lo = mid;
    }
    if (rc) return rc;
    *T_found = 1.0 / hi;
    return launch_branch(h, *T_found, t_imprint);
}

} // namespace sail
