// branch.cu — imprinted branching (Eq. 24-26; readings B1-B5 in
// DESIGN.md §2): fixed-point weights -> integer prefix sum -> comb multipliers (sum m = W exactly) ->
// donor map by binary search -> coalesced 128-bit imprint copy of (spectrum, model) + residue.
#include "sail_internal.cuh"
#include <cooperative_groups.h>
#include <math.h>
#include <string.h>

namespace sail {

namespace cg = cooperative_groups;

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

// ---- the whole multiplier plan of one branching event in ONE cooperative kernel -----------------------------------
// weights (B1, B3) -> u64 inclusive scan -> comb multipliers (B2) -> scans of recipient flags and donor extras -> donor
// map (B4), with grid-wide barriers between the phases instead of kernel boundaries; in the search modes the first two
// phases run once per trial of 1/T (reading B6: bracketing by doubling / halving from 1/(chi2_max - chi2_min), then 40
// bisection steps; fp64 arithmetic steered by integer counts, identical on every CTA, so the grid stays in step).
// Every CTA owns a contiguous chunk of walkers; all integer arithmetic is order independent, so the multipliers are the
// ones of the definition bit for bit.
constexpr int kPlanThreads = 512;
constexpr int kPlanWarps = kPlanThreads / 32;

struct PlanArgs {
    long long W;
    const double *chi2;
    int mode;                          // 0: T given; 1: search for `fraction`; 2 / 3: the same with T / fraction from ctl[0] / ctl[1]
    double T, fraction;
    const double *ctl;                 // DEVICE (T, fraction) of modes 2, 3
    uint32_t seed_lo, seed_hi, sweep;
    unsigned long long *ehat, *scanA, *scanB, *part, *scalars;
    int32_t *mult;
    int64_t *donor_of, *rec_list;
};

__device__ __forceinline__ unsigned long long warp_incl_scan(unsigned long long v, int lane)
{
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const unsigned long long o = __shfl_up_sync(0xffffffffu, v, off);
        if (lane >= off) v += o;
    }
    return v;
}
// inclusive scan of one value per thread over the CTA; *total = sum over the CTA (sm: kPlanWarps slots, reusable after return)
__device__ __forceinline__ unsigned long long block_incl_scan(unsigned long long v, unsigned long long *sm, unsigned long long *total)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const unsigned long long inc = warp_incl_scan(v, lane);
    if (lane == 31) sm[wid] = inc;
    __syncthreads();
    unsigned long long prefix = 0, tot = 0;
#pragma unroll
    for (int w2 = 0; w2 < kPlanWarps; ++w2) { const unsigned long long t = sm[w2]; if (w2 < wid) prefix += t; tot += t; }
    __syncthreads();
    *total = tot;
    return inc + prefix;
}
template <int OP>   // 0 sum, 1 min, 2 max
__device__ __forceinline__ unsigned long long block_reduce(unsigned long long v, unsigned long long *sm)
{
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        const unsigned long long o = __shfl_xor_sync(0xffffffffu, v, off);
        v = (OP == 0) ? v + o : (OP == 1) ? (o < v ? o : v) : (o > v ? o : v);
    }
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
    __syncthreads();
    unsigned long long r = sm[0];
#pragma unroll
    for (int w2 = 1; w2 < kPlanWarps; ++w2) { const unsigned long long o = sm[w2]; r = (OP == 0) ? r + o : (OP == 1) ? (o < r ? o : r) : (o > r ? o : r); }
    __syncthreads();
    return r;
}
// (sum of part[0..n), sum of part[0..me)) — every thread gets both
__device__ __forceinline__ void grid_totals(const unsigned long long *part, int n, int me, unsigned long long *sm,
                                            unsigned long long *total, unsigned long long *before)
{
    unsigned long long t = 0, b = 0;
    for (int c = threadIdx.x; c < n; c += blockDim.x) { const unsigned long long v = part[c]; t += v; if (c < me) b += v; }
    *total = block_reduce<0>(t, sm);
    *before = block_reduce<0>(b, sm);
}

__global__ void __launch_bounds__(kPlanThreads) branch_plan_kernel(const PlanArgs a)
{
    cg::grid_group grid = cg::this_grid();
    __shared__ unsigned long long sm[kPlanWarps];
    __shared__ unsigned long long sm_hi[kPlanThreads + 1];
    const int G = gridDim.x, me = blockIdx.x, tid = threadIdx.x;
    const long long W = a.W;
    const long long chunk = (W + G - 1) / G;
    const long long c0 = (long long)me * chunk < W ? (long long)me * chunk : W;
    const long long c1 = c0 + chunk < W ? c0 + chunk : W;
    unsigned long long *pE = a.part, *pZ = a.part + G, *pX = a.part + 2 * G, *pMin = a.part + 3 * G, *pMax = a.part + 4 * G, *pM = a.part + 5 * G;

    // ---- smallest / largest residue --------------------------------------------------------------------
    unsigned long long kmin = ~0ull, kmax = 0ull;
    for (long long i = c0 + tid; i < c1; i += kPlanThreads) {
        const unsigned long long k = ordered_key(a.chi2[i]);
        kmin = k < kmin ? k : kmin;
        kmax = k > kmax ? k : kmax;
    }
    kmin = block_reduce<1>(kmin, sm);
    kmax = block_reduce<2>(kmax, sm);
    if (tid == 0) { pMin[me] = kmin; pMax[me] = kmax; }
    grid.sync();
    kmin = ~0ull; kmax = 0ull;
    for (int c = tid; c < G; c += kPlanThreads) { kmin = pMin[c] < kmin ? pMin[c] : kmin; kmax = pMax[c] > kmax ? pMax[c] : kmax; }
    kmin = block_reduce<1>(kmin, sm);
    kmax = block_reduce<2>(kmax, sm);
    const double cmin = key_value(kmin), cmax = key_value(kmax);

    uint32_t x[4];
    philox4x32_10(0u, a.sweep, 0u, 1u, a.seed_lo, a.seed_hi, x);

    // one pass of the multiplier chain at temperature T; final: also multipliers, recipient / extras scans.
    // Returns the number of zero multipliers over the whole population.
    auto pass = [&](double T, bool final) -> unsigned long long {
        // B1 + B3: e_i = exp(-(chi2_i - chi2_min)/T), E_i = floor(e_i 2^40); inclusive scan within the chunk
        unsigned long long carry = 0;
        for (long long t0 = c0; t0 < c1; t0 += kPlanThreads) {
            const long long i = t0 + tid;
            unsigned long long E = 0;
            if (i < c1) {
                // chi2_i >= chi2_min makes the exponent <= 0 and the weight <= 2^40; a NaN residue gets weight 0
                const double e = exp(-(a.chi2[i] - cmin) / T);
                E = (e == e) ? (unsigned long long)floor(fmin(e, 1.0) * 1099511627776.0) : 0ull;
            }
            unsigned long long tot;
            const unsigned long long inc = block_incl_scan(E, sm, &tot);
            if (i < c1) a.ehat[i] = inc + carry;
            carry += tot;
        }
        if (tid == 0) pE[me] = carry;
        grid.sync();
        unsigned long long S, off;
        grid_totals(pE, G, me, sm, &S, &off);
        // B2: comb multipliers m_i = floor((C_i W + Xi)/S) - floor((C_{i-1} W + Xi)/S), Xi = (x0 S) >> 32
        const unsigned __int128 Xi = ((unsigned __int128)x[0] * S) >> 32;
        auto comb = [&](unsigned long long C) { return (unsigned long long)(((unsigned __int128)C * (unsigned long long)W + Xi) / S); };
        unsigned long long prev_hi = comb(off);          // C_{c0-1} = the sum of the chunks before this one
        unsigned long long zeros = 0, rec_carry = 0, ext_carry = 0;
        int mmax = 0;
        for (long long t0 = c0; t0 < c1; t0 += kPlanThreads) {
            const long long i = t0 + tid;
            const unsigned long long hi = (i < c1) ? comb(a.ehat[i] + off) : 0ull;
            sm_hi[tid + 1] = hi;
            if (tid == 0) sm_hi[0] = prev_hi;
            __syncthreads();
            const int m = (i < c1) ? (int)(hi - sm_hi[tid]) : 1;
            const long long last = (c1 - t0 < kPlanThreads ? c1 - t0 : kPlanThreads);
            prev_hi = sm_hi[last];
            __syncthreads();
            if (i < c1 && m == 0) zeros++;
            if (final) {
                unsigned long long tr, te;
                const unsigned long long ri = block_incl_scan((i < c1 && m == 0) ? 1ull : 0ull, sm, &tr);
                const unsigned long long xi = block_incl_scan((i < c1 && m > 1) ? (unsigned long long)(m - 1) : 0ull, sm, &te);
                if (i < c1) { a.mult[i] = m; a.scanA[i] = ri + rec_carry; a.scanB[i] = xi + ext_carry; }
                rec_carry += tr; ext_carry += te;
                if (i < c1) mmax = m > mmax ? m : mmax;
            }
        }
        zeros = block_reduce<0>(zeros, sm);
        if (final) mmax = (int)block_reduce<2>((unsigned long long)mmax, sm);
        if (tid == 0) { pZ[me] = zeros; if (final) { pX[me] = ext_carry; pM[me] = (unsigned long long)mmax; } }
        if (final && me == 0 && tid == 0) a.scalars[1] = S;
        grid.sync();
        unsigned long long zt = 0;
        for (int c = tid; c < G; c += kPlanThreads) zt += pZ[c];
        return block_reduce<0>(zt, sm);
    };

    // ---- temperature: given, or searched (reading B6) ------------------------------------------------------------
    double T = (a.mode == 2) ? a.ctl[0] : a.T;
    // a population whose smallest residue is not finite (all NaN, or -inf) has no weights: every E_i would be 0 and the
    // comb would divide by S = 0.  No event then (identical on every CTA, so the grid leaves together).
    bool event = isfinite(cmin) && (a.mode == 1 || a.mode == 3 || T > 0.0);
    if (a.mode == 1 || a.mode == 3) {
        const double fraction = (a.mode == 3) ? a.ctl[1] : a.fraction;
        const long long n0 = (long long)floor(fraction * (double)W + 0.5);
        T = 0.0;
        event = event && n0 > 0 && cmax > cmin;
        if (event) {
            double lo, hi = 1.0 / (cmax - cmin);
            if ((long long)pass(1.0 / hi, false) >= n0) {
                lo = 0.5 * hi;
                for (int it = 0; it < 200 && (long long)pass(1.0 / lo, false) >= n0; ++it) { hi = lo; lo = 0.5 * lo; }
            } else {
                lo = hi; hi = 2.0 * hi;
                int it = 0;
                for (; it < 200 && (long long)pass(1.0 / hi, false) < n0; ++it) { lo = hi; hi = 2.0 * hi; }
                if (it == 200) event = false;                // the fraction cannot be reached
            }
            if (event) {
                for (int it = 0; it < 40; ++it) {
                    const double mid = 0.5 * (lo + hi);
                    if ((long long)pass(1.0 / mid, false) >= n0) hi = mid; else lo = mid;
                }
                T = 1.0 / hi;
            }
        }
    }
    if (!event) {                                            // degenerate population or nothing asked for: no recipients
        if (me == 0 && tid == 0) {
            a.scalars[0] = kmin; a.scalars[1] = 0; a.scalars[2] = 0; a.scalars[3] = 1;
            a.scalars[5] = (unsigned long long)__double_as_longlong(0.0);
        }
        for (long long i = c0 + tid; i < c1; i += kPlanThreads) { a.mult[i] = 1; a.donor_of[i] = -1; }
        return;
    }
    const unsigned long long n_rec = pass(T, true);
    // ---- recipient ranks and donor extras: chunk-local scans -> global (B4) ----------------------------------------
    unsigned long long tot_r, off_r, tot_x, off_x;
    grid_totals(pZ, G, me, sm, &tot_r, &off_r);
    grid_totals(pX, G, me, sm, &tot_x, &off_x);
    for (long long i = c0 + tid; i < c1; i += kPlanThreads) { a.scanA[i] += off_r; a.scanB[i] += off_x; }
    unsigned long long mm = 0;
    for (int c = tid; c < G; c += kPlanThreads) mm = pM[c] > mm ? pM[c] : mm;
    mm = block_reduce<2>(mm, sm);
    if (me == 0 && tid == 0) {
        a.scalars[0] = kmin; a.scalars[2] = n_rec; a.scalars[3] = mm;
        a.scalars[5] = (unsigned long long)__double_as_longlong(T);
    }
    grid.sync();
    // recipient of rank r takes the donor with X_i <= r < X_i + x_i (binary search on the inclusive scan of the extras)
    for (long long i = c0 + tid; i < c1; i += kPlanThreads) {
        long long donor = -1;
        if (a.mult[i] == 0) {
            const unsigned long long r = a.scanA[i] - 1;
            long long lo = 0, hi = W - 1;            // first index with ext_inc > r
            while (lo < hi) {
                const long long mid = (lo + hi) >> 1;
                if (a.scanB[mid] > r) hi = mid; else lo = mid + 1;
            }
            donor = lo;
            a.rec_list[r] = i;
        }
        a.donor_of[i] = donor;
    }
}

// Eq. 26: a(l1) <- t a(l2) + (1-t) a(l1) for spectrum and model (linearity).  One CTA per recipient,
// 128-bit accesses when rows are 16-byte aligned: a and mt of the recipient become t * donor + (1 - t) * self (two roundings per product
// and one per sum, exactly the definition), chi^2 is recomputed from the new model.  COPY (t == 1): t * z + 0 * x
// is z bit for bit, so the recipient is not read at all (two streams instead of three).  All loads of a CTA's
// pass are issued before its first store (8 x 16 B per thread in flight).
template <bool COPY>
__global__ void __launch_bounds__(256) imprint_kernel(int n_omega, int n_tau, double t_arg, const double *t_dev, const int64_t *__restrict__ rec_list,
                                                      const int64_t *__restrict__ donor_of, const unsigned long long *scalars,
                                                      double *a, double *mt, double *chi2,
                                                      const double *__restrict__ Wj, const double *__restrict__ fj)
{
    __shared__ double red[8];
    const long long n_rec = (long long)scalars[2];
    const double t = t_dev ? *t_dev : t_arg;           // t on the device: the self-cooling protocol (B7)
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

// the multiplier plan (one cooperative launch); the number of recipients ends up in scalars[2], the temperature used
// in scalars[5].  No walker state is touched.  mode / T / fraction / ctl as in PlanArgs.
static int branch_plan(sail_handle *h, int mode, double T, double fraction, const double *ctl)
{
    BranchScratch &b = h->br;
    PlanArgs a{};
    a.W = h->W; a.chi2 = h->st.chi2; a.mode = mode; a.T = T; a.fraction = fraction; a.ctl = ctl;
    a.seed_lo = (uint32_t)(h->seed & 0xFFFFFFFFu); a.seed_hi = (uint32_t)(h->seed >> 32); a.sweep = (uint32_t)h->sweep;
    a.ehat = b.ehat; a.scanA = b.scanA; a.scanB = b.scanB; a.part = b.block_sums; a.scalars = b.scalars;
    a.mult = b.mult; a.donor_of = b.donor_of; a.rec_list = b.rec_list;
    if (h->plan_ctas == 0) {
        int per_sm = 0;
        SAIL_CUDA_OK(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, branch_plan_kernel, kPlanThreads, 0));
        if (per_sm < 1) return set_err(h, SAIL_ERR_CUDA, "branch_plan_kernel does not fit an SM");
        h->plan_ctas = h->num_sms;                     // one CTA per SM: all co-resident (cooperative launch)
    }
    int ctas = h->plan_ctas;
    const long long need = (h->W + kPlanThreads - 1) / kPlanThreads;
    if (need < ctas) ctas = (int)(need < 1 ? 1 : need);
    void *args[] = {(void *)&a};
    SAIL_CUDA_OK(h, cudaLaunchCooperativeKernel((const void *)branch_plan_kernel, dim3(ctas), dim3(kPlanThreads), args, 0, h->stream));
    h->launches++;
    return SAIL_OK;
}

static int branch_imprint(sail_handle *h, double t_imprint, const double *t_dev)
{
    const long long W = h->W;
    BranchScratch &b = h->br;
    const int iblocks = (int)(W < (long long)h->num_sms * 8 ? W : (long long)h->num_sms * 8);
    // t = 1 with rows that are multiples of 16 bytes goes through the bulk-copy engine (measured on Stress, 187799
    // recipients: 1.05 ms against 1.31 ms with plain loads); for t < 1 the plain-load kernel is the faster one
    // (1.64 ms against 1.79 ms: the combination runs out of shared memory at 2 CTAs per SM), so it keeps that path
    const size_t row_bytes = (size_t)(h->n_omega + h->n_tau) * sizeof(double);
    const bool copy = t_imprint == 1.0 && !t_dev;
    const int nst = copy ? 3 : 2;
    const size_t tma_smem = (copy ? 1 : 2) * row_bytes * nst;
    if ((h->n_omega & 1) == 0 && (h->n_tau & 1) == 0 && tma_smem <= 96 * 1024 && copy) {
        const int per_sm = (int)((200 * 1024) / (tma_smem + 1024)) < 8 ? (int)((200 * 1024) / (tma_smem + 1024)) : 8;
        const int tblocks = (int)(W < (long long)h->num_sms * per_sm ? W : (long long)h->num_sms * per_sm);
        SAIL_CUDA_OK(h, cudaFuncSetAttribute(imprint_tma_kernel<true, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tma_smem));
        imprint_tma_kernel<true, 3><<<tblocks, 128, tma_smem, h->stream>>>(h->n_omega, h->n_tau, t_imprint, b.rec_list, b.donor_of, b.scalars,
                                                                          h->st.a, h->st.mt, h->st.chi2, h->tab.Wj, h->tab.fj);
        SAIL_LAUNCH_OK(h, "imprint_tma_kernel");
        return SAIL_OK;
    }
    if (copy)
        imprint_kernel<true><<<iblocks, 256, 0, h->stream>>>(h->n_omega, h->n_tau, t_imprint, nullptr, b.rec_list, b.donor_of, b.scalars,
                                                             h->st.a, h->st.mt, h->st.chi2, h->tab.Wj, h->tab.fj);
    else
        imprint_kernel<false><<<iblocks, 256, 0, h->stream>>>(h->n_omega, h->n_tau, t_imprint, t_dev, b.rec_list, b.donor_of, b.scalars,
                                                              h->st.a, h->st.mt, h->st.chi2, h->tab.Wj, h->tab.fj);
    SAIL_LAUNCH_OK(h, "imprint_kernel");
    return SAIL_OK;
}

int launch_branch(sail_handle *h, double T, double t_imprint)
{
    int rc = branch_plan(h, 0, T, 0.0, nullptr);
    if (rc) return rc;
    return branch_imprint(h, t_imprint, nullptr);
}

// SURVEY §8f row f2 (reading B6): 1/T such that `fraction` of the walkers get multiplier zero, found
// inside the plan kernel (bracketing + 40 bisection steps, every trial a pass of the multiplier chain with the same comb
// offset), then the event itself at that T.  The temperature found stays on the device (scalars[5]).
int launch_branch_fraction(sail_handle *h, double fraction, double t_imprint)
{
    int rc = branch_plan(h, 1, 0.0, fraction, nullptr);
    if (rc) return rc;
    return branch_imprint(h, t_imprint, nullptr);
}

// the same two events with their parameters on the device: ctl = (T, fraction, t_imprint) written by an earlier kernel
// on the stream (the self-cooling protocol: no host round trip inside a block)
int launch_branch_ctl(sail_handle *h, bool by_fraction, const double *ctl)
{
    int rc = branch_plan(h, by_fraction ? 3 : 2, 0.0, 0.0, ctl);
    if (rc) return rc;
    return branch_imprint(h, 0.5, ctl + 2);
}

} // namespace sail
