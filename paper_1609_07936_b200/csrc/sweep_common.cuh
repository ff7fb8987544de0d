// sweep_common.cuh — helpers of the sweep kernel (sweep.cu): launch arguments, PTX accessors, the DMMA warp sum,
// the staged proposal (row A2) and Eq. 30.  Not part of the ABI.
#pragma once
#include "sail_internal.cuh"

namespace sail {

struct SweepArgs {
    int n_omega, n_tau;
    long long W;
    long long walker0;                 // global index of this handle's walker 0 (Philox counter word 0)
    double A, B, domega, eta, amp_p, amp_m, y_min;
    int amp_mode;
    uint32_t seed_lo, seed_hi;
    const double *Wj, *fj, *ratio, *E0, *invd, *omega;
    int fact, fact_shift, n_hi, n_lo;
    double *a, *mt, *chi2, *y;
    unsigned long long *n_acc, *n_eval;
    const double *T;
    long long sweep0;
    int n_sweeps;
    int walk_len;                      // length of the index-selection walk (section 2.3); 0 = uniform indices
    int spec_smem;                     // WALK: every warp keeps a copy of its walker's spectrum in shared memory
    double walk_uniform;               // fraction of moves that keep the uniform indices (:158)
    long long trace_lo, trace_hi;
    sail_trace_rec *trace;
    uint8_t *flags;
    long long call_sweeps, call_off;   // sweeps in the whole sail_anneal call / offset of this launch
};

// 1/x for x close to 1 (|x - 1| < 0.5): hardware seed + two Newton steps, relative error ~1e-16.
__device__ __forceinline__ double fast_recip(double x)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    double e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    e = fma(-x, r, 1.0);
    return fma(r, e, r);
}

// shared-memory accesses by 32-bit shared-window address (no generic-address arithmetic in the hot loop)
__device__ __forceinline__ double lds_f64(uint32_t addr)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ double2 lds_f64x2(uint32_t addr)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ int4 lds_s32x4(uint32_t addr)
{
    int4 v;
    asm volatile("ld.shared.v4.s32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}

// element pointer a + idx (idx < 2^32) in one IMAD.WIDE
__device__ __forceinline__ double *elem_ptr(double *base, uint32_t idx)
{
    unsigned long long r;
    asm("mad.wide.u32 %0, %1, 8, %2;" : "=l"(r) : "r"(idx), "l"(reinterpret_cast<unsigned long long>(base)));
    return reinterpret_cast<double *>(r);
}
__device__ __forceinline__ double ldg_f64(const double *p)
{
    double v;
    asm volatile("ld.global.f64 %0, [%1];" : "=d"(v) : "l"(p) : "memory");
    return v;
}
// generic-address load (shared or global), never cached in a register across a warp synchronisation
__device__ __forceinline__ double ld_f64(const double *p)
{
    double v;
    asm volatile("ld.f64 %0, [%1];" : "=d"(v) : "l"(p) : "memory");
    return v;
}
// predicated (not branched) store: only the lanes with pred != 0 write
__device__ __forceinline__ void stg_f64_if(double *p, double v, int pred)
{
    asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.s32 q, %2, 0;\n\t@q st.global.f64 [%0], %1;\n\t}" :: "l"(p), "d"(v), "r"(pred) : "memory");
}

// Sum of one double per lane over the whole warp, result in every lane, on the FP64 tensor-core path (DMMA, no
// shuffles): D = ones(8x4) . B(4x8) with B[k = lane%4][n = lane/4] = x puts the 8 column sums in every row of D;
// a lane owns columns 2(lane%4), 2(lane%4)+1, and their sum h(lane%4), fed through the same product, is the total.
// Measured on B200 (sail_microbench): a DMMA m8n8k4 occupies the FP64 pipe like 8 DFMAs (it has no unit of its own);
// the two products + DADD take ~77 cycles of latency against ~190 for the 5-stage shuffle butterfly.
__device__ __forceinline__ double warp_sum_dmma(double x)
{
    double c0, c1, t0, t1;
    const double one = 1.0, zero = 0.0;
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%4,%4};"
        : "=d"(c0), "=d"(c1) : "d"(one), "d"(x), "d"(zero));
    const double h = c0 + c1;
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%4,%4};"
        : "=d"(t0), "=d"(t1) : "d"(one), "d"(h), "d"(zero));
    (void)t1;
    return t0;
}

// Eq. 30: y from the sweep's acceptance rate
__device__ __forceinline__ double amp_factor(const SweepArgs &P, int acc_sweep, double y)
{
    if (P.amp_mode != 1) return y;
    const double rate = (double)acc_sweep / (double)P.n_omega;
    if (rate >= P.amp_p) return 1.0;
    const double x = rate / P.amp_p;
    const double yy = (P.amp_m == 2.0) ? x * x : pow(x, P.amp_m);
    return yy < P.y_min ? P.y_min : yy;
}

__device__ __forceinline__ double u01(uint32_t x) { return ((double)x + 0.5) * 2.3283064365386962890625e-10; }

// One staged proposal in shared memory (80 bytes; 112 with the index walk):
//   [ 0] p, s (int32), alpha = rho - 1   [16] delta_p, delta_s (Eq. 20-21)   [32] delta_p r_p, delta_s r_s
//   [48] r_p + r_s, -(r_p r_s)           [64] thr = -T ln u_acc, 1/rho
//   [80] [96] (walk only) the Philox words of the first two walk steps
constexpr int kRecBytes = 80;
constexpr int kRecWalkBytes = 112;

// the index-dependent half of a proposal: Eq. 20-21 in the method's operation order (only the division by
// (p - s) domega is a multiplication by the correctly rounded reciprocal: delta within 2 ulp of the division form) and
// the coefficients of the two-term recurrence of delta_p E_p + delta_s E_s along a lane's tau-points
__device__ __forceinline__ void write_indexed(const SweepArgs &P, int p, int s, double alpha, const double *s_ratio,
                                              const double *s_invd, double wm_s, double wm_p, unsigned char *rec)
{
    const double omr = -alpha;                           // 1 - rho, exact like alpha = rho - 1
    const int dps = p - s;
    const double inv = (dps > 0) ? s_invd[dps] : -s_invd[-dps];
    const double dp = __dmul_rn(__dmul_rn(omr, __dsub_rn(P.B, __dmul_rn(P.A, wm_s))), inv);
    const double ds = -__dmul_rn(__dmul_rn(omr, __dsub_rn(P.B, __dmul_rn(P.A, wm_p))), inv);
    const double rp = s_ratio[p], rs = s_ratio[s];
    *reinterpret_cast<int4 *>(rec) = make_int4(p, s, __double2loint(alpha), __double2hiint(alpha));
    *reinterpret_cast<double2 *>(rec + 16) = make_double2(dp, ds);
    *reinterpret_cast<double2 *>(rec + 32) = make_double2(dp * rp, ds * rs);
    *reinterpret_cast<double2 *>(rec + 48) = make_double2(rp + rs, -(rp * rs));
}

} // namespace sail
