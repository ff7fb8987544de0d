// sail_internal.cuh — internals of libsail_b200 (sm_100a). Not part of the ABI; see include/sail.h.
// Shares nothing with oracle/ (the CPU oracle): tables, Philox and all arithmetic are restated here.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>
#include <string>
#include <vector>

#include "../../include/sail.h"

namespace sail {

constexpr int kSelfcoolBlocksMax = 4096;   // blocks of the self-cooling protocol whose (T, chi2_ave, chi2_min) are kept on the device per pass
constexpr int kMaxTau = 512;        // 32 lanes x 16 tau-points per lane (register-resident residual)
constexpr int kMaxOmega = 8192;     // sweep-kernel tables (ratio, 1/(k domega), start values) + proposal records fit 227 KB of shared memory

// ------------------------------------------------------------------------------------------------
// Device-side layout of one handle.  All arrays live in ONE workspace (caller- or library-owned).
// Residual state is kept in the "pure exponential" basis:
//   mt_j  = M_j / c_j = sum_k a_k exp(-omega_k tau_j)          (so kernel rows are geometric in j)
//   Wj    = (c_j / sigma_j)^2,   fj = F_j / c_j,   chi^2 = sum_j Wj (mt_j - fj)^2
// ------------------------------------------------------------------------------------------------
struct DevTables {
    const double *omega;   // [n_omega] bin left edges
    const double *tau;     // [n_tau]
    const double *c;       // [n_tau]  Eq. 8
    const double *Wj;      // [n_tau]
    const double *fj;      // [n_tau]
    const double *E;       // [n_omega][n_tau] exp(-omega_k tau_j), for the dense forward transform
    double *ET;            // [n_tau][n_omega] the same, transposed (k contiguous: the B operand of the DMMA forward kernel)
};

struct DevState {
    double *a;             // [W][n_omega] true spectral coefficients (scale folded at kernel end)
    double *mt;            // [W][n_tau]
    double *chi2;          // [W]
    double *y;             // [W] Eq. 30 amplitude factor
    unsigned long long *n_acc;   // [W] accepted moves since init
    unsigned long long *n_eval;  // [W] feasible (evaluated) moves since init
};

struct BranchScratch {
    unsigned long long *ehat;    // [W] fixed-point weights, then inclusive scan (in place)
    unsigned long long *scanA;   // [W] scan of recipient flags
    unsigned long long *scanB;   // [W] scan of donor extras
    unsigned long long *block_sums; // [6 * 1024] per-CTA partials of the cooperative branching-plan kernel (<= 1024 CTAs)
    int32_t *mult;               // [W]
    int64_t *donor_of;           // [W]
    int64_t *rec_list;           // [W] recipient indices in ascending order
    unsigned long long *scalars; // [8]: 0 chi2_min (ordered key), 1 S, 2 n_rec, 3 max_mult, 4 (chi2 statistics), 5 T used (double bits), 6-7 scratch
};

} // namespace sail

struct sail_handle {
    int device = 0;
    cudaStream_t stream = nullptr;
    int num_sms = 0;
    int n_omega = 0, n_tau = 0;
    int64_t max_walkers = 0, W = 0;
    double omega0 = 0, domega = 0, tau0 = 0, dtau = 0;
    double A = 0, B = 0;
    std::vector<double> omega_host;   // the caller's omega grid (sail_create copies it)
    uint64_t seed = 0;
    int64_t sweep = 0;          // absolute sweep counter
    int64_t walker0 = 0;        // global index of walker 0 (sail_set_walker_offset)
    bool initialised = false;

    void *workspace = nullptr;  // base of everything below
    size_t workspace_bytes = 0;
    bool owns_workspace = false;

    sail::DevTables tab{};
    sail::DevState st{};
    sail::BranchScratch br{};
    // sweep-kernel tables (built by the first sail_anneal)
    bool tables_ready = false;
    int plan_ctas = 0;           // grid of the cooperative branching-plan kernel (all CTAs co-resident)
    bool tables_fact = false;
    int fact_shift = 0;
    double *sw_ratio = nullptr;  // [n_omega] exp(-omega_k G dtau)
    double *sw_invd = nullptr;   // [n_omega] 1/(k domega)
    double *sw_E0 = nullptr;     // direct: [n_omega][G]; factored: H[n_hi][G] then L[n_lo][G]
    double *d_T = nullptr;       // device copy of the schedule piece in flight (a fixed slice of the workspace)
    size_t d_T_cap = 0;
    double *ctl = nullptr;             // [32] device control block: 0 T, 1 branching fraction, 2 imprint strength (branch.cu), 8.. self-cooling state (selfcool.cu)
    double *block_out = nullptr;       // [3][kSelfcoolBlocksMax] T, chi2_ave, chi2_min per block of the self-cooling protocol
    const double *halt = nullptr;      // DEVICE flag (ctl[12]) while sail_anneal_selfcool runs: non-zero = its rule failed, later work is skipped
    double *model_scratch = nullptr;   // [max_walkers][n_tau]: sail_get_model's scaled copy M = c mt for the host

    int64_t launches = 0;
    std::string err;
};

namespace sail {

// ---- error helpers -------------------------------------------------------------------------------
int set_err(sail_handle *h, int code, const char *fmt, ...);
#define SAIL_CUDA_OK(h, expr)                                                                    \
    do {                                                                                         \
        cudaError_t e__ = (expr);                                                                \
        if (e__ != cudaSuccess)                                                                  \
            return sail::set_err((h), SAIL_ERR_CUDA, "%s failed: %s (%s:%d)", #expr,             \
                                 cudaGetErrorString(e__), __FILE__, __LINE__);                   \
    } while (0)
#define SAIL_LAUNCH_OK(h, what)                                                                  \
    do {                                                                                         \
        cudaError_t e__ = cudaGetLastError();                                                    \
        (h)->launches++;                                                                         \
        if (e__ != cudaSuccess)                                                                  \
            return sail::set_err((h), SAIL_ERR_CUDA, "launch of %s failed: %s", what,            \
                                 cudaGetErrorString(e__));                                       \
    } while (0)

// ---- Philox4x32-10 (Salmon et al. SC'11), restated for the device ---------------------------------
__host__ __device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                       uint32_t k0, uint32_t k1, uint32_t (&out)[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// order-preserving key of a double as written by the residue min / max kernels (branch.cu), decoded on the host
inline double ordered_key_value(unsigned long long k)
{
    const unsigned long long b = (k >> 63) ? (k & 0x7fffffffffffffffull) : ~k;
    double v;
    memcpy(&v, &b, sizeof v);
    return v;
}

// ---- entry points implemented in the other translation units ---------------------------------------
int launch_problem_tables(sail_handle *h, const double *d_F, const double *d_sigma, double *c, double *Wj,
                          double *fj, double *E);
int launch_forward(sail_handle *h, int64_t w0, int64_t n);            // mt, chi2 of walkers [w0, w0+n)
int launch_sweeps(sail_handle *h, const double *d_T, int64_t n_sweeps, const sail_anneal_params *p,
                  int64_t sweeps_in_call, int64_t call_offset);
int check_anneal_params(sail_handle *h, const sail_anneal_params *p);
int anneal_device_schedule(sail_handle *h, const double *d_T, int64_t n, const sail_anneal_params *p, int64_t sweeps_in_call,
                           int64_t call_offset);
int launch_branch(sail_handle *h, double T, double t_imprint);
int launch_branch_fraction(sail_handle *h, double fraction, double t_imprint);                     // row f2; T found -> scalars[5]
int launch_branch_ctl(sail_handle *h, bool by_fraction, const double *ctl);                         // (T, fraction, t) on the device
int launch_smooth(sail_handle *h, double s);                          // Eq. 27-29 + renormalisation + forward
int launch_scale_model(sail_handle *h, double *dst);                  // dst[w][j] = c_j mt[w][j]
int ensure_sweep_tables(sail_handle *h);
bool sweep_fits(int n_omega);                                         // tables + records within one SM's shared memory

} // namespace sail
