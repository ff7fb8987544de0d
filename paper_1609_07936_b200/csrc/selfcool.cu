// selfcool.cu — population statistics and the self-cooling block protocol (PAPER.md:160-162,
// :216-220; readings C1-C3 in DESIGN.md §2).  The temperature of a block follows the residues the population has
// reached: T = 10 starting residues for block 0 (:216), T = chi2_ave while "boiling", a linear ramp to chi2_min,
// then a freeze-out below chi2_min that falls like 1 / steps (:162).  A block is the smoothing step (if asked for; :199),
// sweeps_per_block sweeps at that T and one imprinted-branching event (:218-220).
// The whole feedback loop stays on the device: the statistics (two kernels with a fixed summation order, bit-reproducible
// run to run), the rule (one CTA), the block's schedule slice, the acceptance-driven strength (reading B7) and the
// parameters of the branching event live in the handle's control block; the host only enqueues.  T / chi2_ave /
// chi2_min per block come back once at the end of the call.
#include <mutex>

#include "sail_internal.cuh"

namespace sail {

constexpr int kStatBlocks = 256, kStatThreads = 256;
// control block (h->ctl): 0 T of the block, 1 branching fraction, 2 imprint strength (read by branch.cu);
// 8 chi2_min, 9 chi2_ave (statistics); 10 chi2_0; 11 largest block acceptance rate so far; 12 error flag
constexpr int kCtlT = 0, kCtlFrac = 1, kCtlImp = 2, kCtlMin = 8, kCtlAve = 9, kCtlChi0 = 10, kCtlAccMax = 11, kCtlErr = 12;

// partial[b] = sum of chi2[i] over i = b * 256 + t + k * (blocks * 256), added per thread in increasing i, then over
// the threads of the block in a fixed tree; pmin[b] likewise
__global__ void __launch_bounds__(kStatThreads) chi2_stats_partial_kernel(long long W, const double *__restrict__ chi2,
                                                                          double *partial, double *pmin)
{
    __shared__ double ss[kStatThreads], sm[kStatThreads];
    double s = 0.0, m = 1.0 / 0.0;
    for (long long i = (long long)blockIdx.x * kStatThreads + threadIdx.x; i < W; i += (long long)gridDim.x * kStatThreads) {
        const double v = chi2[i];
        s += v;
        m = v < m ? v : m;
    }
    ss[threadIdx.x] = s; sm[threadIdx.x] = m;
    __syncthreads();
    for (int h = kStatThreads / 2; h > 0; h >>= 1) {
        if ((int)threadIdx.x < h) {
            ss[threadIdx.x] += ss[threadIdx.x + h];
            sm[threadIdx.x] = sm[threadIdx.x + h] < sm[threadIdx.x] ? sm[threadIdx.x + h] : sm[threadIdx.x];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) { partial[blockIdx.x] = ss[0]; pmin[blockIdx.x] = sm[0]; }
}

__global__ void chi2_stats_final_kernel(int blocks, long long W, const double *partial, const double *pmin, double *out)
{
    double s = 0.0, m = 1.0 / 0.0;
    for (int b = 0; b < blocks; ++b) { s += partial[b]; m = pmin[b] < m ? pmin[b] : m; }
    out[0] = m;
    out[1] = s / (double)W;
}

// (chi2_min, chi2_ave) of the population -> ctl[8], ctl[9]; stream-ordered, no host access
static int enqueue_chi2_stats(sail_handle *h)
{
    const long long W = h->W;
    int blocks = (int)((W + kStatThreads - 1) / kStatThreads);
    if (blocks > kStatBlocks) blocks = kStatBlocks;
    if (blocks > W / 2) blocks = (int)(W / 2 > 0 ? W / 2 : 1);          // partial sums and minima share scanA [W]
    double *partial = reinterpret_cast<double *>(h->br.scanA);
    double *pmin = W >= 2 ? partial + blocks : reinterpret_cast<double *>(h->br.scanB);
    chi2_stats_partial_kernel<<<blocks, kStatThreads, 0, h->stream>>>(W, h->st.chi2, partial, pmin);
    SAIL_LAUNCH_OK(h, "chi2_stats_partial_kernel");
    chi2_stats_final_kernel<<<1, 1, 0, h->stream>>>(blocks, W, partial, pmin, h->ctl + kCtlMin);
    SAIL_LAUNCH_OK(h, "chi2_stats_final_kernel");
    return SAIL_OK;
}

int launch_chi2_stats(sail_handle *h, double *host_min, double *host_mean)
{
    int rc = enqueue_chi2_stats(h);
    if (rc) return rc;
    double res[2];
    SAIL_CUDA_OK(h, cudaMemcpyAsync(res, h->ctl + kCtlMin, sizeof res, cudaMemcpyDeviceToHost, h->stream));
    SAIL_CUDA_OK(h, cudaStreamSynchronize(h->stream));
    if (host_min) *host_min = res[0];
    if (host_mean) *host_mean = res[1];
    return SAIL_OK;
}

// exact (integer) total of the accepted-move counters: the acceptance rate of a block is a difference of two of these
__global__ void sum_u64_kernel(long long W, const unsigned long long *__restrict__ v, unsigned long long *dst)
{
    unsigned long long s = 0ull;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < W; i += (long long)gridDim.x * blockDim.x) s += v[i];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    if ((threadIdx.x & 31) == 0) atomicAdd(dst, s);
}

// scalars[6] <- sum of the accepted-move counters (scalars[7] keeps the previous total)
static int enqueue_accepted_total(sail_handle *h)
{
    unsigned long long *dst = h->br.scalars + 6;
    SAIL_CUDA_OK(h, cudaMemsetAsync(dst, 0, 8, h->stream));
    const int blocks = (int)((h->W + 255) / 256 < 256 ? (h->W + 255) / 256 : 256);
    sum_u64_kernel<<<blocks, 256, 0, h->stream>>>(h->W, h->st.n_acc, dst);
    SAIL_LAUNCH_OK(h, "sum_u64_kernel");
    return SAIL_OK;
}

struct CoolRule { int n_boil, n_ramp; double T_start, freeze_rate, t_imprint, fraction; };

// readings C1-C3: the temperature of block b from the residues measured before it (ctl[8], ctl[9]); fills the block's
// schedule slice, the branching parameters and the per-block outputs.  Thread 0 applies the rule, the CTA fills the slice.
// A rule that gives T <= 0 (chi2_min is a running sum and can go negative next to an exact fit) HALTS the call: the flag
// ctl[12] is set and stays set, the slice gets T = 0 — the sweep kernel returns at once on such a slice — and T = 0,
// fraction = 0 make the branching event a no-op; sail_smooth's kernel reads the flag.  Every later block of the call does
// the same, so the population stays as it was when the rule failed; the host reports the block at the end of the call.
constexpr int kRuleThreads = 256;
__global__ void __launch_bounds__(kRuleThreads) selfcool_rule_kernel(long long b, int out_slot, CoolRule r, int has_override, double T_override, int k,
                                                                     double *ctl, double *d_T, double *block_out, int out_stride)
{
    __shared__ double sT;
    if (threadIdx.x == 0) {
        const double mn = ctl[kCtlMin], ave = ctl[kCtlAve];
        if (b == 0) { ctl[kCtlChi0] = ave; ctl[kCtlAccMax] = 0.0; }   // the unit of T and of the residue (:216)
        double T;
        if (has_override) T = T_override;
        else if (b == 0) T = r.T_start * ctl[kCtlChi0];
        else if (b <= r.n_boil) T = ave;
        else if (b <= (long long)r.n_boil + r.n_ramp) T = ave + (mn - ave) * ((double)(b - r.n_boil) / (double)r.n_ramp);
        else T = mn / (1.0 + r.freeze_rate * (double)(b - r.n_boil - r.n_ramp));
        const bool halted = ctl[kCtlErr] != 0.0;
        if (!halted && !(T > 0.0)) ctl[kCtlErr] = 1.0 + (double)b;   // first failure: remember the block
        if (halted || !(T > 0.0)) T = 0.0;
        ctl[kCtlT] = T; ctl[kCtlFrac] = T > 0.0 ? r.fraction : 0.0; ctl[kCtlImp] = T > 0.0 ? r.t_imprint : 0.0;
        block_out[out_slot] = T; block_out[out_stride + out_slot] = ave; block_out[2 * out_stride + out_slot] = mn;
        sT = T;
    }
    __syncthreads();
    const double T = sT;
    for (int i = threadIdx.x; i < k; i += kRuleThreads) d_T[i] = T;
}

// :184 (reading B7): less imprinting and a smaller branching fraction as the acceptance rate falls — both are
// multiplied by (acceptance rate of the block's sweeps) / (largest block acceptance rate so far); the rate is an exact
// integer count over W k N_omega
__global__ void selfcool_strength_kernel(double moves_per_block, CoolRule r, unsigned long long *scalars, double *ctl)
{
    const unsigned long long now = scalars[6], prev = scalars[7];
    scalars[7] = now;
    const double rate = (double)(now - prev) / moves_per_block;
    if (rate > ctl[kCtlAccMax]) ctl[kCtlAccMax] = rate;
    const double scale = (ctl[kCtlAccMax] > 0.0 && ctl[kCtlErr] == 0.0) ? rate / ctl[kCtlAccMax] : 0.0;   // halted: no branching
    ctl[kCtlFrac] = r.fraction * scale;
    ctl[kCtlImp] = r.t_imprint * scale;
}

__global__ void copy_u64_kernel(const unsigned long long *src, unsigned long long *dst) { *dst = *src; }

} // namespace sail

extern "C" {

int sail_chi2_stats(sail_t *h, double *chi2_min, double *chi2_mean)
{
    if (!h) return SAIL_ERR_ARG;
    if (!h->initialised) return sail::set_err(h, SAIL_ERR_STATE, "sail_chi2_stats before sail_init_walkers");
    SAIL_CUDA_OK(h, cudaSetDevice(h->device));
    return sail::launch_chi2_stats(h, chi2_min, chi2_mean);
}

int sail_anneal_selfcool(sail_t *h, const sail_selfcool_params *p, int64_t n_blocks, double *T_out, double *chi2_ave_out,
                         double *chi2_min_out)
{
    using namespace sail;
    if (!h || !p) return SAIL_ERR_ARG;
    if (!h->initialised) return set_err(h, SAIL_ERR_STATE, "sail_anneal_selfcool before sail_init_walkers");
    if (n_blocks < 0 || p->sweeps_per_block < 1 || p->n_boil < 0 || p->n_ramp < 1 || !(p->T_start > 0.0) || !(p->freeze_rate > 0.0) ||
        !(p->t_imprint >= 0.0 && p->t_imprint <= 1.0) || !(p->smooth_s >= 0.0 && p->smooth_s <= 0.5) || !(p->branch_fraction >= 0.0 && p->branch_fraction < 1.0))
        return set_err(h, SAIL_ERR_ARG, "bad self-cooling parameters");
    if ((size_t)p->sweeps_per_block > h->d_T_cap) return set_err(h, SAIL_ERR_ARG, "sweeps_per_block > %zu", h->d_T_cap);
    if (p->anneal.trace || p->anneal.flags)
        return set_err(h, SAIL_ERR_ARG, "sail_anneal_selfcool does not trace (trace and flags of the anneal parameters must be NULL)");
    { const int rcp = check_anneal_params(h, &p->anneal); if (rcp) return rcp; }
    if (p->T_override)
        for (int64_t b = 0; b < n_blocks; ++b)
            if (!(p->T_override[b] > 0.0)) return set_err(h, SAIL_ERR_ARG, "T_override[%lld] must be > 0", (long long)b);
    SAIL_CUDA_OK(h, cudaSetDevice(h->device));
    const CoolRule rule{p->n_boil, p->n_ramp, p->T_start, p->freeze_rate, p->t_imprint, p->branch_fraction};
    const double moves_per_block = (double)h->W * (double)p->sweeps_per_block * (double)h->n_omega;
    const int k = p->sweeps_per_block;
    SAIL_CUDA_OK(h, cudaMemsetAsync(h->ctl + kCtlErr, 0, sizeof(double), h->stream));
    struct HaltScope {                                   // the smoothing launches of THIS call read the halt flag
        sail_handle *h;
        ~HaltScope() { h->halt = nullptr; }
    } halt_scope{h};
    h->halt = h->ctl + kCtlErr;
    int rc;
    if (p->adapt) {                                      // scalars[7] = accepted moves so far
        if ((rc = enqueue_accepted_total(h))) return rc;
        copy_u64_kernel<<<1, 1, 0, h->stream>>>(h->br.scalars + 6, h->br.scalars + 7);
        SAIL_LAUNCH_OK(h, "copy_u64_kernel");
    }
    for (int64_t b0 = 0; b0 < n_blocks; b0 += kSelfcoolBlocksMax) {
        const int64_t nb = n_blocks - b0 < kSelfcoolBlocksMax ? n_blocks - b0 : kSelfcoolBlocksMax;
        for (int64_t b = b0; b < b0 + nb; ++b) {
            if ((rc = enqueue_chi2_stats(h))) return rc;
            selfcool_rule_kernel<<<1, kRuleThreads, 0, h->stream>>>(b, (int)(b - b0), rule, p->T_override ? 1 : 0, p->T_override ? p->T_override[b] : 0.0, k,
                                                         h->ctl, h->d_T, h->block_out, kSelfcoolBlocksMax);
            SAIL_LAUNCH_OK(h, "selfcool_rule_kernel");
            // reading C3 as amended (smoothed and renormalised transforms "undergo Metropolis updates and
            // branching.  The process is then repeated."): smoothing opens the block, the k sweeps relax it, then branching
            if (p->smooth_s > 0.0 && (rc = launch_smooth(h, p->smooth_s))) return rc;
            if ((rc = anneal_device_schedule(h, h->d_T, k, &p->anneal, k, 0))) return rc;
            if (p->adapt) {
                if ((rc = enqueue_accepted_total(h))) return rc;
                selfcool_strength_kernel<<<1, 1, 0, h->stream>>>(moves_per_block, rule, h->br.scalars, h->ctl);
                SAIL_LAUNCH_OK(h, "selfcool_strength_kernel");
            }
            if (p->branch && (rc = launch_branch_ctl(h, p->branch_fraction > 0.0, h->ctl))) return rc;
        }
        // one read-back per pass of up to 4096 blocks: the trajectory and the error flag
        double err = 0.0;
        if (T_out) SAIL_CUDA_OK(h, cudaMemcpyAsync(T_out + b0, h->block_out, (size_t)nb * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
        if (chi2_ave_out) SAIL_CUDA_OK(h, cudaMemcpyAsync(chi2_ave_out + b0, h->block_out + kSelfcoolBlocksMax, (size_t)nb * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
        if (chi2_min_out) SAIL_CUDA_OK(h, cudaMemcpyAsync(chi2_min_out + b0, h->block_out + 2 * kSelfcoolBlocksMax, (size_t)nb * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
        SAIL_CUDA_OK(h, cudaMemcpyAsync(&err, h->ctl + kCtlErr, sizeof err, cudaMemcpyDeviceToHost, h->stream));
        SAIL_CUDA_OK(h, cudaStreamSynchronize(h->stream));
        if (err != 0.0) return set_err(h, SAIL_ERR_ARG, "self-cooling reached T <= 0 at block %lld", (long long)(err - 1.0));
    }
    return SAIL_OK;
}

} // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// sail_chi2_stats_static — the population statistics for callers that may not allocate (include/sail.h says who: a
// monitoring thread without the handle, or a process whose HBM a caching allocator already owns).  The two kernels above
// are reused unchanged; only the place their per-CTA partial results go differs: a fixed array in the library image
// instead of a slice of a handle's workspace.
// ---------------------------------------------------------------------------------------------------------------------
namespace sail {

// kStatBlocks partial sums followed by kStatBlocks partial minima = SAIL_STATS_STATIC_SCRATCH_BYTES.  One copy per GPU
// that loads the library, alive until the process exits, shared by every call on that GPU.
static __device__ __align__(256) double g_stats_static_scratch[2 * kStatBlocks];
static_assert(sizeof(double) * 2 * kStatBlocks == SAIL_STATS_STATIC_SCRATCH_BYTES, "sail.h states the size of the static scratch array");
static_assert(SAIL_STATS_STATIC_MAX_W == (int64_t)kStatBlocks * kStatThreads * 256, "sail.h: at most 256 residues per thread");

// In host code the name g_stats_static_scratch is only a stand-in for the symbol, NOT a device address: a kernel handed
// `g_stats_static_scratch` from the host faults (or scribbles over host memory where the GPU can reach it).  The device
// address differs from GPU to GPU and is looked up once per device with cudaGetSymbolAddress, with that device current.
constexpr int kStaticMaxDevices = 64;
static std::mutex g_stats_static_mutex;
static double *g_stats_static_addr[kStaticMaxDevices];      // nullptr = this device has not been set up yet

// `device` must be current.  Allocates nothing: the array already exists in the module loaded on the device.
static int stats_static_scratch(int device, double **scratch)
{
    std::lock_guard<std::mutex> lock(g_stats_static_mutex);
    if (!g_stats_static_addr[device]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_stats_static_scratch);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return set_err(nullptr, SAIL_ERR_CUDA, "sail_chi2_stats_static: cudaGetSymbolAddress on device %d failed: %s", device,
                           cudaGetErrorString(e));
        }
        g_stats_static_addr[device] = static_cast<double *>(p);
    }
    *scratch = g_stats_static_addr[device];
    return SAIL_OK;
}

} // namespace sail

extern "C" int sail_chi2_stats_static(int32_t device, void *stream, const double *chi2, int64_t W, double *out)
{
    using namespace sail;
    if (!chi2 || !out) return set_err(nullptr, SAIL_ERR_ARG, "sail_chi2_stats_static: chi2 and out must be device pointers, not NULL");
    if (W < 1 || W > SAIL_STATS_STATIC_MAX_W)
        return set_err(nullptr, SAIL_ERR_ARG, "sail_chi2_stats_static: W=%lld outside [1, %lld] (SAIL_STATS_STATIC_MAX_W: the fixed %d-byte "
                       "scratch array is laid out for at most that many residues; use sail_chi2_stats or split the array)",
                       (long long)W, (long long)SAIL_STATS_STATIC_MAX_W, SAIL_STATS_STATIC_SCRATCH_BYTES);
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1 || device < 0 || device >= ndev) {
        cudaGetLastError();
        return set_err(nullptr, SAIL_ERR_CUDA, "sail_chi2_stats_static: no usable CUDA device (count=%d, requested=%d); there is no CPU fallback", ndev, device);
    }
    if (device >= kStaticMaxDevices) return set_err(nullptr, SAIL_ERR_ARG, "sail_chi2_stats_static: device ordinal %d >= %d", device, kStaticMaxDevices);
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return set_err(nullptr, SAIL_ERR_CUDA, "sail_chi2_stats_static: cudaSetDevice(%d) failed", device); }
    double *scratch = nullptr;
    if (const int rc = stats_static_scratch(device, &scratch)) return rc;
    // the grid of enqueue_chi2_stats, so that the summation order (and with it every bit of the result) is the same
    int blocks = (int)((W + kStatThreads - 1) / kStatThreads);
    if (blocks > kStatBlocks) blocks = kStatBlocks;
    if (blocks > W / 2) blocks = (int)(W / 2 > 0 ? W / 2 : 1);
    double *partial = scratch, *pmin = scratch + kStatBlocks;
    // Nothing to clear: the first kernel writes slots [0, blocks) of both halves, the second reads exactly those, so what an
    // earlier call (possibly with more CTAs) left behind is never read.
    cudaStream_t st = (cudaStream_t)stream;
    chi2_stats_partial_kernel<<<blocks, kStatThreads, 0, st>>>((long long)W, chi2, partial, pmin);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) {
        chi2_stats_final_kernel<<<1, 1, 0, st>>>(blocks, (long long)W, partial, pmin, out);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) return set_err(nullptr, SAIL_ERR_CUDA, "sail_chi2_stats_static: kernel launch failed: %s", cudaGetErrorString(e));
    return SAIL_OK;
}
