// selfcool.cu — population statistics and the self-cooling block protocol (PAPER.md:160-162,
// :216-220; readings C1-C3 in DESIGN.md §2).  The temperature of a block follows the residues the population has
// reached: T = 10 starting residues for block 0 (:216), T = chi2_ave while "boiling", a linear ramp to chi2_min,
// then a freeze-out below chi2_min that falls like 1 / steps (:162).  A block is sweeps_per_block sweeps at that T,
// the smoothing step (if asked for) and one imprinted-branching event (:218-220).
// The statistics are two kernels with a fixed summation order (bit-reproducible run to run); the rule itself is
// scalar host arithmetic on their two results, as in the paper's own driver.
#include "sail_internal.cuh"
#include <vector>

namespace sail {

constexpr int kStatBlocks = 256, kStatThreads = 256;

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

int launch_chi2_stats(sail_handle *h, double *host_min, double *host_mean)
{
    const long long W = h->W;
    int blocks = (int)((W + kStatThreads - 1) / kStatThreads);
    if (blocks > kStatBlocks) blocks = kStatBlocks;
    if (blocks > W / 2) blocks = (int)(W / 2 > 0 ? W / 2 : 1);          // partial sums and minima share scanA [W]
    double *partial = reinterpret_cast<double *>(h->br.scanA);
    double *pmin = W >= 2 ? partial + blocks : reinterpret_cast<double *>(h->br.scanB);
    double *out = reinterpret_cast<double *>(h->br.scalars + 4);
    chi2_stats_partial_kernel<<<blocks, kStatThreads, 0, h->stream>>>(W, h->st.chi2, partial, pmin);
    SAIL_LAUNCH_OK(h, "chi2_stats_partial_kernel");
    chi2_stats_final_kernel<<<1, 1, 0, h->stream>>>(blocks, W, partial, pmin, out);
    SAIL_LAUNCH_OK(h, "chi2_stats_final_kernel");
    double res[2];
    SAIL_CUDA_OK(h, cudaMemcpyAsync(res, out, sizeof res, cudaMemcpyDeviceToHost, h->stream));
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

static int accepted_total(sail_handle *h, unsigned long long *total)
{
    unsigned long long *dst = h->br.scalars + 7;
    SAIL_CUDA_OK(h, cudaMemsetAsync(dst, 0, 8, h->stream));
    const int blocks = (int)((h->W + 255) / 256 < 256 ? (h->W + 255) / 256 : 256);
    sum_u64_kernel<<<blocks, 256, 0, h->stream>>>(h->W, h->st.n_acc, dst);
    SAIL_LAUNCH_OK(h, "sum_u64_kernel");
    SAIL_CUDA_OK(h, cudaMemcpyAsync(total, dst, 8, cudaMemcpyDeviceToHost, h->stream));
    SAIL_CUDA_OK(h, cudaStreamSynchronize(h->stream));
    return SAIL_OK;
}

// readings C1-C3: the temperature of block b from the residues measured before it
static double selfcool_T(int64_t b, double chi2_0, double ave, double mn, const sail_selfcool_params *p)
{
    if (b == 0) return p->T_start * chi2_0;
    if (b <= p->n_boil) return ave;
    if (b <= (int64_t)p->n_boil + p->n_ramp) return ave + (mn - ave) * ((double)(b - p->n_boil) / (double)p->n_ramp);
    return mn / (1.0 + p->freeze_rate * (double)(b - p->n_boil - p->n_ramp));
}

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
    SAIL_CUDA_OK(h, cudaSetDevice(h->device));
    double chi2_0 = 0.0, acc_max = 0.0;
    unsigned long long acc_prev = 0ull;
    if (p->adapt) { int rc0 = accepted_total(h, &acc_prev); if (rc0) return rc0; }
    std::vector<double> T((size_t)p->sweeps_per_block);
    for (int64_t b = 0; b < n_blocks; ++b) {
        double mn = 0.0, ave = 0.0;
        int rc = launch_chi2_stats(h, &mn, &ave);
        if (rc) return rc;
        if (b == 0) chi2_0 = ave;                        // the unit of T and of the residue (:216)
        const double Tb = p->T_override ? p->T_override[b] : selfcool_T(b, chi2_0, ave, mn, p);
        if (!(Tb > 0.0)) return set_err(h, SAIL_ERR_ARG, "self-cooling reached T = %g at block %lld", Tb, (long long)b);
        if (T_out) T_out[b] = Tb;
        if (chi2_ave_out) chi2_ave_out[b] = ave;
        if (chi2_min_out) chi2_min_out[b] = mn;
        for (auto &x : T) x = Tb;
        if ((rc = sail_anneal(h, T.data(), p->sweeps_per_block, &p->anneal))) return rc;
        if (p->smooth_s > 0.0 && (rc = sail_smooth(h, p->smooth_s))) return rc;
        // :184 (reading B7): less imprinting and a smaller branching fraction as the acceptance rate falls
        double scale = 1.0;
        if (p->adapt) {
            unsigned long long acc_now = 0ull;
            if ((rc = accepted_total(h, &acc_now))) return rc;
            const double rate = (double)(acc_now - acc_prev) / ((double)h->W * (double)p->sweeps_per_block * (double)h->n_omega);
            acc_prev = acc_now;
            if (rate > acc_max) acc_max = rate;
            scale = acc_max > 0.0 ? rate / acc_max : 0.0;
        }
        if (p->branch) {
            if (p->branch_fraction > 0.0) rc = sail_branch_fraction(h, p->branch_fraction * scale, p->t_imprint * scale, nullptr, nullptr, nullptr, nullptr);
            else rc = sail_branch(h, Tb, p->t_imprint * scale, nullptr, nullptr, nullptr);
            if (rc) return rc;
        }
    }
    return SAIL_OK;
}

} // extern "C"
