// microbench.cu — sail_microbench: the per-SM issue rates and latencies the sweep-kernel design rests on
// (DESIGN.md §6.1), measured on the device the library runs on.  Diagnostics only; not part of the method.
//   FP64 FMA rate, DMMA m8n8k4 rate alone and mixed with DFMA (do they share a pipe?), warp-shuffle rate,
//   broadcast and per-lane shared-memory load rates, and the dependent-issue latencies of DFMA / SHFL / DMMA.
#include "sail_internal.cuh"

namespace sail {

constexpr int kUbIter = 4096;

#define SAIL_DMMA(c0, c1, a, b)                                                                              \
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"         \
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b))

// MODE 0: 8 independent DFMA chains   1: 4 independent DMMA chains   2: 2 DMMA + 8 DFMA interleaved
//      3: 8 independent SHFL          4: LDS.128, one address for the whole warp
//      5: LDS.64, lane-contiguous     6: dependent DFMA   7: dependent SHFL   8: dependent DMMA
template <int MODE>
__global__ void ub_kernel(double a, double b, double *sink)
{
    __shared__ __align__(16) double sm[512];
    for (int i = threadIdx.x; i < 512; i += blockDim.x) sm[i] = (double)i;
    __syncthreads();
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    int s0 = threadIdx.x, s1 = s0 * 3, s2 = s0 * 5, s3 = s0 * 7, s4 = s0 + 11, s5 = s0 + 13, s6 = s0 + 17, s7 = s0 + 19;
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(sm) + ((MODE == 5) ? (threadIdx.x & 31) * 8 : 0);
#pragma unroll 1
    for (int i = 0; i < kUbIter; ++i) {
        if (MODE == 0) {
            x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
            x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
        } else if (MODE == 1) {
            SAIL_DMMA(x0, x1, a, b); SAIL_DMMA(x2, x3, a, b); SAIL_DMMA(x4, x5, a, b); SAIL_DMMA(x6, x7, a, b);
        } else if (MODE == 2) {
            double y0 = x0, y1 = x1;
            SAIL_DMMA(y0, y1, a, b); x0 = y0; x1 = y1;
            x2 = fma(x2, a, b); x3 = fma(x3, a, b); x4 = fma(x4, a, b); x5 = fma(x5, a, b);
            double z0 = x6, z1 = x7;
            SAIL_DMMA(z0, z1, a, b); x6 = z0; x7 = z1;
            x2 = fma(x2, a, b); x3 = fma(x3, a, b); x4 = fma(x4, a, b); x5 = fma(x5, a, b);
        } else if (MODE == 3) {
            s0 = __shfl_xor_sync(0xffffffffu, s0, 1); s1 = __shfl_xor_sync(0xffffffffu, s1, 2);
            s2 = __shfl_xor_sync(0xffffffffu, s2, 4); s3 = __shfl_xor_sync(0xffffffffu, s3, 8);
            s4 = __shfl_xor_sync(0xffffffffu, s4, 16); s5 = __shfl_xor_sync(0xffffffffu, s5, 1);
            s6 = __shfl_xor_sync(0xffffffffu, s6, 2); s7 = __shfl_xor_sync(0xffffffffu, s7, 4);
        } else if (MODE == 4 || MODE == 5) {
#pragma unroll
            for (int u = 0; u < 8; ++u) {           // the address depends on i; results are folded with integer ops
                const uint32_t ad = base + (uint32_t)(((i + u) & 7) * ((MODE == 4) ? 16 : 256));
                unsigned long long p, q = 0ull;
                if (MODE == 4) asm volatile("ld.shared.v2.b64 {%0,%1}, [%2];" : "=l"(p), "=l"(q) : "r"(ad));
                else           asm volatile("ld.shared.b64 %0, [%1];" : "=l"(p) : "r"(ad));
                s0 ^= (int)(p ^ q); s1 ^= (int)((p ^ q) >> 32);
            }
        } else if (MODE == 6) {
#pragma unroll
            for (int u = 0; u < 8; ++u) x0 = fma(x0, a, b);
        } else if (MODE == 7) {
#pragma unroll
            for (int u = 0; u < 8; ++u) s0 = __shfl_xor_sync(0xffffffffu, s0, 1 << (u & 3));
        } else {
#pragma unroll
            for (int u = 0; u < 4; ++u) SAIL_DMMA(x0, x1, a, b);
        }
    }
    const double r = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7 + (double)(s0 + s1 + s2 + s3 + s4 + s5 + s6 + s7);
    if (r == 123.456) *sink = r;
}

template <int MODE>
static double ub_cycles_per_instr(cudaStream_t st, int blocks, int threads, double instr_per_iter, double clock_hz, double *sink,
                                  bool per_sm)
{
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    ub_kernel<MODE><<<blocks, threads, 0, st>>>(1.0000001, 1e-9, sink);
    float best = 1e30f;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(e0, st);
        ub_kernel<MODE><<<blocks, threads, 0, st>>>(1.0000001, 1e-9, sink);
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    const double cycles = best * 1e-3 * clock_hz;
    const double warps_per_sm = threads / 32.0;        // one CTA per SM
    const double instr = kUbIter * instr_per_iter * (per_sm ? warps_per_sm : 1.0);
    return cycles / instr;                              // cycles per warp-instruction (per SM, or per warp)
}

} // namespace sail

extern "C" {

int sail_microbench(int32_t device, void *stream, double *out, int32_t n_out)
{
    using namespace sail;
    if (!out || n_out < SAIL_MICROBENCH_N) return SAIL_ERR_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) { cudaGetLastError(); return set_err(nullptr, SAIL_ERR_CUDA, "no usable CUDA device"); }
    if (cudaSetDevice(device) != cudaSuccess) return set_err(nullptr, SAIL_ERR_CUDA, "cudaSetDevice failed");
    int sms = 0, khz = 0;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, device);
    const double hz = khz * 1e3;
    cudaStream_t st = (cudaStream_t)stream;
    double *sink = nullptr;
    if (cudaMalloc(&sink, 8) != cudaSuccess) return set_err(nullptr, SAIL_ERR_ALLOC, "cudaMalloc failed");
    const int T = 32 * 32;                              // 8 warps per sub-partition
    out[0] = 1.0 / ub_cycles_per_instr<0>(st, sms, T, 8, hz, sink, true);     // DFMA warp-instr / clk / SM
    out[1] = 1.0 / ub_cycles_per_instr<1>(st, sms, T, 4, hz, sink, true);     // DMMA m8n8k4 / clk / SM
    out[2] = ub_cycles_per_instr<2>(st, sms, T, 1, hz, sink, true);           // cycles per SM for 2 DMMA + 8 DFMA
    out[3] = 1.0 / ub_cycles_per_instr<3>(st, sms, T, 8, hz, sink, true);     // SHFL / clk / SM
    out[4] = 1.0 / ub_cycles_per_instr<4>(st, sms, T, 8, hz, sink, true);     // LDS.128 (uniform address) / clk / SM
    out[5] = 1.0 / ub_cycles_per_instr<5>(st, sms, T, 8, hz, sink, true);     // LDS.64 (lane-contiguous) / clk / SM
    out[6] = ub_cycles_per_instr<6>(st, sms, 32, 8, hz, sink, false);         // dependent DFMA latency, cycles
    out[7] = ub_cycles_per_instr<7>(st, sms, 32, 8, hz, sink, false);         // dependent SHFL latency, cycles
    out[8] = ub_cycles_per_instr<8>(st, sms, 32, 4, hz, sink, false);         // dependent DMMA latency, cycles
    out[9] = 1.0 / ub_cycles_per_instr<0>(st, sms, 4 * 32, 8, hz, sink, true); // DFMA / clk / SM at ONE warp per sub-partition
    cudaFree(sink);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return set_err(nullptr, SAIL_ERR_CUDA, "microbenchmark failed: %s", cudaGetErrorString(e));
    return SAIL_OK;
}

} // extern "C"
