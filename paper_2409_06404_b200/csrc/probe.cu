#include <algorithm>
// probe.cu -- sustained FP64 pipe rate: register-only DFMA chains on every SM.
// 8 independent chains per thread, 256 threads per block, 8 blocks per SM: enough warps and ILP
// to cover the DFMA latency, no memory traffic.  The measured instructions/s is the denominator
// bench.py reports next to the nominal one (148 SM x 64 lanes x SM clock).
#include "crf_internal.h"
#include "launch.h"

namespace {

__global__ void __launch_bounds__(256) fp64_probe_kernel(int iters, double seed, double *sink)
{
    double a0 = seed + threadIdx.x, a1 = a0 + 1.0, a2 = a0 + 2.0, a3 = a0 + 3.0, a4 = a0 + 4.0, a5 = a0 + 5.0,
           a6 = a0 + 6.0, a7 = a0 + 7.0;
    const double m = 0.999999, c = 1.0e-6;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            a0 = fma(a0, m, c), a1 = fma(a1, m, c), a2 = fma(a2, m, c), a3 = fma(a3, m, c);
            a4 = fma(a4, m, c), a5 = fma(a5, m, c), a6 = fma(a6, m, c), a7 = fma(a7, m, c);
        }
    }
    const double s = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (s == 123.456) *sink = s;  // never true: keeps the chains alive
}

}  // namespace

cudaError_t launch_fp64_probe(int iters, double *inst_per_s)
{
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    double *sink = nullptr;
    cudaError_t e = cudaMalloc(&sink, sizeof(double));
    if (e != cudaSuccess) return e;
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0);
    cudaEventCreate(&t1);
    const int blocks = sms * 8;
    fp64_probe_kernel<<<blocks, 256>>>(iters / 8 + 1, 1.0, sink);  // warm-up
    crf_count_launch();
    cudaEventRecord(t0);
    fp64_probe_kernel<<<blocks, 256>>>(iters, 1.0, sink);
    crf_count_launch();
    cudaEventRecord(t1);
    e = cudaEventSynchronize(t1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, t0, t1);
    cudaEventDestroy(t0);
    cudaEventDestroy(t1);
    cudaFree(sink);
    if (e != cudaSuccess) return e;
    const double warp_inst = (double)blocks * 8.0 * (double)iters * 128.0;  // 8 warps x iters x 16 x 8 DFMA
    *inst_per_s = warp_inst * 32.0 / (ms * 1.0e-3);                        // thread-level FP64 instructions/s
    return cudaGetLastError();
}

// ---- double -> float, round to nearest (the single-precision staging of crf_step_host_f32) ------------------------
namespace {
__global__ void __launch_bounds__(256) f64_to_f32_kernel(const double *__restrict__ in, float *__restrict__ out, int64_t count)
{
    for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < count; i += (int64_t)gridDim.x * 256) out[i] = __double2float_rn(in[i]);
}
}  // namespace

cudaError_t launch_f64_to_f32(const double *in, float *out, int64_t count, cudaStream_t st)
{
    if (count <= 0) return cudaSuccess;
    const int64_t blocks = std::min<int64_t>((count + 255) / 256, 148 * 8);
    f64_to_f32_kernel<<<(unsigned)blocks, 256, 0, st>>>(in, out, count);
    crf_count_launch();
    return cudaGetLastError();
}
