// bench_fp64_peak.cu -- bench.py's own measurement helper, not part of liblp_b200.so: the fp64 FMA rate of the
// device, the denominator of the arithmetic roofline bench.py reports beside the HBM one (SURVEY.md 8(d):
// "B200 fp64 vector peak is not in MEASURED_PEAKS.json -- measure it").  bench.py builds it into
// bench_fp64_peak.so (nvcc, sm_100a) and samples the SM clock around the call.  Returns 0 on success.
#include <cuda_runtime.h>

namespace {

constexpr int kChains = 8;          // independent dependent-FMA chains per thread (DFMA latency is hidden by 16 warps x 8)
constexpr int kThreads = 512;

__global__ void __launch_bounds__(kThreads) bench_dfma_chain_kernel(double *out, int iters, double a, double b)
{
    double x[kChains];
#pragma unroll
    for (int i = 0; i < kChains; ++i) x[i] = threadIdx.x * 1e-3 + i;
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < kChains; ++i) x[i] = fma(x[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < kChains; ++i) s += x[i];
    out[(size_t)blockIdx.x * kThreads + threadIdx.x] = s;      // keeps the chains alive
}

}  // namespace

extern "C" __attribute__((visibility("default"))) int bench_fp64_peak(int device, double *tflops_out)
{
    if (!tflops_out) return -1;
    *tflops_out = 0.0;
    if (cudaSetDevice(device) != cudaSuccess) return -3;
    int sm = 0;
    if (cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, device) != cudaSuccess || sm < 1) return -3;
    const int blocks = sm * 4, iters = 100000;
    double *out = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int st = -3;
    float best = 0.f;
    if (cudaMalloc(&out, sizeof(double) * (size_t)blocks * kThreads) != cudaSuccess) return -3;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) goto done;
    bench_dfma_chain_kernel<<<blocks, kThreads>>>(out, 2000, 0.999999, 1e-9);          // warm-up
    for (int rep = 0; rep < 3; ++rep) {                                             // best of three
        float ms = 0.f;
        if (cudaEventRecord(e0) != cudaSuccess) goto done;
        bench_dfma_chain_kernel<<<blocks, kThreads>>>(out, iters, 0.999999, 1e-9);
        if (cudaEventRecord(e1) != cudaSuccess || cudaEventSynchronize(e1) != cudaSuccess) goto done;
        if (cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess || !(ms > 0.f)) goto done;
        const float rate = (float)(2.0 * kChains * (double)iters * blocks * kThreads / (ms * 1e-3) / 1e12);
        best = rate > best ? rate : best;
    }
    *tflops_out = best;
    st = 0;
done:
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(out);
    return st;
}
