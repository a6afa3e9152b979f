// Bench-only: measures the fp32 FMA rate of this GPU, the denominator of bench.py's `roofline.peak_measured`
// (SURVEY.md 8(d) asks for fractions of MEASURED peaks; MEASURED_PEAKS.json holds no fp32 figure).  Not part of
// libtpctrk.so: built into libtpcbench.so by paper_1709_00618_b200/build.py and loaded by bench.py only.
#include <cuda_runtime.h>
#include <stdint.h>

namespace {
constexpr int kThreads = 256;
constexpr int kChains = 8;  // independent FMA chains per thread: enough to cover the 4-cycle FMA latency at 8 warps/scheduler

__global__ void __launch_bounds__(kThreads) fma_chain_kernel(float* out, int iters, float a, float b) {
    float x[kChains];
#pragma unroll
    for (int k = 0; k < kChains; k++) x[k] = (float)(threadIdx.x + k) * 1e-3f;
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int u = 0; u < 8; u++)
#pragma unroll
            for (int k = 0; k < kChains; k++) x[k] = fmaf(x[k], a, b);
    }
    float s = 0.0f;
#pragma unroll
    for (int k = 0; k < kChains; k++) s += x[k];
    if (s == 123.456f) out[0] = s;  // never true in practice; keeps the chains alive
}
}  // namespace

// Runs the kernel `reps` times on `cuda_stream` (one warm-up first) and returns the best rate in TFLOP/s (2 flop per
// FMA) in *tflops; `out` is a device float the caller owns.  Returns 0 or the cudaError_t.
extern "C" int tpc_bench_fp32_peak(float* out, int iters, int reps, void* cuda_stream, double* tflops) {
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    int dev = 0, n_sm = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    cudaEvent_t a = nullptr, b = nullptr;
    if (e == cudaSuccess) e = cudaEventCreate(&a);
    if (e == cudaSuccess) e = cudaEventCreate(&b);
    const int grid = n_sm * 8;  // 8 CTAs of 256 threads = 64 warps per SM
    double best = 0.0;
    for (int r = 0; r <= reps && e == cudaSuccess; r++) {
        cudaEventRecord(a, s);
        fma_chain_kernel<<<grid, kThreads, 0, s>>>(out, iters, 0.999f, 1e-4f);
        cudaEventRecord(b, s);
        e = cudaEventSynchronize(b);
        float ms = 0.0f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
        const double flop = 2.0 * 8.0 * kChains * (double)iters * kThreads * (double)grid;
        if (r > 0 && ms > 0.0f && flop / (ms * 1e-3) / 1e12 > best) best = flop / (ms * 1e-3) / 1e12;
    }
    if (a) cudaEventDestroy(a);
    if (b) cudaEventDestroy(b);
    *tflops = best;
    return (int)e;
}
