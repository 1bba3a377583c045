// fp64_peak.cu -- measures the FP64 roofline denominators on the device the benchmark runs on.
//
// MEASURED_PEAKS.json (driver-written) holds HBM GB/s and bf16 TFLOP/s but no FP64 figure, and
// BASELINE.json's north_star asks for "the FP64 peak measured on the device".  This file is
// measurement infrastructure, NOT part of the hot path: register-resident operands, no memory
// traffic, every SM busy.  Two kernels: FP64 tensor-pipe (DMMA: mma.sync.m8n8k4.f64, the only FP64
// MMA SASS on sm_100a) and plain FP64 FMA (DFMA).  The larger sustained figure is the FP64 peak.
//
// C ABI (host):  double gs_peak_fp64(int kind, double seconds, double* tflops_burst)
//   kind 0 = DMMA, 1 = DFMA.  Returns sustained TFLOP/s over ~`seconds`; *tflops_burst = best single
//   launch.  Negative return = CUDA error.
#include <cuda_runtime.h>
#include <cstdio>

namespace {

constexpr int kIters = 4096;
constexpr int kAcc = 16;  // independent accumulator fragments per thread

__global__ void __launch_bounds__(256) dmma_peak_kernel(double* out, double a0, double b0)
{
    double c[kAcc][2];
#pragma unroll
    for (int i = 0; i < kAcc; ++i) { c[i][0] = 0.0; c[i][1] = 0.0; }
    double a = a0 + threadIdx.x * 1e-9, b = b0;
#pragma unroll 1
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
        for (int i = 0; i < kAcc; ++i) {
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
        }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < kAcc; ++i) s += c[i][0] + c[i][1];
    if (s == 12345.678) out[0] = s;  // never true; keeps the loop alive
}

__global__ void __launch_bounds__(256) dfma_peak_kernel(double* out, double a0, double b0)
{
    double c[kAcc * 2];
#pragma unroll
    for (int i = 0; i < kAcc * 2; ++i) c[i] = i;
    double a = a0 + threadIdx.x * 1e-9, b = b0;
#pragma unroll 1
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
        for (int i = 0; i < kAcc * 2; ++i) c[i] = fma(c[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < kAcc * 2; ++i) s += c[i];
    if (s == 12345.678) out[0] = s;
}

}  // namespace

extern "C" double gs_peak_fp64(int kind, double seconds, double* tflops_burst)
{
    cudaDeviceProp prop;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return -1.0;
    const int threads = 256;
    const int blocks = prop.multiProcessorCount * 8;  // 2048 threads/SM resident = 8 CTAs of 256
    double* out = nullptr;
    if (cudaMalloc(&out, 8) != cudaSuccess) return -1.0;
    // flops per launch
    const double warps = double(blocks) * threads / 32.0;
    const double flop = kind == 0 ? warps * double(kIters) * kAcc * (8.0 * 8.0 * 4.0 * 2.0)
                                  : double(blocks) * threads * double(kIters) * (kAcc * 2) * 2.0;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    auto launch = [&]() {
        if (kind == 0) dmma_peak_kernel<<<blocks, threads>>>(out, 1.0000001, 0.9999999);
        else dfma_peak_kernel<<<blocks, threads>>>(out, 1.0000001, 0.9999999);
    };
    for (int i = 0; i < 3; ++i) launch();
    if (cudaDeviceSynchronize() != cudaSuccess) { cudaFree(out); return -1.0; }
    // burst: best of 5 single launches
    double best = 0.0;
    float one_ms = 1.0f;
    for (int i = 0; i < 5; ++i) {
        cudaEventRecord(e0);
        launch();
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        one_ms = ms;
        const double tf = flop / (ms * 1e-3) / 1e12;
        if (tf > best) best = tf;
    }
    if (tflops_burst) *tflops_burst = best;
    // sustained: back-to-back launches for ~seconds
    int n = int(seconds * 1e3 / (one_ms > 0.01f ? one_ms : 0.01f));
    if (n < 1) n = 1;
    cudaEventRecord(e0);
    for (int i = 0; i < n; ++i) launch();
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    const cudaError_t err = cudaDeviceSynchronize();
    cudaFree(out);
    if (err != cudaSuccess) return -1.0;
    return flop * n / (ms * 1e-3) / 1e12;
}

#ifdef GS_PEAK_MAIN
int main()
{
    for (int kind = 0; kind < 2; ++kind) {
        double burst = 0.0;
        const double sus = gs_peak_fp64(kind, 3.0, &burst);
        std::printf("%s: burst %.2f TFLOP/s, sustained(3s) %.2f TFLOP/s\n", kind == 0 ? "DMMA" : "DFMA", burst, sus);
    }
    return 0;
}
#endif
