// dp_measure_peaks: microbenchmarks of the arithmetic pipes the hot path is bound by ("fp64/fp32/SFU peaks are
// not in MEASURED_PEAKS.json: measure them in the same bench run and quote fractions against measured").  Each kernel keeps
// every SM busy with independent dependency chains of one instruction kind; the rate is instructions x work / CUDA-event time.
// Not part of dp_compute; bench.py calls it once per run and prints the numbers beside the roofline fractions.
#include <cstdio>
#include "dp_internal.h"

namespace {

constexpr int PK_THREADS = 256;
constexpr int PK_CHAINS = 8;

// fp64 FMA pipe (DFMA): PK_CHAINS independent chains per thread
__global__ void __launch_bounds__(PK_THREADS) k_peak_dfma(int iters, double *out) {
    double a[PK_CHAINS];
    const double x = 1.0 + 1e-9 * threadIdx.x, y = 1e-9;
#pragma unroll
    for (int c = 0; c < PK_CHAINS; ++c) a[c] = (double)c;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int c = 0; c < PK_CHAINS; ++c) a[c] = fma(a[c], x, y);
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < PK_CHAINS; ++c) s += a[c];
    if (s == 12345.678) out[0] = s;      // never true: keeps the chains alive
}

// fp64 tensor pipe (DMMA m8n8k4, the shape of the FP64 kernels): PK_CHAINS independent accumulator pairs per warp
__global__ void __launch_bounds__(PK_THREADS) k_peak_dmma(int iters, double *out) {
    double c0[PK_CHAINS], c1[PK_CHAINS];
    const double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-9 * (threadIdx.x & 3);
#pragma unroll
    for (int c = 0; c < PK_CHAINS; ++c) { c0[c] = (double)c; c1[c] = 0.5 * c; }
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int c = 0; c < PK_CHAINS; ++c)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c0[c]), "+d"(c1[c]) : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < PK_CHAINS; ++c) s += c0[c] + c1[c];
    if (s == 12345.678) out[0] = s;
}

// fp32 FMA pipe (FFMA)
__global__ void __launch_bounds__(PK_THREADS) k_peak_ffma(int iters, float *out) {
    float a[2 * PK_CHAINS];
    const float x = 1.0f + 1e-6f * threadIdx.x, y = 1e-6f;
#pragma unroll
    for (int c = 0; c < 2 * PK_CHAINS; ++c) a[c] = (float)c;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int c = 0; c < 2 * PK_CHAINS; ++c) a[c] = fmaf(a[c], x, y);
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < 2 * PK_CHAINS; ++c) s += a[c];
    if (s == 12345.678f) out[0] = s;
}

// special-function unit: tanh.approx.f32 (MUFU.TANH), the activation of the mixed-precision nets
__global__ void __launch_bounds__(PK_THREADS) k_peak_tanh(int iters, float *out) {
    float a[PK_CHAINS];
#pragma unroll
    for (int c = 0; c < PK_CHAINS; ++c) a[c] = 0.1f * c + 1e-3f * threadIdx.x;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int c = 0; c < PK_CHAINS; ++c) asm volatile("tanh.approx.f32 %0, %0;" : "+f"(a[c]));
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < PK_CHAINS; ++c) s += a[c];
    if (s == 12345.678f) out[0] = s;
}

// legacy tensor path (mma.sync m16n8k16 fp16 -> fp32), the pipe of the MIX-32 backward and fitting kernels
__global__ void __launch_bounds__(PK_THREADS) k_peak_hmma(int iters, float *out) {
    float c[PK_CHAINS][4];
    const uint32_t a0 = 0x3c003c00u, b0 = 0x38003800u;      // fp16 pairs (1, 1), (0.5, 0.5)
#pragma unroll
    for (int k = 0; k < PK_CHAINS; ++k) c[k][0] = c[k][1] = c[k][2] = c[k][3] = (float)k;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < PK_CHAINS; ++k)
            asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%4,%4,%4}, {%5,%5}, {%0,%1,%2,%3};"
                         : "+f"(c[k][0]), "+f"(c[k][1]), "+f"(c[k][2]), "+f"(c[k][3]) : "r"(a0), "r"(b0));
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < PK_CHAINS; ++k) s += c[k][0] + c[k][1] + c[k][2] + c[k][3];
    if (s == 12345.678f) out[0] = s;
}

template <typename F>
double time_ms(F launch, cudaStream_t st) {
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return -1.0;
    launch();                                   // warm-up
    float best = 1e30f;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(e0, st);
        launch();
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { best = -1.f; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    return (double)best;
}

}  // namespace

extern "C" int dp_measure_peaks(double *out_host, int n_out, void *cuda_stream) {
    if (!out_host || n_out < DP_NPEAKS) return DP_EINVAL;
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return DP_ECUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double *scratch = nullptr;
    if (cudaMalloc(&scratch, 64) != cudaSuccess) return DP_ECUDA;
    const int grid = prop.multiProcessorCount * 8;       // 8 CTAs of 256 threads per SM: full occupancy
    const double threads = (double)grid * PK_THREADS, warps = threads / 32.0;
    const int it64 = 1 << 14, it32 = 1 << 16, itmu = 1 << 14, itmma = 1 << 14;
    double ms;
    ms = time_ms([&] { k_peak_dfma<<<grid, PK_THREADS, 0, st>>>(it64, scratch); }, st);
    out_host[0] = ms > 0 ? 2.0 * threads * PK_CHAINS * it64 / (ms * 1e-3) / 1e12 : 0.0;                    // DFMA TFLOP/s
    ms = time_ms([&] { k_peak_dmma<<<grid, PK_THREADS, 0, st>>>(itmma, scratch); }, st);
    out_host[1] = ms > 0 ? 2.0 * 8 * 8 * 4 * warps * PK_CHAINS * itmma / (ms * 1e-3) / 1e12 : 0.0;         // DMMA TFLOP/s
    ms = time_ms([&] { k_peak_ffma<<<grid, PK_THREADS, 0, st>>>(it32, (float *)scratch); }, st);
    out_host[2] = ms > 0 ? 2.0 * threads * 2 * PK_CHAINS * it32 / (ms * 1e-3) / 1e12 : 0.0;               // FFMA TFLOP/s
    ms = time_ms([&] { k_peak_tanh<<<grid, PK_THREADS, 0, st>>>(itmu, (float *)scratch); }, st);
    out_host[3] = ms > 0 ? threads * PK_CHAINS * itmu / (ms * 1e-3) / 1e12 : 0.0;                         // tanh.approx.f32, T/s
    ms = time_ms([&] { k_peak_hmma<<<grid, PK_THREADS, 0, st>>>(itmma, (float *)scratch); }, st);
    out_host[4] = ms > 0 ? 2.0 * 16 * 8 * 16 * warps * PK_CHAINS * itmma / (ms * 1e-3) / 1e12 : 0.0;      // mma.sync fp16 TFLOP/s
    out_host[5] = (double)prop.multiProcessorCount;
    cudaFree(scratch);
    return cudaGetLastError() == cudaSuccess ? DP_OK : DP_ECUDA;
}
