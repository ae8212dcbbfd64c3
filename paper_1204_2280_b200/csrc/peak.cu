// Measurement support, not part of the method: the FP32 peak of the device this context runs on, MEASURED with the
// two instruction forms the walk's interaction loops are made of (FFMA2 = fma.rn.f32x2, and scalar FFMA), so that
// bench.py can report the walk's flop/s against a measured denominator next to the derived one
// (SMs x 128 lanes x 2 flop x clock).  Every thread runs kChains independent dependent chains for `iters` rounds;
// the result is written only when it is NaN-free garbage nobody reads, which keeps the loop alive.
#include "internal.cuh"

namespace bonsai {

constexpr int kPeakChains = 8;
constexpr int kPeakThreads = 256;

__global__ void __launch_bounds__(kPeakThreads) k_peak_ffma2(int iters, float seed, float* __restrict__ sink) {
    unsigned long long acc[kPeakChains];
    unsigned long long a, b;
    const float x = seed + (float)threadIdx.x * 1e-9f;
    asm("mov.b64 %0, {%1, %2};" : "=l"(a) : "f"(1.0f - 1e-7f), "f"(1.0f + 1e-7f));
    asm("mov.b64 %0, {%1, %2};" : "=l"(b) : "f"(x), "f"(-x));
#pragma unroll
    for (int k = 0; k < kPeakChains; ++k) asm("mov.b64 %0, {%1, %2};" : "=l"(acc[k]) : "f"(x + k), "f"(x - k));
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < kPeakChains; ++k)
            asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(acc[k]) : "l"(acc[k]), "l"(a), "l"(b));
    }
    float s = 0.0f;
#pragma unroll
    for (int k = 0; k < kPeakChains; ++k) {
        float lo, hi;
        asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(acc[k]));
        s += lo + hi;
    }
    if (s == 123.456f) sink[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(kPeakThreads) k_peak_ffma(int iters, float seed, float* __restrict__ sink) {
    float acc[2 * kPeakChains];
    const float x = seed + (float)threadIdx.x * 1e-9f;
    const float a = 1.0f - 1e-7f, b = x;
#pragma unroll
    for (int k = 0; k < 2 * kPeakChains; ++k) acc[k] = x + k;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 2 * kPeakChains; ++k) asm volatile("fma.rn.f32 %0, %1, %2, %3;" : "=f"(acc[k]) : "f"(acc[k]), "f"(a), "f"(b));
    }
    float s = 0.0f;
#pragma unroll
    for (int k = 0; k < 2 * kPeakChains; ++k) s += acc[k];
    if (s == 123.456f) sink[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace bonsai

using namespace bonsai;

extern "C" int bonsai_measure_fp32_peak(void* cuda_stream, int packed, int iters, double* tflops_out) {
    if (!tflops_out || iters < 1) return BONSAI_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return BONSAI_ECUDA;
    const int blocks = sms * 8;  // 8 x 256 threads = 64 warps per SM: every scheduler has 16 warps to pick from
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return BONSAI_ECUDA;
    float best = 0.0f;
    for (int rep = 0; rep < 4; ++rep) {  // first repetition warms up; best of the rest
        cudaEventRecord(e0, st);
        if (packed) k_peak_ffma2<<<blocks, kPeakThreads, 0, st>>>(iters, 0.5f, nullptr);
        else k_peak_ffma<<<blocks, kPeakThreads, 0, st>>>(iters, 0.5f, nullptr);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) return BONSAI_ECUDA;
        float ms = 0.0f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && (best == 0.0f || ms < best)) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (cudaGetLastError() != cudaSuccess || best <= 0.0f) return BONSAI_ECUDA;
    // per thread and iteration: kPeakChains packed FMAs = 2 kPeakChains scalar FMAs = 4 kPeakChains flop either way
    const double flop = (double)blocks * kPeakThreads * (double)iters * (4.0 * kPeakChains);
    *tflops_out = flop / (best * 1e-3) / 1e12;
    return BONSAI_OK;
}
