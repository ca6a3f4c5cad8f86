// kf_peak.cu -- register-only FP32 FMA microbenchmark (measurement utility, not on the hot path).
//
// SURVEY.md 8(d) asks for the sustained FP32 FMA peak measured on the box as the denominator of the
// ALU roofline: every thread runs 8 independent FMA chains, nothing touches memory until the end.
#include "kf_internal.h"

namespace kf {

namespace {

constexpr int kPeakBlock = 256;
constexpr int kChains = 8;
constexpr int kInner = 512;

__global__ void __launch_bounds__(kPeakBlock)
fma_peak_kernel(int outer, float a, float b, float* sink) {
    float x[kChains];
#pragma unroll
    for (int c = 0; c < kChains; ++c) x[c] = (float)(threadIdx.x + c) * 1e-3f;
    for (int o = 0; o < outer; ++o) {
#pragma unroll 16
        for (int i = 0; i < kInner; ++i) {
#pragma unroll
            for (int c = 0; c < kChains; ++c) x[c] = fmaf(x[c], a, b);
        }
    }
    float s = 0.0f;
#pragma unroll
    for (int c = 0; c < kChains; ++c) s += x[c];
    if (s == 123.456f) sink[0] = s;  // never true; keeps the chains alive
}

}  // namespace

// Returns TFLOP/s (FMA = 2 flop) of the best of `repeats` timed launches, or a negative cudaError.
double measure_fp32_peak(cudaStream_t stream, int repeats, float* sink) {
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int blocks = sms * 8;  // 2048 threads per SM
    const int outer = 64;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    double best = 0.0;
    for (int r = 0; r < repeats + 1; ++r) {
        cudaEventRecord(e0, stream);
        fma_peak_kernel<<<blocks, kPeakBlock, 0, stream>>>(outer, 0.999f, 1e-3f, sink);
        cudaEventRecord(e1, stream);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { best = -(double)e; break; }
        float ms = 0.0f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flop = 2.0 * (double)blocks * kPeakBlock * kChains * (double)kInner * outer;
        if (r > 0 && ms > 0.0f) best = best > flop / (ms * 1e-3) / 1e12 ? best : flop / (ms * 1e-3) / 1e12;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return best;
}

}  // namespace kf
