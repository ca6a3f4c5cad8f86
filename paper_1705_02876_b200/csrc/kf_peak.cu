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

// The same for the PACKED instruction the two-tracks-per-thread kernels are made of (FFMA2: one fp32x2 FMA per
// lane).  MODE 0: x = x * A + B with A, B shared by every chain (the operand-reuse cache serves them: the rate of the
// FMA pipe itself).  MODE 1: x = x * y + z with three DISTINCT register pairs per instruction, loaded per thread so
// that none of them becomes a uniform register or an immediate -- what matrix arithmetic on per-track values issues.
constexpr int kPackedChains = 8;
template <int MODE>
__global__ void __launch_bounds__(128)
ffma2_rate_kernel(int outer, float a, float b, const float* __restrict__ init, float* sink) {
    float2 x[kPackedChains], y[kPackedChains], z[kPackedChains];
#pragma unroll
    for (int c = 0; c < kPackedChains; ++c) {
        const float2* g = reinterpret_cast<const float2*>(init) + (threadIdx.x & 31) * 3 * kPackedChains + 3 * c;
        x[c] = g[0]; y[c] = g[1]; z[c] = g[2];
        x[c].x += (float)threadIdx.x * 1e-3f;
    }
    const float2 A = make_float2(a, a), B = make_float2(b, b);
    for (int o = 0; o < outer; ++o) {
#pragma unroll 8
        for (int i = 0; i < kInner; ++i) {
#pragma unroll
            for (int c = 0; c < kPackedChains; ++c) x[c] = MODE == 0 ? __ffma2_rn(x[c], A, B) : __ffma2_rn(x[c], y[c], z[c]);
        }
    }
    float s = 0.0f;
#pragma unroll
    for (int c = 0; c < kPackedChains; ++c) s += x[c].x + x[c].y;
    if (s == 123.456f) sink[0] = s;
}

}  // namespace

// TFLOP/s of FFMA2 (4 flop per lane and instruction) with shared operands and with three distinct register pairs;
// `scratch`: >= 32 * 3 * 8 float2 of device memory holding finite values + 1 float for the sink behind them.
cudaError_t measure_fp32_packed_rate(cudaStream_t stream, int repeats, float* scratch, double* shared_tflops,
                                     double* distinct_tflops) {
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int blocks = sms * 16;  // 2048 threads per SM
    const int outer = 32;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    float* sink = scratch + 32 * 3 * kPackedChains * 2;
    cudaError_t err = cudaSuccess;
    for (int mode = 0; mode < 2 && err == cudaSuccess; ++mode) {
        double best = 0.0;
        for (int r = 0; r < repeats + 1; ++r) {
            cudaEventRecord(e0, stream);
            if (mode == 0) ffma2_rate_kernel<0><<<blocks, 128, 0, stream>>>(outer, 0.999f, 1e-3f, scratch, sink);
            else ffma2_rate_kernel<1><<<blocks, 128, 0, stream>>>(outer, 0.999f, 1e-3f, scratch, sink);
            cudaEventRecord(e1, stream);
            err = cudaEventSynchronize(e1);
            if (err != cudaSuccess) break;
            float ms = 0.0f;
            cudaEventElapsedTime(&ms, e0, e1);
            const double flop = 4.0 * (double)blocks * 128 * kPackedChains * (double)kInner * outer;
            if (r > 0 && ms > 0.0f && flop / (ms * 1e-3) / 1e12 > best) best = flop / (ms * 1e-3) / 1e12;
        }
        *(mode == 0 ? shared_tflops : distinct_tflops) = best;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return err;
}

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
