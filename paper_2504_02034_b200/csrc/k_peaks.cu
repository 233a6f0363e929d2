// k_peaks.cu -- plain-ALU peak micro-benchmarks: the roofline denominators of the KDE and sample kernels.
//
// The hot path is bound by the SMs' arithmetic pipes, not by HBM or the tensor cores:
// MEASURED_PEAKS.json only holds a copy bandwidth and a bf16 GEMM rate, so the library measures the three
// pipe rates it is bound by -- MUFU.EX2 (the KDE pair loop), FFMA (its companion pipe) and DFMA (the fp64
// sample/injection weights) -- on the device it runs on.  Each kernel is 8 independent dependency chains per
// thread, unrolled, enough warps to cover the pipe latency; the rate is thread-level instructions / second.
#include "chim_internal.cuh"

namespace chim {

constexpr int kPeakThreads = 256, kPeakIters = 2048, kPeakChains = 8;

__global__ void __launch_bounds__(kPeakThreads) k_peak_ex2(float* out, float seed) {
    float x[kPeakChains];
#pragma unroll
    for (int c = 0; c < kPeakChains; ++c) x[c] = seed + 0.001f * (threadIdx.x + c);
#pragma unroll 1
    for (int it = 0; it < kPeakIters; ++it) {
#pragma unroll
        for (int c = 0; c < kPeakChains; ++c) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(x[c]));
#pragma unroll
        for (int c = 0; c < kPeakChains; ++c) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(x[c]));
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < kPeakChains; ++c) s += x[c];
    if (s == 123.456f) out[0] = s;
}

__global__ void __launch_bounds__(kPeakThreads) k_peak_ffma(float* out, float a, float b) {
    float x[kPeakChains];
#pragma unroll
    for (int c = 0; c < kPeakChains; ++c) x[c] = 0.001f * (threadIdx.x + c);
#pragma unroll 1
    for (int it = 0; it < kPeakIters; ++it) {
#pragma unroll
        for (int c = 0; c < kPeakChains; ++c) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(x[c]) : "f"(a), "f"(b));
#pragma unroll
        for (int c = 0; c < kPeakChains; ++c) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(x[c]) : "f"(a), "f"(b));
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < kPeakChains; ++c) s += x[c];
    if (s == 123.456f) out[0] = s;
}

__global__ void __launch_bounds__(kPeakThreads) k_peak_dfma(double* out, double a, double b) {
    double x[kPeakChains];
#pragma unroll
    for (int c = 0; c < kPeakChains; ++c) x[c] = 0.001 * (threadIdx.x + c);
#pragma unroll 1
    for (int it = 0; it < kPeakIters; ++it) {
#pragma unroll
        for (int c = 0; c < kPeakChains; ++c) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(x[c]) : "d"(a), "d"(b));
#pragma unroll
        for (int c = 0; c < kPeakChains; ++c) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(x[c]) : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < kPeakChains; ++c) s += x[c];
    if (s == 123.456) out[0] = s;
}

__global__ void __launch_bounds__(kPeakThreads) k_peak_ffma2(float* out, float a, float b) {
    unsigned long long x[kPeakChains];
    const float2 ab = make_float2(a, a), bb = make_float2(b, b);
    const unsigned long long a2 = *reinterpret_cast<const unsigned long long*>(&ab), b2 = *reinterpret_cast<const unsigned long long*>(&bb);
#pragma unroll
    for (int c = 0; c < kPeakChains; ++c) {
        float2 v = make_float2(0.001f * (threadIdx.x + c), 0.002f * (threadIdx.x + c));
        x[c] = *reinterpret_cast<unsigned long long*>(&v);
    }
#pragma unroll 1
    for (int it = 0; it < kPeakIters; ++it) {
#pragma unroll
        for (int c = 0; c < kPeakChains; ++c) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(x[c]) : "l"(a2), "l"(b2));
#pragma unroll
        for (int c = 0; c < kPeakChains; ++c) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(x[c]) : "l"(a2), "l"(b2));
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < kPeakChains; ++c) { float2 v = *reinterpret_cast<float2*>(&x[c]); s += v.x + v.y; }
    if (s == 123.456f) out[0] = s;
}

// Runs each micro-benchmark `reps` times after one warm-up and returns the best rates in G lane-instructions/s:
// out_g = {MUFU.EX2, FFMA, DFMA, FFMA2 counted as two lane-instructions}.
cudaError_t measure_alu_peaks(int n_sm, int reps, cudaStream_t st, double out_g[4]) {
    void* scratch = nullptr;
    cudaError_t e = cudaMalloc(&scratch, 64);
    if (e != cudaSuccess) return e;
    cudaEvent_t a, b;
    cudaEventCreate(&a);
    cudaEventCreate(&b);
    const int grid = n_sm * 8;
    const double ops = (double)grid * kPeakThreads * kPeakIters * kPeakChains * 2.0;
    double best[4] = {0.0, 0.0, 0.0, 0.0};
    for (int k = 0; k < 4; ++k) {
        for (int r = 0; r <= reps; ++r) {
            cudaEventRecord(a, st);
            if (k == 0) k_peak_ex2<<<grid, kPeakThreads, 0, st>>>(static_cast<float*>(scratch), -0.5f);
            else if (k == 1) k_peak_ffma<<<grid, kPeakThreads, 0, st>>>(static_cast<float*>(scratch), 0.999f, 0.001f);
            else if (k == 2) k_peak_dfma<<<grid, kPeakThreads, 0, st>>>(static_cast<double*>(scratch), 0.999, 0.001);
            else k_peak_ffma2<<<grid, kPeakThreads, 0, st>>>(static_cast<float*>(scratch), 0.999f, 0.001f);
            cudaEventRecord(b, st);
            e = cudaEventSynchronize(b);
            if (e != cudaSuccess) break;
            float ms = 0.f;
            cudaEventElapsedTime(&ms, a, b);
            if (r > 0 && ms > 0.f) best[k] = fmax(best[k], (k == 3 ? 2.0 : 1.0) * ops / (ms * 1e-3) / 1e9);
        }
        if (e != cudaSuccess) break;
    }
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    cudaFree(scratch);
    if (e == cudaSuccess) e = cudaGetLastError();
    for (int k = 0; k < 4; ++k) out_g[k] = best[k];
    return e;
}

}  // namespace chim
