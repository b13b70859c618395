// rpy_probe.cu -- rpy_pipe_peak_probe: register-only chains of independent fused multiply-adds
// (or MUFU.RSQ) on every SM, timed with CUDA events.  It measures the denominator of the ALU
// roofline on the very GPU and at the very clocks the matvec runs at,
// because MEASURED_PEAKS.json holds only the HBM and bf16 tensor peaks.
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/rpy_matvec.h"

namespace {

constexpr int kChains = 16;     // independent accumulators per thread
constexpr int kThreads = 256;
constexpr int kCtasPerSM = 8;
constexpr int kNumSMs = 148;

template <int KIND>
__global__ void __launch_bounds__(kThreads) probe_kernel(int iters, float seed, double* sink)
{
    if (KIND == 0) {            // scalar FFMA
        float acc[kChains];
        float a = 1.0f + seed * 1e-9f, b = seed * 1e-9f;
#pragma unroll
        for (int c = 0; c < kChains; ++c) acc[c] = (float)(threadIdx.x + c);
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int c = 0; c < kChains; ++c) acc[c] = fmaf(acc[c], a, b);
        }
        float s = 0.f;
#pragma unroll
        for (int c = 0; c < kChains; ++c) s += acc[c];
        if (s == 12345.678f) sink[0] = s;
    } else if (KIND == 1) {     // packed FFMA2
        float2 acc[kChains];
        float2 a = make_float2(1.0f + seed * 1e-9f, 1.0f - seed * 1e-9f), b = make_float2(seed * 1e-9f, -seed * 1e-9f);
#pragma unroll
        for (int c = 0; c < kChains; ++c) acc[c] = make_float2((float)(threadIdx.x + c), (float)c);
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int c = 0; c < kChains; ++c) acc[c] = __ffma2_rn(acc[c], a, b);
        }
        float s = 0.f;
#pragma unroll
        for (int c = 0; c < kChains; ++c) s += acc[c].x + acc[c].y;
        if (s == 12345.678f) sink[0] = s;
    } else if (KIND == 2) {     // DFMA
        double acc[kChains];
        double a = 1.0 + seed * 1e-12, b = seed * 1e-12;
#pragma unroll
        for (int c = 0; c < kChains; ++c) acc[c] = (double)(threadIdx.x + c);
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int c = 0; c < kChains; ++c) acc[c] = fma(acc[c], a, b);
        }
        double s = 0.0;
#pragma unroll
        for (int c = 0; c < kChains; ++c) s += acc[c];
        if (s == 12345.678) sink[0] = s;
    } else if (KIND == 4) {     // packed FFMA2, three distinct register-pair operands per instruction
        float2 acc[kChains], x[kChains];
#pragma unroll
        for (int c = 0; c < kChains; ++c) {
            acc[c] = make_float2((float)(threadIdx.x + c), (float)c);
            x[c] = make_float2(1.0f + seed * (c + 1) * 1e-9f, 1.0f - seed * (c + 2) * 1e-9f);
        }
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int c = 0; c < kChains; ++c) acc[c] = __ffma2_rn(acc[c], x[c], x[(c + 5) % kChains]);
        }
        float s = 0.f;
#pragma unroll
        for (int c = 0; c < kChains; ++c) s += acc[c].x + acc[c].y;
        if (s == 12345.678f) sink[0] = s;
    } else if (KIND == 5) {     // scalar FFMA, three distinct register operands per instruction
        float acc[kChains], x[kChains];
#pragma unroll
        for (int c = 0; c < kChains; ++c) {
            acc[c] = (float)(threadIdx.x + c);
            x[c] = 1.0f + seed * (c + 1) * 1e-9f;
        }
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int c = 0; c < kChains; ++c) acc[c] = fmaf(acc[c], x[c], x[(c + 5) % kChains]);
        }
        float s = 0.f;
#pragma unroll
        for (int c = 0; c < kChains; ++c) s += acc[c];
        if (s == 12345.678f) sink[0] = s;
    } else {                    // MUFU.RSQ
        float acc[kChains];
#pragma unroll
        for (int c = 0; c < kChains; ++c) acc[c] = 1.0f + (float)(threadIdx.x + c) + seed;
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int c = 0; c < kChains; ++c) asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(acc[c]));
        }
        float s = 0.f;
#pragma unroll
        for (int c = 0; c < kChains; ++c) s += acc[c];
        if (s == 12345.678f) sink[0] = s;
    }
}

}  // namespace

extern "C" rpy_status rpy_pipe_peak_probe(int kind, int iters, void* d_sink, float* h_elapsed_ms,
                                          double* h_fma_count, void* cuda_stream)
{
    if (kind < 0 || kind > 5 || iters < 1) return RPY_ERR_ARG;
    if (!d_sink || !h_elapsed_ms || !h_fma_count) return RPY_ERR_NULL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return RPY_ERR_CUDA;
    dim3 grid(kNumSMs * kCtasPerSM);
    double* sink = static_cast<double*>(d_sink);
    auto launch = [&](int n) {
        switch (kind) {
            case 0: probe_kernel<0><<<grid, kThreads, 0, st>>>(n, 0.f, sink); break;
            case 1: probe_kernel<1><<<grid, kThreads, 0, st>>>(n, 0.f, sink); break;
            case 2: probe_kernel<2><<<grid, kThreads, 0, st>>>(n, 0.f, sink); break;
            case 4: probe_kernel<4><<<grid, kThreads, 0, st>>>(n, 0.f, sink); break;
            case 5: probe_kernel<5><<<grid, kThreads, 0, st>>>(n, 0.f, sink); break;
            default: probe_kernel<3><<<grid, kThreads, 0, st>>>(n, 0.f, sink); break;
        }
    };
    launch(iters > 64 ? 64 : iters);            // warm-up
    cudaEventRecord(e0, st);
    launch(iters);
    cudaEventRecord(e1, st);
    cudaError_t e = cudaEventSynchronize(e1);
    if (e == cudaSuccess) e = cudaGetLastError();
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (e != cudaSuccess) return RPY_ERR_CUDA;
    *h_elapsed_ms = ms;
    double per_thread = (double)iters * kChains * ((kind == 1 || kind == 4) ? 2.0 : 1.0);
    *h_fma_count = per_thread * kThreads * (double)grid.x;
    return RPY_OK;
}
