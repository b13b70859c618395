// rpy_bench_aids.cu -- measurement aids of bench.py (bench_aids/rpy_bench_aids.h); not product code.
//   rpy_bench_pipe_probe     register-only chains of independent fused multiply-adds (or MUFU.RSQ) on
//                            every SM, timed with CUDA events: the denominator of the ALU roofline
//                             on the very GPU and at the very clocks the matvec runs
//                            at, because MEASURED_PEAKS.json holds only the HBM and bf16 tensor peaks;
//   rpy_bench_coissue_probe  DFMA chains and FFMA2 chains co-resident on every SM;
//   rpy_bench_matvec_phases  the product with CUDA events around each of its kernels.
#include <cuda_runtime.h>
#include <stdint.h>
#include "rpy_bench_aids.h"
#include "../paper_1602_02170_b200/csrc/rpy_internal.h"

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

// ---- cost of an FP-pipe instruction by operand form (rpy_bench_operand_probe)
// 12 independent accumulators per thread, 128 threads per CTA, `ctas_per_sm` CTAs per SM (the symmetric kernel runs 3
// (fp32) / 4 (fp64) such CTAs per SM).  Operands come from device memory as 64-bit loads so that every packed value sits
// in an aligned register pair (values built from scalars make the compiler insert MOVs into the loop).
constexpr int kFormChains = 12;

template <int KIND>
__global__ void __launch_bounds__(128, 4) form_kernel(int iters, const double* __restrict__ in, double* sink)
{
    constexpr int NC = kFormChains;
    if (KIND < 5) {
        const float2* in2 = reinterpret_cast<const float2*>(in);
        float2 acc[NC], x[NC], y[NC];
        float sc[NC];
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            acc[c] = in2[(3 * c + 0) * 128 + threadIdx.x];
            x[c] = in2[(3 * c + 1) * 128 + threadIdx.x];
            y[c] = in2[(3 * c + 2) * 128 + threadIdx.x];
            sc[c] = in2[(3 * NC + c) * 128 + threadIdx.x].x;
        }
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int c = 0; c < NC; ++c) {
                if (KIND == 0) acc[c] = __ffma2_rn(x[c], x[c], acc[c]);                        // two distinct register pairs
                if (KIND == 1) acc[c] = __ffma2_rn(x[c], make_float2(1.5f, 1.5f), acc[c]);     // two pairs and an immediate
                if (KIND == 2) acc[c] = __ffma2_rn(x[c], y[(c + 5) % NC], acc[c]);             // three distinct pairs, none shared with the neighbours
                if (KIND == 3) acc[c] = __ffma2_rn(x[c], y[0], acc[c]);                        // three distinct pairs, one the same as the neighbour's (.reuse)
                if (KIND == 4) acc[c] = __ffma2_rn(x[c], make_float2(sc[c], sc[c]), acc[c]);   // two pairs and one 32-bit scalar (.F32 operand)
            }
        }
        float s = 0.f;
#pragma unroll
        for (int c = 0; c < NC; ++c) s += acc[c].x + acc[c].y;
        if (s == 12345.678f) sink[0] = s;
    } else {
        double acc[NC], x[NC], y[NC];
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            acc[c] = in[(3 * c + 0) * 128 + threadIdx.x];
            x[c] = in[(3 * c + 1) * 128 + threadIdx.x];
            y[c] = in[(3 * c + 2) * 128 + threadIdx.x];
        }
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int c = 0; c < NC; ++c) {
                if (KIND == 5) acc[c] = fma(x[c], x[c], acc[c]);
                if (KIND == 6) acc[c] = fma(x[c], y[(c + 5) % NC], acc[c]);
                if (KIND == 7) acc[c] = fma(x[c], y[0], acc[c]);
            }
        }
        double s = 0.;
#pragma unroll
        for (int c = 0; c < NC; ++c) s += acc[c];
        if (s == 12345.678) sink[0] = s;
    }
}

// ---- FP64 pipe beside the FP32 pipe
constexpr int kMixChains = 12;
constexpr int kMixThreads = 128;
constexpr int kMixCtasPerSM = 8;

template <int THREE>
__device__ __forceinline__ void mix_f32(int iters, float seed, double* sink)
{
    float2 acc[kMixChains], x[kMixChains];
#pragma unroll
    for (int c = 0; c < kMixChains; ++c) {
        acc[c] = make_float2((float)(threadIdx.x + c), (float)c);
        x[c] = make_float2(1.0f + seed * (c + 1) * 1e-9f, 1.0f - seed * (c + 2) * 1e-9f);
    }
    const float2 a = make_float2(1.0f + seed * 1e-9f, 1.0f - seed * 1e-9f), b = make_float2(seed * 1e-9f, -seed * 1e-9f);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int c = 0; c < kMixChains; ++c)
            acc[c] = THREE ? __ffma2_rn(acc[c], x[c], x[(c + 5) % kMixChains]) : __ffma2_rn(acc[c], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < kMixChains; ++c) s += acc[c].x + acc[c].y;
    if (s == 12345.678f) sink[0] = s;
}

template <int THREE>
__device__ __forceinline__ void mix_f64(int iters, float seed, double* sink)
{
    double acc[kMixChains], x[kMixChains];
#pragma unroll
    for (int c = 0; c < kMixChains; ++c) { acc[c] = (double)(threadIdx.x + c); x[c] = 1.0 + seed * (c + 1) * 1e-12; }
    const double a = 1.0 + seed * 1e-12, b = seed * 1e-12;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int c = 0; c < kMixChains; ++c)
            acc[c] = THREE ? fma(acc[c], x[c], x[(c + 5) % kMixChains]) : fma(acc[c], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < kMixChains; ++c) s += acc[c];
    if (s == 12345.678) sink[0] = s;
}

// every CTA takes a slot number on its SM (arrival order); slots < n64 run DFMA chains, the others FFMA2 chains
template <int THREE>
__global__ void __launch_bounds__(kMixThreads) mix_kernel(int n64, int it32, int it64, float seed, double* sink, unsigned* slots)
{
    __shared__ unsigned s_slot;
    if (threadIdx.x == 0) {
        unsigned smid;
        asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
        s_slot = atomicAdd(&slots[smid & 255u], 1u);
    }
    __syncthreads();
    if ((int)s_slot < n64) mix_f64<THREE>(it64, seed, sink);
    else mix_f32<THREE>(it32, seed, sink);
}

}  // namespace

extern "C" int rpy_bench_coissue_probe(int n64_per_sm, int iters32, int iters64, int three_reg, void* d_scratch,
                                       float* h_elapsed_ms, double* h_ops32, double* h_ops64, void* cuda_stream)
{
    if (n64_per_sm < 0 || n64_per_sm > kMixCtasPerSM || iters32 < 0 || iters64 < 0) return 2;
    if (!d_scratch || !h_elapsed_ms || !h_ops32 || !h_ops64) return 1;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    double* sink = static_cast<double*>(d_scratch);
    unsigned* slots = reinterpret_cast<unsigned*>(sink + 1);
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return 5;
    float best = 0.f;
    cudaError_t e = cudaSuccess;
    for (int rep = 0; rep < 3 && e == cudaSuccess; ++rep) {      // rep 0 warms up; the faster of the other two counts
        cudaMemsetAsync(slots, 0, 256 * sizeof(unsigned), st);
        cudaEventRecord(e0, st);
        if (three_reg) mix_kernel<1><<<kNumSMs * kMixCtasPerSM, kMixThreads, 0, st>>>(n64_per_sm, iters32, iters64, 0.f, sink, slots);
        else           mix_kernel<0><<<kNumSMs * kMixCtasPerSM, kMixThreads, 0, st>>>(n64_per_sm, iters32, iters64, 0.f, sink, slots);
        cudaEventRecord(e1, st);
        e = cudaEventSynchronize(e1);
        if (e == cudaSuccess) e = cudaGetLastError();
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (rep == 1 || (rep == 2 && ms < best)) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (e != cudaSuccess) return 5;
    *h_elapsed_ms = best;
    *h_ops32 = (double)kNumSMs * (kMixCtasPerSM - n64_per_sm) * kMixThreads * (double)iters32 * kMixChains * 2.0;
    *h_ops64 = (double)kNumSMs * n64_per_sm * kMixThreads * (double)iters64 * kMixChains;
    return 0;
}

extern "C" int rpy_bench_matvec_phases(int wall, int prec, int64_t n_blobs, int n_rhs, const void* d_pos,
                                       const void* d_force, void* d_vel, double a, double eta, void* d_workspace,
                                       size_t workspace_bytes, void* cuda_stream, void* const* cuda_events4)
{
    return (int)rpy::matvec_phases(wall != 0, static_cast<rpy_prec>(prec), n_blobs, n_rhs, d_pos, d_force, d_vel, a, eta,
                                   d_workspace, workspace_bytes, cuda_stream, cuda_events4);
}

extern "C" int rpy_bench_pipe_probe(int kind, int iters, void* d_sink, float* h_elapsed_ms,
                                    double* h_fma_count, void* cuda_stream)
{
    if (kind < 0 || kind > 5 || iters < 1) return 2;
    if (!d_sink || !h_elapsed_ms || !h_fma_count) return 1;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return 5;
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
    if (e != cudaSuccess) return 5;
    *h_elapsed_ms = ms;
    double per_thread = (double)iters * kChains * ((kind == 1 || kind == 4) ? 2.0 : 1.0);
    *h_fma_count = per_thread * kThreads * (double)grid.x;
    return 0;
}

extern "C" int rpy_bench_operand_probe(int kind, int ctas_per_sm, int iters, void* d_scratch, float* h_elapsed_ms,
                                       double* h_lane_ops, void* cuda_stream)
{
    if (kind < 0 || kind > 7 || iters < 1 || ctas_per_sm < 1 || ctas_per_sm > 4) return 2;
    if (!d_scratch || !h_elapsed_ms || !h_lane_ops) return 1;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return 5;
    dim3 grid(kNumSMs * ctas_per_sm);
    const double* in = static_cast<const double*>(d_scratch) + 1;      // [0] is the sink
    double* sink = static_cast<double*>(d_scratch);
    auto launch = [&](int n) {
        switch (kind) {
            case 0: form_kernel<0><<<grid, 128, 0, st>>>(n, in, sink); break;
            case 1: form_kernel<1><<<grid, 128, 0, st>>>(n, in, sink); break;
            case 2: form_kernel<2><<<grid, 128, 0, st>>>(n, in, sink); break;
            case 3: form_kernel<3><<<grid, 128, 0, st>>>(n, in, sink); break;
            case 4: form_kernel<4><<<grid, 128, 0, st>>>(n, in, sink); break;
            case 5: form_kernel<5><<<grid, 128, 0, st>>>(n, in, sink); break;
            case 6: form_kernel<6><<<grid, 128, 0, st>>>(n, in, sink); break;
            default: form_kernel<7><<<grid, 128, 0, st>>>(n, in, sink); break;
        }
    };
    launch(iters > 64 ? 64 : iters);
    cudaEventRecord(e0, st);
    launch(iters);
    cudaEventRecord(e1, st);
    cudaError_t e = cudaEventSynchronize(e1);
    if (e == cudaSuccess) e = cudaGetLastError();
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (e != cudaSuccess) return 5;
    *h_elapsed_ms = ms;
    *h_lane_ops = (double)iters * kFormChains * (kind < 5 ? 2.0 : 1.0) * 128.0 * (double)grid.x;
    return 0;
}
