// rpy_launch.cuh -- programmatic dependent launch, shared by the product (rpy_kernels.cuh) and the rigid layer.
#pragma once
#include <cuda_runtime.h>

namespace rpy {

// ---------------------------------------------------------------------------- programmatic dependent launch
// The product is three dependent kernels and a Krylov iteration seven; below N ~ 10^4 the gaps between them are
// a visible share of the time.  Every kernel of those chains starts with pdl_enter() and is launched with
// launch_pdl(): its CTAs may be scheduled while the last CTAs of the kernel before it are still running, and
// block in griddepcontrol.wait until that kernel has completed and its writes are visible -- only the launch
// latency overlaps, no data is touched early.  Every CTA waits before it does anything else (also before an
// early return), so completion stays transitive along the chain.  Launched the ordinary way (<<< >>>), both
// instructions are no-ops.
__device__ __forceinline__ void pdl_enter()
{
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}
// The long kernels (all-pairs) only wait: their dependents are released when they complete.  Released at entry, the
// CTAs of every later kernel of a chain cascade into residency and wait there for the whole all-pairs kernel --
// measured (ten products replayed from a CUDA graph, fp64, N = 4,000): 100.6 us per product against 63.9 without.
__device__ __forceinline__ void pdl_wait()
{
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

// chained = false: an ordinary launch (the kernel starts after everything before it in the stream has completed).
template <class... P, class... A>
inline cudaError_t launch_chain(bool chained, void (*kernel)(P...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, A... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = chained ? 1 : 0;
#ifdef RPY_NO_PDL                     // A/B measurement: cfg 1 product 48.9 -> 44.5 us, cfg 2 mixed solve 16.09 -> 15.60 ms
    cfg.numAttrs = 0;
#endif
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<P>(args)...);
}

template <class... P, class... A>
inline cudaError_t launch_pdl(void (*kernel)(P...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, A... args)
{
    return launch_chain(true, kernel, grid, block, smem, st, args...);
}

}  // namespace rpy
