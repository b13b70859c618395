// rpy_internal.h -- the few host-side helpers the translation units of librpy_matvec.so share
// (not part of the C ABI; nothing here is exported with C linkage).
#pragma once
#include <cuda_runtime.h>
#include "../../include/rpy_matvec.h"

namespace rpy {
// Records `e` as the calling thread's last CUDA error (rpy_last_cuda_error) and returns RPY_ERR_CUDA.
rpy_status set_cuda_error(cudaError_t e);

// The device product with explicit element strides between the right-hand sides of force and vel
// (>= 3 n each): lets the batched solver hand over the lambda parts of its solver vectors in place.
rpy_status matvec_strided(bool wall, rpy_prec prec, int64_t n, int n_rhs, const void* d_pos, const void* d_force,
                          int64_t force_stride3, void* d_vel, int64_t vel_stride3, double a, double eta,
                          void* ws, size_t ws_bytes, cudaStream_t st);

// The whole-matrix product with four caller-owned CUDA events (cudaEvent_t as void*) recorded on the
// launch stream: [0] before prepack, [1] before the all-pairs kernel, [2] after it, [3] after finalise
// (first right-hand-side group).  Not part of the C ABI: bench_aids/ links against it to time the
// dominant kernel on the stream it is launched on.
__attribute__((visibility("default")))
rpy_status matvec_phases(bool wall, rpy_prec prec, int64_t n_blobs, int n_rhs, const void* d_pos, const void* d_force,
                         void* d_vel, double a, double eta, void* ws, size_t ws_bytes, void* stream, void* const* events4);
}  // namespace rpy
