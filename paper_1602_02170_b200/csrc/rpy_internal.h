// rpy_internal.h -- the few host-side helpers the translation units of librpy_matvec.so share
// (not part of the C ABI; nothing here is exported with C linkage).
#pragma once
#include <cuda_runtime.h>
#include "../../include/rpy_matvec.h"

namespace rpy {
// Records `e` as the calling thread's last CUDA error (rpy_last_cuda_error) and returns RPY_ERR_CUDA.
rpy_status set_cuda_error(cudaError_t e);

// The per-slice partial sums of one product whose finalise step is left to the caller:
//   u[s][row][c] = scale * sum_{slice < n_slices} partial[slice * per_chunk + (s * n + row) * 3 + c]
// (s = right-hand side, n = n_blobs).  They live in the product's workspace until its next use.
struct PartialSums { const double* partial; int n_slices; int64_t per_chunk; double scale; };

// The device product with explicit element strides between the right-hand sides of force and vel
// (>= 3 n each): lets the batched solver hand over the lambda parts of its solver vectors in place.
//   d_skip    optional device flag; when it is non-zero at execution time every kernel of the call returns
//             at once (the Krylov solver enqueues an iteration ahead of the device-side convergence test);
//   partials  optional: prepack and all-pairs only, *partials describes the slices (d_vel is not written and
//             may be NULL); n_rhs must then be 1, 2, 4 or 8 (one right-hand-side group);
//   shard / n_shards  (0, 1) for the whole product; otherwise 1/n_shards of the unordered tile pairs of the
//             symmetric kernel (n_rhs == 1 and matvec_shardable(n) required), contributing to every row;
//   vel_f64   d_vel is double whatever the path (the fp32 path's result without the final rounding to float).
rpy_status matvec_strided(bool wall, rpy_prec prec, int64_t n, int n_rhs, const void* d_pos, const void* d_force,
                          int64_t force_stride3, void* d_vel, int64_t vel_stride3, double a, double eta,
                          void* ws, size_t ws_bytes, cudaStream_t st, const int* d_skip = nullptr,
                          PartialSums* partials = nullptr, int shard = 0, int n_shards = 1, bool vel_f64 = false);
bool matvec_shardable(int64_t n);

// The whole-matrix product with four caller-owned CUDA events (cudaEvent_t as void*) recorded on the
// launch stream: [0] before prepack, [1] before the all-pairs kernel, [2] after it, [3] after finalise
// (first right-hand-side group).  Not part of the C ABI: bench_aids/ links against it to time the
// dominant kernel on the stream it is launched on.
__attribute__((visibility("default")))
rpy_status matvec_phases(bool wall, rpy_prec prec, int64_t n_blobs, int n_rhs, const void* d_pos, const void* d_force,
                         void* d_vel, double a, double eta, void* ws, size_t ws_bytes, void* stream, void* const* events4);
}  // namespace rpy
