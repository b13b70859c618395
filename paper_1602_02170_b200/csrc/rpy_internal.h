// rpy_internal.h -- the few host-side helpers the translation units of librpy_matvec.so share
// (not part of the C ABI; nothing here is exported with C linkage).
#pragma once
#include <cuda_runtime.h>
#include "../../include/rpy_matvec.h"

namespace rpy {
// Records `e` as the calling thread's last CUDA error (rpy_last_cuda_error) and returns RPY_ERR_CUDA.
rpy_status set_cuda_error(cudaError_t e);
}  // namespace rpy
