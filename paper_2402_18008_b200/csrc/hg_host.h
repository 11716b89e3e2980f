// hg_host.h -- host-side helpers shared by the translation units of libhg.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/hg.h"

namespace hg {

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
inline bool aligned4(const void* p)  { return (reinterpret_cast<uintptr_t>(p) & 3u) == 0; }

inline int cuda_status(cudaError_t e) { return e == cudaSuccess ? HG_OK : HG_ERR_CUDA; }

// Result of the last launch on this thread -> hg status (clears the sticky-less error state).
inline int launch_status() { return cuda_status(cudaGetLastError()); }

// Device-pointer solve shared by the device and the host-buffer entry points (hg_batched.cu).
int solve_batched(int method, const float* src, const float* dst, float* H, int64_t n,
                  int64_t plane_stride, hg_layout_t layout, hg_norm_t norm, hg_precision_t prec,
                  cudaStream_t stream);

}  // namespace hg
