// Shared host/device helpers of libgtb_kpm.so (product code; nothing here is used by oracle/).
#pragma once

#include <cuda_runtime.h>

#include <cstddef>
#include <cstdint>

#include "gtb.h"

namespace gtb {

constexpr int kSmCount = 148;  // B200: 2 dies x 74 SMs; grids are sized in multiples of this

// ---- error plumbing ---------------------------------------------------------
void note_cuda_error(cudaError_t e, const char* where);
void count_launch(int64_t k = 1);

#define GTB_CUDA_TRY(expr)                         \
  do {                                             \
    cudaError_t e__ = (expr);                      \
    if (e__ != cudaSuccess) {                      \
      ::gtb::note_cuda_error(e__, #expr);          \
      return GTB_ERR_CUDA;                         \
    }                                              \
  } while (0)

// after a <<<>>> launch
#define GTB_LAUNCHED()                             \
  do {                                             \
    ::gtb::count_launch();                         \
    cudaError_t e__ = cudaGetLastError();          \
    if (e__ != cudaSuccess) {                      \
      ::gtb::note_cuda_error(e__, "kernel launch"); \
      return GTB_ERR_CUDA;                         \
    }                                              \
  } while (0)

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

// Carves aligned sub-buffers out of the caller's workspace.
struct Carver {
  char* base;
  size_t off = 0;
  explicit Carver(void* p) : base(static_cast<char*>(p)) {}
  template <typename T>
  T* take(size_t count) {
    T* p = reinterpret_cast<T*>(base + off);
    off += align_up(count * sizeof(T));
    return p;
  }
};

// ---- device reductions --------------------------------------------------------
#ifdef __CUDACC__
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double warp_min(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_down_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ int warp_max_i(int v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = max(v, __shfl_down_sync(0xffffffffu, v, o));
  return v;
}
#endif

}  // namespace gtb
