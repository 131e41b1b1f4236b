// Vector loads/stores of the fused passes (product code; nothing here is used by oracle/).
// A vector element is VW doubles (VW = 2: one complex; VW = 4: two complex, one 256-bit access).
#pragma once

#include "cheb.cuh"

namespace gtb {

// ---- vector element = VW doubles (VW = 2: one complex; VW = 4: two complex, 256-bit) -----
template <int VW>
struct Vec {
  double v[VW];
};

template <int VW>
__device__ __forceinline__ Vec<VW> load_gather(const double* p);  // read-only path, keep in L1
template <int VW>
__device__ __forceinline__ Vec<VW> load_stream(const double* p);  // read once: do not allocate L1
template <int VW>
__device__ __forceinline__ void store_stream(double* p, const Vec<VW>& x);

template <>
__device__ __forceinline__ Vec<2> load_gather<2>(const double* p) {
  Vec<2> r;
  asm volatile("ld.global.nc.v2.f64 {%0,%1}, [%2];" : "=d"(r.v[0]), "=d"(r.v[1]) : "l"(p));
  return r;
}
template <>
__device__ __forceinline__ Vec<4> load_gather<4>(const double* p) {
  Vec<4> r;
  asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];"
               : "=d"(r.v[0]), "=d"(r.v[1]), "=d"(r.v[2]), "=d"(r.v[3])
               : "l"(p));
  return r;
}
template <>
__device__ __forceinline__ Vec<2> load_stream<2>(const double* p) {
  Vec<2> r;
  asm volatile("ld.global.L1::no_allocate.v2.f64 {%0,%1}, [%2];"
               : "=d"(r.v[0]), "=d"(r.v[1])
               : "l"(p)
               : "memory");
  return r;
}
template <>
__device__ __forceinline__ Vec<4> load_stream<4>(const double* p) {
  Vec<4> r;
  asm volatile("ld.global.L1::no_allocate.v4.f64 {%0,%1,%2,%3}, [%4];"
               : "=d"(r.v[0]), "=d"(r.v[1]), "=d"(r.v[2]), "=d"(r.v[3])
               : "l"(p)
               : "memory");
  return r;
}
template <>
__device__ __forceinline__ void store_stream<2>(double* p, const Vec<2>& x) {
  asm volatile("st.global.L1::no_allocate.v2.f64 [%0], {%1,%2};" ::"l"(p), "d"(x.v[0]), "d"(x.v[1])
               : "memory");
}
template <>
__device__ __forceinline__ void store_stream<4>(double* p, const Vec<4>& x) {
  asm volatile("st.global.L1::no_allocate.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(x.v[0]),
               "d"(x.v[1]), "d"(x.v[2]), "d"(x.v[3])
               : "memory");
}

__device__ __forceinline__ int32_t ld_stream_i32(const int32_t* p) {
  int32_t v;
  asm volatile("ld.global.nc.L1::no_allocate.s32 %0, [%1];" : "=r"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ double ld_stream_f64(const double* p) {
  double v;
  asm volatile("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(p));
  return v;
}

// acc += c * y on the complex numbers of a vector element (c = cr + i ci); the arithmetic of caxpy_kernel
template <int VW>
__device__ __forceinline__ void axpy_into(Vec<VW>& acc, const Vec<VW>& y, double cr, double ci) {
#pragma unroll
  for (int p = 0; p < VW / 2; ++p) {
    acc.v[2 * p] = fma(cr, y.v[2 * p], fma(-ci, y.v[2 * p + 1], acc.v[2 * p]));
    acc.v[2 * p + 1] = fma(cr, y.v[2 * p + 1], fma(ci, y.v[2 * p], acc.v[2 * p + 1]));
  }
}

// block sums of the two dot products -> one double2 per block
template <int kThreads>
__device__ __forceinline__ void block_store_sums(double s1, double s2, double2* out) {
  __shared__ double red[kThreads / 32][2];
  s1 = warp_sum(s1);
  s2 = warp_sum(s2);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) {
    red[wid][0] = s1;
    red[wid][1] = s2;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int w = 1; w < kThreads / 32; ++w) {
      s1 += red[w][0];
      s2 += red[w][1];
    }
    *out = make_double2(s1, s2);
  }
}

}  // namespace gtb
