// Chebyshev moments on the device: random-phase fill (K5), first pass (K6), fused recursion pass
// (K7) and moment finalisation (K8).
//
// The paper names the ingredients (sec. 2.4: Chebyshev expansion, kernel polynomial
// method, sparse matrix-vector multiplication, random phase approximation) and the quantity
// (Eq. 4); BASELINE.json:north_star fixes the recursion
//     |phi_{n+1}> = 2 H~ |phi_n> - |phi_{n-1}>,   H~ = (H - b)/a,
// the doubling identities m_{2n} = 2<phi_n|phi_n> - m_0, m_{2n+1} = 2 Re<phi_{n+1}|phi_n> - m_1 and
// the counter hash of the random phases (readings C3-C5 in DESIGN.md).
//
// K7 is the hot kernel: ONE pass over HBM per Chebyshev step.  Per row it streams the ELL slots
// (int32 column + fp64 hopping, slot-major so a warp reads contiguous words), gathers phi_n at the
// columns (R vectors interleaved per atom: one gather = R*16 contiguous bytes, 32 B = one sector
// and one 256-bit load for a pair of vectors), streams phi_{n-1}, writes phi_{n+1} over it, and
// accumulates <phi_n|phi_n> and Re<phi_{n+1}|phi_n> in registers -> warp shuffles -> one slot per
// block.  H is read once per pass for all R vectors.
#include <cooperative_groups.h>

#include <cmath>
#include <cstdlib>

#include "cheb.cuh"

namespace gtb {
namespace {

constexpr uint64_t kGamma = 0x9E3779B97F4A7C15ull;

// ---- counter hash (reading C3) ----------------------------------------------------------
__host__ __device__ __forceinline__ uint64_t mix64(uint64_t z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

// K5: phi[i][k] = exp(i theta), theta = fl(2 pi u(seed, r0 + k, i))
__global__ void __launch_bounds__(kBlock) random_phase_kernel(uint64_t seed, int32_t r0, int32_t R,
                                                              int64_t n, double2* __restrict__ phi) {
  const int64_t total = n * R;
  for (int64_t e = (int64_t)blockIdx.x * kBlock + threadIdx.x; e < total;
       e += (int64_t)gridDim.x * kBlock) {
    const int64_t i = e / R;
    const int32_t k = (int32_t)(e - i * R);
    const uint64_t key = mix64(seed + ((uint64_t)(uint32_t)(r0 + k) + 1ull) * kGamma);
    const uint64_t h = mix64(key + ((uint64_t)i + 1ull) * kGamma);
    const double u = (double)(h >> 11) * 0x1.0p-53;
    const double theta = 6.283185307179586 * u;
    double s, c;
    sincos(theta, &s, &c);
    phi[e] = make_double2(c, s);
  }
}

// exact-trace mode: phi[i][k] = delta(i, r0 + k)   (basis vectors e_{r0} .. e_{r0+R-1})
__global__ void __launch_bounds__(kBlock) basis_fill_kernel(int64_t r0, int32_t R, int64_t n,
                                                            double2* __restrict__ phi) {
  const int64_t total = n * R;
  for (int64_t e = (int64_t)blockIdx.x * kBlock + threadIdx.x; e < total;
       e += (int64_t)gridDim.x * kBlock) {
    const int64_t i = e / R;
    const int64_t k = e - i * R;
    phi[e] = make_double2(i == r0 + k ? 1.0 : 0.0, 0.0);
  }
}

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


// K6 / K7.  Thread e handles element e of phi viewed as an array of Vec<VW>: row = e / T, vector
// group t = e % T, so a warp touches one contiguous 32*VW*8-byte span of phi_{n-1}/phi_{n+1}, and
// every gather of a row's neighbour is T consecutive threads reading R*16 contiguous bytes.
template <int VW, int LOG2T, bool kFirst, bool kDiag, int CH, bool kDotL>
__global__ void __launch_bounds__(kBlock) cheb_step_kernel(const StepArgs a) {
  const int64_t n = a.n;
  const int T = LOG2T >= 0 ? (1 << LOG2T) : a.T;
  const int64_t total = n * T;
  const int width = a.width;
  const double scale = a.scale, b = a.b;
  double s1 = 0.0, s2 = 0.0;
  for (int64_t e = (int64_t)blockIdx.x * kBlock + threadIdx.x; e < total;
       e += (int64_t)gridDim.x * kBlock) {
    const int64_t row = LOG2T >= 0 ? (e >> LOG2T) : (e / T);
    const int64_t t = e - row * T;
    const double* xt = a.phi_cur + t * VW;
    const int32_t* cp = a.cols + row;
    const double* vp = a.vals + row;
    Vec<VW> acc;
#pragma unroll
    for (int q = 0; q < VW; ++q) acc.v[q] = 0.0;
    Vec<VW> prev;
    if (!kFirst) prev = load_stream<VW>(a.phi_io + e * VW);
    const Vec<VW> own = load_gather<VW>(a.phi_cur + e * VW);
    Vec<VW> with;
    if (kDotL) with = load_stream<VW>(a.dot_with + e * VW);
    if (CH == 0) {
#pragma unroll 4
      for (int k = 0; k < width; ++k) {
        const int64_t c = __ldg(cp + (size_t)k * n);
        const double v = __ldg(vp + (size_t)k * n);
        const Vec<VW> x = load_gather<VW>(xt + c * T * VW);
#pragma unroll
        for (int q = 0; q < VW; ++q) acc.v[q] = fma(v, x.v[q], acc.v[q]);
      }
    } else {
      // wide rows: CH slots at a time -- all CH column/hopping loads are issued before the CH
      // gathers that depend on them, so a thread keeps 2*CH + CH loads in flight instead of 4
      constexpr int C = CH > 0 ? CH : 1;
      for (int k0 = 0; k0 < width; k0 += C) {
        int32_t c[C];
        double v[C];
#pragma unroll
        for (int j = 0; j < C; ++j) {
          const bool ok = k0 + j < width;
          c[j] = ok ? __ldg(cp + (size_t)(k0 + j) * n) : (int32_t)row;
          v[j] = ok ? __ldg(vp + (size_t)(k0 + j) * n) : 0.0;
        }
        Vec<VW> x[C];
#pragma unroll
        for (int j = 0; j < C; ++j) x[j] = load_gather<VW>(xt + (int64_t)c[j] * T * VW);
#pragma unroll
        for (int j = 0; j < C; ++j)
#pragma unroll
          for (int q = 0; q < VW; ++q) acc.v[q] = fma(v[j], x[j].v[q], acc.v[q]);
      }
    }
    if (kDiag) {
      const double d = __ldg(a.diag + row);
#pragma unroll
      for (int q = 0; q < VW; ++q) acc.v[q] = fma(d, own.v[q], acc.v[q]);
    }
    Vec<VW> y;
#pragma unroll
    for (int q = 0; q < VW; ++q) {
      y.v[q] = (acc.v[q] - b * own.v[q]) * scale;
      if (!kFirst) y.v[q] -= prev.v[q];
      s1 = fma(own.v[q], kDotL ? with.v[q] : own.v[q], s1);
      s2 = fma(y.v[q], kDotL ? with.v[q] : own.v[q], s2);
    }
    store_stream<VW>(a.phi_io + e * VW, y);
  }
  __shared__ double red[kBlock / 32][2];
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
    for (int w = 1; w < kBlock / 32; ++w) {
      s1 += red[w][0];
      s2 += red[w][1];
    }
    a.partial[blockIdx.x] = make_double2(s1, s2);
  }
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

// ---- K7x2: K7 for narrow rows with two independent elements in flight per thread --------------------
// K7 above is latency-bound at K = 3 (ncu: 94 % of the stall cycles on long_scoreboard, DRAM at 76 %):
// per element a thread issues its two streamed loads and the K column/hopping loads, and only then the K
// gathers that depend on the columns.  Here every thread works on TWO elements per iteration, one grid
// stride apart: all 2 x (2 + 2W) independent loads are issued first, then the 2 x W gathers, then the FMAs
// and the two stores.  W (3 or 4) is a compile-time bound on the row width, so everything is unrolled and
// lives in registers (64 registers: still 4 blocks per SM).  Same arithmetic order per element as K7.
// Config 5: 2.20 -> 1.99 ms per pass.
template <int LOG2T, bool kDiag, int W, bool kDotL>
__global__ void __launch_bounds__(kBlock) cheb_step_x2_kernel(const StepArgs a) {
  constexpr int VW = 4;
  constexpr int T = 1 << LOG2T;
  constexpr int NE = 2;
  const int64_t n = a.n;
  const int64_t total = n * T;
  const int width = a.width;
  const double scale = a.scale, b = a.b;
  const int64_t stride = (int64_t)gridDim.x * kBlock;
  double s1 = 0.0, s2 = 0.0;
  for (int64_t e0 = (int64_t)blockIdx.x * kBlock + threadIdx.x; e0 < total; e0 += NE * stride) {
    int64_t e[NE];
    bool live[NE];
#pragma unroll
    for (int r = 0; r < NE; ++r) {
      e[r] = e0 + r * stride;   // one grid stride apart (adjacent 256-element chunks measured 4 % slower)
      live[r] = e[r] < total;
      if (!live[r]) e[r] = e0;   // a harmless duplicate: loaded, never stored or summed
    }
    int64_t row[NE];
    Vec<VW> prev[NE], own[NE], acc[NE], with[NE];
    int32_t c[NE][W];
    double v[NE][W];
#pragma unroll
    for (int r = 0; r < NE; ++r) {
      row[r] = e[r] >> LOG2T;
      prev[r] = load_stream<VW>(a.phi_io + e[r] * VW);
      own[r] = load_gather<VW>(a.phi_cur + e[r] * VW);
      if (kDotL) with[r] = load_stream<VW>(a.dot_with + e[r] * VW);
#pragma unroll
      for (int k = 0; k < W; ++k) {
        const bool ok = k < width;
        // the H stream is read once: keep it out of L1, which the gathers use
        c[r][k] = ok ? ld_stream_i32(a.cols + (size_t)k * n + row[r]) : (int32_t)row[r];
        v[r][k] = ok ? ld_stream_f64(a.vals + (size_t)k * n + row[r]) : 0.0;
      }
    }
    Vec<VW> x[NE][W];
#pragma unroll
    for (int r = 0; r < NE; ++r) {
      const double* xt = a.phi_cur + (e[r] - row[r] * T) * VW;
#pragma unroll
      for (int k = 0; k < W; ++k) x[r][k] = load_gather<VW>(xt + (int64_t)c[r][k] * T * VW);
    }
#pragma unroll
    for (int r = 0; r < NE; ++r) {
#pragma unroll
      for (int q = 0; q < VW; ++q) acc[r].v[q] = 0.0;
#pragma unroll
      for (int k = 0; k < W; ++k)
#pragma unroll
        for (int q = 0; q < VW; ++q) acc[r].v[q] = fma(v[r][k], x[r][k].v[q], acc[r].v[q]);
      if (kDiag) {
        const double d = __ldg(a.diag + row[r]);
#pragma unroll
        for (int q = 0; q < VW; ++q) acc[r].v[q] = fma(d, own[r].v[q], acc[r].v[q]);
      }
      if (live[r]) {
        Vec<VW> y;
#pragma unroll
        for (int q = 0; q < VW; ++q) {
          y.v[q] = (acc[r].v[q] - b * own[r].v[q]) * scale - prev[r].v[q];
          s1 = fma(own[r].v[q], kDotL ? with[r].v[q] : own[r].v[q], s1);
          s2 = fma(y.v[q], kDotL ? with[r].v[q] : own[r].v[q], s2);
        }
        store_stream<VW>(a.phi_io + e[r] * VW, y);
      }
    }
  }
  __shared__ double red[kBlock / 32][2];
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
    for (int w = 1; w < kBlock / 32; ++w) {
      s1 += red[w][0];
      s2 += red[w][1];
    }
    a.partial[blockIdx.x] = make_double2(s1, s2);
  }
}

template <int LOG2T, int W, bool DOT>
StepFn pick_x2(bool diag) {
  return diag ? cheb_step_x2_kernel<LOG2T, true, W, DOT> : cheb_step_x2_kernel<LOG2T, false, W, DOT>;
}
template <int LOG2T>
StepFn pick_x2(bool diag, int width, bool dot) {
  if (width <= 3) return dot ? pick_x2<LOG2T, 3, true>(diag) : pick_x2<LOG2T, 3, false>(diag);
  return dot ? pick_x2<LOG2T, 4, true>(diag) : pick_x2<LOG2T, 4, false>(diag);
}

// ---- K7t: the same pass with the Hamiltonian stream staged by TMA ------------------------------
// With wide rows (K ~ 10-20) the register path above is latency-bound: every gather waits for a
// column index that itself comes from HBM.  Here one lane-parallel producer (warp 0) copies the
// next tiles' ELL slots (cols, vals, diag) into a ring of shared-memory stages with
// cp.async.bulk (TMA, completion on an mbarrier) and bulk-prefetches the tiles' phi_{n-1}/phi_n
// lines into L2, so the consumers' dependent chain is  LDS column -> gather  only.
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        " selp.u32 %0, 1, 0, p;\n}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
  } while (!ok);
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
      "l"(src), "r"(bytes), "r"(bar)
      : "memory");
}
__device__ __forceinline__ void bulk_prefetch_l2(const void* src, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}

constexpr int kBarBytes = 128;  // mbarrier ring at the start of dynamic shared memory

// stage layout (TR rows): vals [width][TR] f64 | diag [TR] f64 | cols [width][TR] i32
__host__ __device__ inline uint32_t tile_stage_bytes(int width, int TR, bool diag) {
  return (uint32_t)((width * TR * 12 + (diag ? TR * 8 : 0) + 127) / 128 * 128);
}

#ifndef GTB_TILE_BLOCK
#define GTB_TILE_BLOCK 256
#endif
constexpr int kTileBlock = GTB_TILE_BLOCK;  // threads per CTA of K7t

template <int LOG2T, bool kFirst, bool kDiag, int CH, bool kDotL>
__global__ void __launch_bounds__(kTileBlock) cheb_tile_kernel(const StepArgs a, const int nstages) {
  constexpr int VW = 4;
  constexpr int T = 1 << LOG2T;
  constexpr int TR = kTileBlock / T;  // rows per tile: one thread per 256-bit element
  extern __shared__ __align__(128) unsigned char smem[];
  const int64_t n = a.n;
  const int width = a.width;
  const double scale = a.scale, b = a.b;
  const uint32_t stage_bytes = tile_stage_bytes(width, TR, kDiag);
  const uint32_t vals_off = 0, diag_off = (uint32_t)width * TR * 8;
  const uint32_t cols_off = diag_off + (kDiag ? TR * 8 : 0);
  const uint32_t bar0 = smem_u32(smem);
  unsigned char* const stage0 = smem + kBarBytes;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int64_t n_tiles = (n + TR - 1) / TR;
  const int64_t my_tiles = blockIdx.x < n_tiles ? (n_tiles - 1 - blockIdx.x) / gridDim.x + 1 : 0;

  if (tid == 0) {
    for (int s = 0; s < nstages; ++s) mbar_init(bar0 + 8 * s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // producer: executed by all lanes of warp 0
  auto issue = [&](int64_t i) {
    const int s = (int)(i % nstages);
    const int64_t row0 = (blockIdx.x + i * gridDim.x) * TR;
    const uint32_t rows = (uint32_t)min((int64_t)TR, n - row0);
    const uint32_t bar = bar0 + 8 * s;
    const uint32_t base = smem_u32(stage0 + (size_t)s * stage_bytes);
    if (lane == 0) mbar_expect_tx(bar, rows * (uint32_t)(width * 12 + (kDiag ? 8 : 0)));
    __syncwarp();
    for (int j = lane; j < 2 * width + (kDotL ? 4 : 3); j += 32) {
      if (j < width) {
        bulk_g2s(base + cols_off + (uint32_t)j * TR * 4, a.cols + (size_t)j * n + row0, rows * 4, bar);
      } else if (j < 2 * width) {
        const int k = j - width;
        bulk_g2s(base + vals_off + (uint32_t)k * TR * 8, a.vals + (size_t)k * n + row0, rows * 8, bar);
      } else if (j == 2 * width) {
        if (kDiag) bulk_g2s(base + diag_off, a.diag + row0, rows * 8, bar);
      } else if (j == 2 * width + 1) {
        bulk_prefetch_l2(a.phi_cur + row0 * (T * VW), rows * (T * VW * 8));
      } else if (j == 2 * width + 2) {
        if (!kFirst) bulk_prefetch_l2(a.phi_io + row0 * (T * VW), rows * (T * VW * 8));
      } else {
        if (kDotL) bulk_prefetch_l2(a.dot_with + row0 * (T * VW), rows * (T * VW * 8));
      }
    }
  };
  if (wid == 0)
    for (int64_t i = 0; i < min((int64_t)nstages, my_tiles); ++i) issue(i);

  double s1 = 0.0, s2 = 0.0;
  const int rl = tid >> LOG2T;             // row within the tile
  const int t = tid & (T - 1);             // 256-bit element within the row
  const double* xt = a.phi_cur + t * VW;
  for (int64_t i = 0; i < my_tiles; ++i) {
    const int s = (int)(i % nstages);
    const int64_t row = (blockIdx.x + i * gridDim.x) * TR + rl;
    const bool live = row < n;
    const int64_t e = row * T + t;
    Vec<VW> prev, own, acc, with;
#pragma unroll
    for (int q = 0; q < VW; ++q) acc.v[q] = prev.v[q] = own.v[q] = with.v[q] = 0.0;
    if (live) {
      if (!kFirst) prev = load_stream<VW>(a.phi_io + e * VW);
      own = load_gather<VW>(a.phi_cur + e * VW);
    }
    mbar_wait(bar0 + 8 * s, (uint32_t)((i / nstages) & 1));
    const unsigned char* st = stage0 + (size_t)s * stage_bytes;
    const int32_t* sc = reinterpret_cast<const int32_t*>(st + cols_off) + rl;
    const double* sv = reinterpret_cast<const double*>(st + vals_off) + rl;
    if (live) {
      for (int k0 = 0; k0 < width; k0 += CH) {
        int32_t c[CH];
        double v[CH];
#pragma unroll
        for (int j = 0; j < CH; ++j) {
          const bool ok = k0 + j < width;
          c[j] = ok ? sc[(k0 + j) * TR] : (int32_t)row;
          v[j] = ok ? sv[(k0 + j) * TR] : 0.0;
        }
        Vec<VW> x[CH];
#pragma unroll
        for (int j = 0; j < CH; ++j) x[j] = load_gather<VW>(xt + (int64_t)c[j] * (T * VW));
#pragma unroll
        for (int j = 0; j < CH; ++j)
#pragma unroll
          for (int q = 0; q < VW; ++q) acc.v[q] = fma(v[j], x[j].v[q], acc.v[q]);
      }
      if (kDiag) {
        const double d = reinterpret_cast<const double*>(st + diag_off)[rl];
#pragma unroll
        for (int q = 0; q < VW; ++q) acc.v[q] = fma(d, own.v[q], acc.v[q]);
      }
    }
    __syncthreads();  // every thread has read stage s: hand it back to the producer
    if (wid == 0 && i + nstages < my_tiles) issue(i + nstages);
    if (live) {
      if (kDotL) with = load_stream<VW>(a.dot_with + e * VW);  // prefetched into L2 by the producer
      Vec<VW> y;
#pragma unroll
      for (int q = 0; q < VW; ++q) {
        y.v[q] = (acc.v[q] - b * own.v[q]) * scale;
        if (!kFirst) y.v[q] -= prev.v[q];
        s1 = fma(own.v[q], kDotL ? with.v[q] : own.v[q], s1);
        s2 = fma(y.v[q], kDotL ? with.v[q] : own.v[q], s2);
      }
      store_stream<VW>(a.phi_io + e * VW, y);
    }
  }
  __shared__ double red[kTileBlock / 32][2];
  s1 = warp_sum(s1);
  s2 = warp_sum(s2);
  if (lane == 0) {
    red[wid][0] = s1;
    red[wid][1] = s2;
  }
  __syncthreads();
  if (tid == 0) {
#pragma unroll
    for (int w = 1; w < kTileBlock / 32; ++w) {
      s1 += red[w][0];
      s2 += red[w][1];
    }
    a.partial[blockIdx.x] = make_double2(s1, s2);
  }
}

// ---- K7p: all passes of a small system in ONE cooperative launch ----------------------------------
// Config 1 (2 304 atoms) is 128 passes of ~0.5 MB each: as separate launches it runs at the launch
// cadence (4-5 us per pass), not at any memory roof.  When every element of phi has its own resident
// thread (n * T <= SMs x occupancy x 256), one cooperative kernel runs the first pass and all S - 1
// recursion passes with a grid-wide barrier between them; phi never leaves L2.  Gathers bypass L1
// (ld.global.cg): the vectors are rewritten by other SMs between passes.  Same arithmetic order per
// element and the same per-(pass, block) partial sums as K6/K7.
__device__ __forceinline__ Vec<4> load_l2(const double* p) {
  Vec<4> r;
  asm volatile("ld.global.cg.v4.f64 {%0,%1,%2,%3}, [%4];"
               : "=d"(r.v[0]), "=d"(r.v[1]), "=d"(r.v[2]), "=d"(r.v[3])
               : "l"(p)
               : "memory");
  return r;
}

template <int LOG2T, bool kDiag>
__global__ void __launch_bounds__(kBlock) cheb_small_kernel(const StepArgs a, const int S,
                                                            const double inv_a) {
  constexpr int VW = 4;
  constexpr int T = 1 << LOG2T;
  cooperative_groups::grid_group grid = cooperative_groups::this_grid();
  const int64_t n = a.n;
  const int64_t total = n * T;
  const int width = a.width;
  const double b = a.b;
  const int64_t e = (int64_t)blockIdx.x * kBlock + threadIdx.x;   // one element per thread
  const bool live = e < total;
  const int64_t row = live ? (e >> LOG2T) : 0;
  const int64_t t = e - row * T;
  const double* cur = a.phi_cur;
  double* io = a.phi_io;
  __shared__ double red[kBlock / 32][2];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int k = 0; k < S; ++k) {
    const double scale = k == 0 ? inv_a : 2.0 * inv_a;
    double s1 = 0.0, s2 = 0.0;
    if (live) {
      const double* xt = cur + t * VW;
      Vec<VW> acc, prev;
#pragma unroll
      for (int q = 0; q < VW; ++q) acc.v[q] = prev.v[q] = 0.0;
      if (k > 0) prev = load_l2(io + e * VW);
      const Vec<VW> own = load_l2(cur + e * VW);
#pragma unroll 4
      for (int s = 0; s < width; ++s) {
        const int64_t c = __ldg(a.cols + (size_t)s * n + row);
        const double v = __ldg(a.vals + (size_t)s * n + row);
        const Vec<VW> x = load_l2(xt + c * T * VW);
#pragma unroll
        for (int q = 0; q < VW; ++q) acc.v[q] = fma(v, x.v[q], acc.v[q]);
      }
      if (kDiag) {
        const double d = __ldg(a.diag + row);
#pragma unroll
        for (int q = 0; q < VW; ++q) acc.v[q] = fma(d, own.v[q], acc.v[q]);
      }
      Vec<VW> y;
#pragma unroll
      for (int q = 0; q < VW; ++q) {
        y.v[q] = (acc.v[q] - b * own.v[q]) * scale;
        if (k > 0) y.v[q] -= prev.v[q];
        s1 = fma(own.v[q], own.v[q], s1);
        s2 = fma(y.v[q], own.v[q], s2);
      }
      store_stream<VW>(io + e * VW, y);
    }
    s1 = warp_sum(s1);
    s2 = warp_sum(s2);
    if (lane == 0) {
      red[wid][0] = s1;
      red[wid][1] = s2;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
      for (int w = 1; w < kBlock / 32; ++w) {
        s1 += red[w][0];
        s2 += red[w][1];
      }
      a.partial[(size_t)k * kMaxGrid + blockIdx.x] = make_double2(s1, s2);
    }
    grid.sync();  // every phi_{k+1} element is written and visible before anyone gathers it
    const double* tmp = cur;
    cur = io;
    io = const_cast<double*>(tmp);
  }
}

// ---- K7b: the fused pass on an orbital-blocked matrix (4 orbitals per atom) --------------------
// gtb_sk_hamiltonian's scalar ELL is block-structured: rows 4i..4i+3 (atom i) hold, in slots
// 4k..4k+3, the 4x4 block of the pair (i, j_k), column 4 j_k + nu in slot 4k + nu; for fixed nu the
// four entries mu = 0..3 are contiguous (32 bytes).  The scalar kernels ignore that: each orbital
// row gathers the neighbour's four orbitals again (16 gathers per block) and reads 16 column
// indices.  Here one thread owns (atom i, one 256-bit element of the R vectors) for all four
// orbitals: per neighbour it reads ONE column index, the block as four 256-bit loads and the
// neighbour's four orbital elements as four gathers, and does the 4x4xVW FMAs in registers:
// a quarter of the L1 wavefronts and 144 instead of 192 bytes of H per block from HBM.
// Same arithmetic per element as K7 (slot order, then diagonal), so the vectors agree bit for bit.
template <int LOG2T, bool kFirst, bool kDiag, bool kDotL>
__global__ void __launch_bounds__(kBlock, 2) cheb_orb4_kernel(const StepArgs a) {
  constexpr int VW = 4;
  constexpr int T = 1 << LOG2T;
  const int64_t N = a.n;             // orbital rows
  const int64_t n_atoms = N >> 2;
  const int K = a.width >> 2;        // neighbour slots per atom
  const int64_t total = n_atoms * T;
  const double scale = a.scale, b = a.b;
  constexpr int64_t kOrb = (int64_t)T * VW;  // doubles per orbital row of phi
  double s1 = 0.0, s2 = 0.0;
  for (int64_t e = (int64_t)blockIdx.x * kBlock + threadIdx.x; e < total;
       e += (int64_t)gridDim.x * kBlock) {
    const int64_t i = e >> LOG2T;
    const int64_t t = e - i * T;
    const double* xt = a.phi_cur + t * VW;
    const int32_t* cp = a.cols + 4 * i;
    const double* vp = a.vals + 4 * i;
    Vec<VW> acc[4];
#pragma unroll
    for (int mu = 0; mu < 4; ++mu)
#pragma unroll
      for (int q = 0; q < VW; ++q) acc[mu].v[q] = 0.0;
    int64_t j = K > 0 ? (int64_t)(__ldg(cp) >> 2) : 0;
    for (int k = 0; k < K; ++k) {
      const int64_t jn = k + 1 < K ? (int64_t)(__ldg(cp + (size_t)(4 * (k + 1)) * N) >> 2) : 0;
      Vec<VW> B[4], x[4];
#pragma unroll
      for (int nu = 0; nu < 4; ++nu) B[nu] = load_stream<VW>(vp + (size_t)(4 * k + nu) * N);
#pragma unroll
      for (int nu = 0; nu < 4; ++nu) x[nu] = load_gather<VW>(xt + (4 * j + nu) * kOrb);
#pragma unroll
      for (int nu = 0; nu < 4; ++nu)   // slot order 4k + nu, as the scalar kernels
#pragma unroll
        for (int mu = 0; mu < 4; ++mu)
#pragma unroll
          for (int q = 0; q < VW; ++q) acc[mu].v[q] = fma(B[nu].v[mu], x[nu].v[q], acc[mu].v[q]);
      j = jn;
    }
    Vec<VW> dg;
    if (kDiag) dg = load_stream<VW>(a.diag + 4 * i);
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
      const int64_t at = (4 * i + mu) * kOrb + t * VW;
      const Vec<VW> own = load_gather<VW>(a.phi_cur + at);
      Vec<VW> prev, with;
      if (!kFirst) prev = load_stream<VW>(a.phi_io + at);
      if (kDotL) with = load_stream<VW>(a.dot_with + at);
      Vec<VW> y;
#pragma unroll
      for (int q = 0; q < VW; ++q) {
        double h = acc[mu].v[q];
        if (kDiag) h = fma(dg.v[mu], own.v[q], h);
        y.v[q] = (h - b * own.v[q]) * scale;
        if (!kFirst) y.v[q] -= prev.v[q];
        s1 = fma(own.v[q], kDotL ? with.v[q] : own.v[q], s1);
        s2 = fma(y.v[q], kDotL ? with.v[q] : own.v[q], s2);
      }
      store_stream<VW>(a.phi_io + at, y);
    }
  }
  __shared__ double red[kBlock / 32][2];
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
    for (int w = 1; w < kBlock / 32; ++w) {
      s1 += red[w][0];
      s2 += red[w][1];
    }
    a.partial[blockIdx.x] = make_double2(s1, s2);
  }
}

// ---- K7g: the fused pass on row groups (4 consecutive rows share their gathered neighbours) ----------
// With wide rows K7t sits on the L1 data pipe: one wavefront per (row, neighbour) gather.  Consecutive rows
// of a lattice share most of their neighbours (the 4 atoms of a graphene cell within 4.0 A: 33 distinct
// neighbours instead of 4 x 18), so the matrix is regrouped once (gtb_group_rows): for rows 4g..4g+3 the
// sorted UNION of their column lists, and per union column the 4 hoppings (zero where a row lacks it) as one
// 32-byte vector: cols [U][n/4], vals [U][n/4][4].  One thread owns (group, one 256-bit element of the R
// vectors): per union column one index, one 256-bit load of the 4 hoppings, ONE gather, 4 x VW FMAs.
// Gathers per row drop from K to U/4 (8.25 at config 2) at the price of ~25 % more matrix bytes.  Per row
// the slot order of the sum is the union's (ascending column), which is the ELL's own order with exact
// zeros skipped in between: the vectors agree with K7 bit for bit except for the sign of zero.
template <int LOG2T, bool kFirst, bool kDiag, bool kDotL>
__global__ void __launch_bounds__(kBlock) cheb_grp4_kernel(const StepArgs a) {
  constexpr int VW = 4;
  constexpr int T = 1 << LOG2T;
  const int64_t ng = a.n >> 2;
  const int U = a.width;
  const int64_t total = ng * T;
  const double scale = a.scale, b = a.b;
  constexpr int64_t kRow = (int64_t)T * VW;  // doubles per row of phi
  double s1 = 0.0, s2 = 0.0;
  for (int64_t e = (int64_t)blockIdx.x * kBlock + threadIdx.x; e < total;
       e += (int64_t)gridDim.x * kBlock) {
    const int64_t g = e >> LOG2T;
    const int64_t t = e - g * T;
    const double* xt = a.phi_cur + t * VW;
    const int32_t* cp = a.cols + g;
    const double* vp = a.vals + 4 * g;
    Vec<VW> acc[4];
#pragma unroll
    for (int mu = 0; mu < 4; ++mu)
#pragma unroll
      for (int q = 0; q < VW; ++q) acc[mu].v[q] = 0.0;
    // CH union columns at a time: all CH indices are loaded before the CH gathers that depend on them
    constexpr int CH = 8;
    for (int u0 = 0; u0 < U; u0 += CH) {
      int32_t c[CH];
#pragma unroll
      for (int j = 0; j < CH; ++j) c[j] = u0 + j < U ? __ldg(cp + (size_t)(u0 + j) * ng) : (int32_t)(4 * g);
      Vec<VW> x[CH];
#pragma unroll
      for (int j = 0; j < CH; ++j) x[j] = load_gather<VW>(xt + (int64_t)c[j] * kRow);
#pragma unroll
      for (int j = 0; j < CH; ++j) {
        if (u0 + j < U) {
          const Vec<VW> h = load_stream<VW>(vp + (size_t)(u0 + j) * ng * 4);
#pragma unroll
          for (int mu = 0; mu < 4; ++mu)
#pragma unroll
            for (int q = 0; q < VW; ++q) acc[mu].v[q] = fma(h.v[mu], x[j].v[q], acc[mu].v[q]);
        }
      }
    }
    Vec<VW> dg;
    if (kDiag) dg = load_stream<VW>(a.diag + 4 * g);
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
      const int64_t at = (4 * g + mu) * kRow + t * VW;
      const Vec<VW> own = load_gather<VW>(a.phi_cur + at);
      Vec<VW> prev, with;
      if (!kFirst) prev = load_stream<VW>(a.phi_io + at);
      if (kDotL) with = load_stream<VW>(a.dot_with + at);
      Vec<VW> y;
#pragma unroll
      for (int q = 0; q < VW; ++q) {
        double hh = acc[mu].v[q];
        if (kDiag) hh = fma(dg.v[mu], own.v[q], hh);
        y.v[q] = (hh - b * own.v[q]) * scale;
        if (!kFirst) y.v[q] -= prev.v[q];
        s1 = fma(own.v[q], kDotL ? with.v[q] : own.v[q], s1);
        s2 = fma(y.v[q], kDotL ? with.v[q] : own.v[q], s2);
      }
      store_stream<VW>(a.phi_io + at, y);
    }
  }
  __shared__ double red[kBlock / 32][2];
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
    for (int w = 1; w < kBlock / 32; ++w) {
      s1 += red[w][0];
      s2 += red[w][1];
    }
    a.partial[blockIdx.x] = make_double2(s1, s2);
  }
}

// ---- K7gt: K7g with the grouped slots staged by TMA -------------------------------------------------
// K7g alone is latency-bound (column index -> gather, hoppings from HBM).  Here the union columns and the
// hopping vectors of a tile of TG groups arrive in a shared-memory ring by cp.async.bulk (one copy per union
// slot and array), exactly as K7t stages the ELL slots; a stage is U x TG x 36 bytes (76 KB at U = 33,
// TG = 64), so one CTA per SM with two stages and up to 255 registers per thread: the 4 rows' phi_{n-1} and
// phi_n elements are loaded before the wait and the gathers are issued CH at a time from shared indices.
template <int LOG2T, int NT, bool kFirst, bool kDiag, bool kDotL>
__global__ void __launch_bounds__(NT, 1) cheb_grp4_tile_kernel(const StepArgs a, const int nstages) {
  constexpr int VW = 4;
  constexpr int T = 1 << LOG2T;
  constexpr int TG = NT / T;                 // groups per tile
#ifndef GTB_GRP_CH
#define GTB_GRP_CH 11
#endif
  constexpr int CH = GTB_GRP_CH;
  extern __shared__ __align__(128) unsigned char smem[];
  const int64_t ng = a.n >> 2;
  const int U = a.width;
  const double scale = a.scale, b = a.b;
  const uint32_t vals_bytes = (uint32_t)U * TG * 32;
  const uint32_t stage_bytes = vals_bytes + (uint32_t)U * TG * 4;
  const uint32_t bar0 = smem_u32(smem);
  unsigned char* const stage0 = smem + kBarBytes;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int64_t n_tiles = (ng + TG - 1) / TG;
  const int64_t my_tiles = blockIdx.x < n_tiles ? (n_tiles - 1 - blockIdx.x) / gridDim.x + 1 : 0;
  constexpr int64_t kRow = (int64_t)T * VW;
  if (tid == 0) {
    for (int s = 0; s < nstages; ++s) mbar_init(bar0 + 8 * s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  auto issue = [&](int64_t i) {
    const int s = (int)(i % nstages);
    const int64_t g0 = (blockIdx.x + i * gridDim.x) * TG;
    const uint32_t groups = (uint32_t)min((int64_t)TG, ng - g0);
    const uint32_t bar = bar0 + 8 * s;
    const uint32_t base = smem_u32(stage0 + (size_t)s * stage_bytes);
    if (lane == 0) mbar_expect_tx(bar, groups * (uint32_t)U * 36);
    __syncwarp();
    for (int j = lane; j < 2 * U + 3; j += 32) {
      if (j < U) {
        bulk_g2s(base + (uint32_t)j * TG * 32, a.vals + ((size_t)j * ng + g0) * 4, groups * 32, bar);
      } else if (j < 2 * U) {
        const int u = j - U;
        bulk_g2s(base + vals_bytes + (uint32_t)u * TG * 4, a.cols + (size_t)u * ng + g0, groups * 4, bar);
      } else if (j == 2 * U) {
        bulk_prefetch_l2(a.phi_cur + 4 * g0 * kRow, groups * 4 * (uint32_t)(kRow * 8));
      } else if (j == 2 * U + 1) {
        if (!kFirst) bulk_prefetch_l2(a.phi_io + 4 * g0 * kRow, groups * 4 * (uint32_t)(kRow * 8));
      } else {
        if (kDotL) bulk_prefetch_l2(a.dot_with + 4 * g0 * kRow, groups * 4 * (uint32_t)(kRow * 8));
      }
    }
  };
  if (wid == 0)
    for (int64_t i = 0; i < min((int64_t)nstages, my_tiles); ++i) issue(i);
  double s1 = 0.0, s2 = 0.0;
  const int gl = tid >> LOG2T;
  const int t = tid & (T - 1);
  const double* xt = a.phi_cur + t * VW;
  for (int64_t i = 0; i < my_tiles; ++i) {
    const int s = (int)(i % nstages);
    const int64_t g = (blockIdx.x + i * gridDim.x) * TG + gl;
    const bool live = g < ng;
    Vec<VW> own[4], prev[4], acc[4];
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
#pragma unroll
      for (int q = 0; q < VW; ++q) acc[mu].v[q] = own[mu].v[q] = prev[mu].v[q] = 0.0;
      if (live) {
        const int64_t at = (4 * g + mu) * kRow + t * VW;
        own[mu] = load_gather<VW>(a.phi_cur + at);
        if (!kFirst) prev[mu] = load_stream<VW>(a.phi_io + at);
      }
    }
    mbar_wait(bar0 + 8 * s, (uint32_t)((i / nstages) & 1));
    const unsigned char* st = stage0 + (size_t)s * stage_bytes;
    const double* sv = reinterpret_cast<const double*>(st) + gl * 4;
    const int32_t* sc = reinterpret_cast<const int32_t*>(st + vals_bytes) + gl;
    if (live) {
      for (int u0 = 0; u0 < U; u0 += CH) {
        int32_t c[CH];
#pragma unroll
        for (int j = 0; j < CH; ++j) c[j] = u0 + j < U ? sc[(u0 + j) * TG] : (int32_t)(4 * g);
        Vec<VW> x[CH];
#pragma unroll
        for (int j = 0; j < CH; ++j) x[j] = load_gather<VW>(xt + (int64_t)c[j] * kRow);
#pragma unroll
        for (int j = 0; j < CH; ++j) {
          if (u0 + j < U) {
            const double* h = sv + (size_t)(u0 + j) * TG * 4;
#pragma unroll
            for (int mu = 0; mu < 4; ++mu) {
              const double hm = h[mu];
#pragma unroll
              for (int q = 0; q < VW; ++q) acc[mu].v[q] = fma(hm, x[j].v[q], acc[mu].v[q]);
            }
          }
        }
      }
    }
    __syncthreads();  // every thread has read stage s
    if (wid == 0 && i + nstages < my_tiles) issue(i + nstages);
    if (live) {
      Vec<VW> dg;
      if (kDiag) dg = load_stream<VW>(a.diag + 4 * g);
#pragma unroll
      for (int mu = 0; mu < 4; ++mu) {
        const int64_t at = (4 * g + mu) * kRow + t * VW;
        Vec<VW> with;
        if (kDotL) with = load_stream<VW>(a.dot_with + at);
        Vec<VW> y;
#pragma unroll
        for (int q = 0; q < VW; ++q) {
          double hh = acc[mu].v[q];
          if (kDiag) hh = fma(dg.v[mu], own[mu].v[q], hh);
          y.v[q] = (hh - b * own[mu].v[q]) * scale;
          if (!kFirst) y.v[q] -= prev[mu].v[q];
          s1 = fma(own[mu].v[q], kDotL ? with.v[q] : own[mu].v[q], s1);
          s2 = fma(y.v[q], kDotL ? with.v[q] : own[mu].v[q], s2);
        }
        store_stream<VW>(a.phi_io + at, y);
      }
    }
  }
  __shared__ double red[NT / 32][2];
  s1 = warp_sum(s1);
  s2 = warp_sum(s2);
  if (lane == 0) {
    red[wid][0] = s1;
    red[wid][1] = s2;
  }
  __syncthreads();
  if (tid == 0) {
#pragma unroll
    for (int w = 1; w < NT / 32; ++w) {
      s1 += red[w][0];
      s2 += red[w][1];
    }
    a.partial[blockIdx.x] = make_double2(s1, s2);
  }
}

// regrouping: one thread per group merges the 4 sorted column lists (padding = own row index, skipped).
// kFill = false: *width_out = max union size;  kFill = true: writes cols/vals (width U given).
template <bool kFill>
__global__ void __launch_bounds__(kBlock) group_rows_kernel(const int32_t* __restrict__ cols,
                                                            const double* __restrict__ vals, int64_t n,
                                                            int32_t K, int32_t U, int32_t* __restrict__ gcols,
                                                            double* __restrict__ gvals,
                                                            int32_t* __restrict__ width_out) {
  const int64_t ng = n >> 2;
  int worst = 0;
  for (int64_t g = (int64_t)blockIdx.x * kBlock + threadIdx.x; g < ng; g += (int64_t)gridDim.x * kBlock) {
    int pos[4] = {0, 0, 0, 0};
    int u = 0;
    for (;;) {
      int64_t best = INT64_MAX;
      int64_t cur[4];
#pragma unroll
      for (int mu = 0; mu < 4; ++mu) {
        const int64_t row = 4 * g + mu;
        while (pos[mu] < K && cols[(size_t)pos[mu] * n + row] == row) ++pos[mu];  // padding slots
        cur[mu] = pos[mu] < K ? (int64_t)cols[(size_t)pos[mu] * n + row] : INT64_MAX;
        best = min(best, cur[mu]);
      }
      if (best == INT64_MAX) break;
      if (kFill && u < U) {
        gcols[(size_t)u * ng + g] = (int32_t)best;
#pragma unroll
        for (int mu = 0; mu < 4; ++mu)
          gvals[((size_t)u * ng + g) * 4 + mu] =
              cur[mu] == best ? vals[(size_t)pos[mu] * n + 4 * g + mu] : 0.0;
      }
#pragma unroll
      for (int mu = 0; mu < 4; ++mu)
        if (cur[mu] == best) ++pos[mu];
      ++u;
    }
    if (kFill) {
      for (; u < U; ++u) {  // padding: the group's first row, zeros
        gcols[(size_t)u * ng + g] = (int32_t)(4 * g);
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) gvals[((size_t)u * ng + g) * 4 + mu] = 0.0;
      }
    }
    worst = max(worst, u);
  }
  if (!kFill) {
    worst = warp_max_i(worst);
    if ((threadIdx.x & 31) == 0 && worst > 0) atomicMax(width_out, worst);
  } else if (worst > U) {
    atomicMax(width_out, worst);  // overflow: reported by the host wrapper
  }
}

// ---- K7b9: the blocked pass for 9 orbitals per atom (s, p, d) ---------------------------------------
// Same idea as K7b with the block streamed one column at a time: per neighbour one column index, then
// for each of the 9 neighbour orbitals nu one gather of its 256-bit element and the 9 block entries
// E[mu][nu], 36 FMAs; the 9 x VW accumulators stay in registers.  The block columns of a warp's atoms
// are one contiguous run (72 bytes per atom, atoms consecutive): the warp reads the run with coalesced
// 64-bit loads one column ahead, parks it in its own slice of shared memory and every lane picks its
// atom's 9 entries from there (conflict-free: stride 18 words) -- 72-byte-strided loads straight from
// global memory cost 9 times the L1 wavefronts.
template <int LOG2T, bool kFirst, bool kDiag, bool kDotL, bool kStage>
__global__ void __launch_bounds__(kBlock, 2) cheb_orb9_kernel(const StepArgs a) {
  constexpr int VW = 4;
  constexpr int T = 1 << LOG2T;
  constexpr int B = 9;
  constexpr int A = 32 / T;                 // atoms per warp
  constexpr int NL = (B * A + 31) / 32;     // coalesced loads per lane per block column
  __shared__ double s_col[kBlock / 32][kStage ? B * A : 1];
  const int64_t N = a.n;
  const int64_t n_atoms = N / B;
  const int K = a.width / B;
  const int64_t total = n_atoms * T;
  const double scale = a.scale, b = a.b;
  constexpr int64_t kOrb = (int64_t)T * VW;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  double* const sm = s_col[wid];
  double s1 = 0.0, s2 = 0.0;
  for (int64_t e0 = (int64_t)blockIdx.x * kBlock + wid * 32; e0 < total; e0 += (int64_t)gridDim.x * kBlock) {
    const int64_t e = e0 + lane;
    const bool live = e < total;
    const int64_t i0 = e0 >> LOG2T;                                    // first atom of the warp
    const int run = B * (int)min((int64_t)A, n_atoms - i0);            // doubles per block column
    const int64_t i = live ? (e >> LOG2T) : i0;
    const int64_t t = e - (e >> LOG2T) * T;
    const int la = (int)(i - i0);
    const double* xt = a.phi_cur + t * VW;
    const int32_t* cp = a.cols + B * i;
    const double* vrun = a.vals + B * i0;
    Vec<VW> acc[B];
#pragma unroll
    for (int mu = 0; mu < B; ++mu)
#pragma unroll
      for (int q = 0; q < VW; ++q) acc[mu].v[q] = 0.0;
    double pre[NL];
    if (kStage) {
#pragma unroll
      for (int q = 0; q < NL; ++q) pre[q] = (K > 0 && lane + 32 * q < run) ? __ldg(vrun + lane + 32 * q) : 0.0;
    }
    int64_t j = K > 0 ? (int64_t)(__ldg(cp) / B) : 0;
    for (int k = 0; k < K; ++k) {
      const int64_t jn = k + 1 < K ? (int64_t)(__ldg(cp + (size_t)(B * (k + 1)) * N) / B) : 0;
#pragma unroll 3
      for (int nu = 0; nu < B; ++nu) {
        if (kStage) {
          __syncwarp();  // the previous column has been read by every lane
#pragma unroll
          for (int q = 0; q < NL; ++q)
            if (lane + 32 * q < B * A) sm[lane + 32 * q] = pre[q];
          __syncwarp();
          const int nxt = B * k + nu + 1;   // next column of this row of blocks, one ahead
          if (nxt < B * K) {
            const double* src = vrun + (size_t)nxt * N;
#pragma unroll
            for (int q = 0; q < NL; ++q) pre[q] = lane + 32 * q < run ? __ldg(src + lane + 32 * q) : 0.0;
          }
        }
        if (live) {
          const Vec<VW> x = load_gather<VW>(xt + (B * j + nu) * kOrb);
          const double* col = a.vals + (size_t)(B * k + nu) * N + B * i;   // direct path (kStage = 0)
#pragma unroll
          for (int mu = 0; mu < B; ++mu) {
            const double h = kStage ? sm[B * la + mu] : __ldg(col + mu);
#pragma unroll
            for (int q = 0; q < VW; ++q) acc[mu].v[q] = fma(h, x.v[q], acc[mu].v[q]);
          }
        }
      }
      j = jn;
    }
    if (live) {
#pragma unroll
      for (int mu = 0; mu < B; ++mu) {
        const int64_t at = (B * i + mu) * kOrb + t * VW;
        const Vec<VW> own = load_gather<VW>(a.phi_cur + at);
        Vec<VW> prev, with;
        if (!kFirst) prev = load_stream<VW>(a.phi_io + at);
        if (kDotL) with = load_stream<VW>(a.dot_with + at);
        const double dg = kDiag ? __ldg(a.diag + B * i + mu) : 0.0;
        Vec<VW> y;
#pragma unroll
        for (int q = 0; q < VW; ++q) {
          double h = acc[mu].v[q];
          if (kDiag) h = fma(dg, own.v[q], h);
          y.v[q] = (h - b * own.v[q]) * scale;
          if (!kFirst) y.v[q] -= prev.v[q];
          s1 = fma(own.v[q], kDotL ? with.v[q] : own.v[q], s1);
          s2 = fma(y.v[q], kDotL ? with.v[q] : own.v[q], s2);
        }
        store_stream<VW>(a.phi_io + at, y);
      }
    }
  }
  __shared__ double red[kBlock / 32][2];
  s1 = warp_sum(s1);
  s2 = warp_sum(s2);
  if (lane == 0) {
    red[wid][0] = s1;
    red[wid][1] = s2;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int w = 1; w < kBlock / 32; ++w) {
      s1 += red[w][0];
      s2 += red[w][1];
    }
    a.partial[blockIdx.x] = make_double2(s1, s2);
  }
}

// ---- K7s: two Chebyshev steps per HBM sweep (temporal blocking through L2) -----------------------
// One pass of K7 moves 12K + 48R bytes per atom through HBM for one step.  Here one launch advances
// every row by TWO steps: rows are cut into chunks of `chunk_rows`; task (j, l) = step l (0 or 1)
// on chunk j, one WARP per task; tasks are ordered by the key j + skew*l and dealt round-robin to
// the resident warps, so step 1 of a chunk runs shortly after step 0 of the chunks around it, while
// their phi_{n+1} (just written), phi_n and H rows are still in the 126 MB L2.  HBM then sees
// 12K + 32R read + 32R written per atom for two steps instead of 2*(12K + 48R)  (ncu: 17.2 GB
// instead of 26.4 GB per two steps at config 5).
// Dependencies: step 1 on chunk j gathers phi_{n+1} from the rows within `halo` (the largest ring
// distance |col - row| of H) of its own, and overwrites the phi_n rows that step 0 of those rows
// gathers; so it waits until step 0 has finished on every 1024-row group that overlaps that range
// (group counters: release increments, acquire polls).  The task order is a topological order of
// that relation (skew > halo in chunks; the first chunks, whose left neighbours wrap around the
// ring, run step 1 last), step-0 tasks never wait, every warp works through its tasks in increasing
// order and all warps are resident (grid = SMs x occupancy): no deadlock.  A spin limit turns any
// violation into an error flag instead of a hang.  Step 1 reads phi_{n+1} with plain loads, not .nc.
constexpr int kGroupRows = 1024;

struct SweepArgs {
  StepArgs s;            // phi_cur = phi_n, phi_io = phi_{n-1}: roles swap for step 1
  int32_t chunk_rows;    // divides kGroupRows, multiple of 32
  int32_t n_chunks;
  const int32_t* halo_rows;  // device: largest ring distance |col - row| of H
  int32_t slack;         // skew = halo chunks + 1 + slack
  int32_t* group_done;   // [ceil(n / kGroupRows)], zeroed before the launch: step-0 chunks finished
  int32_t* error;        // set to 2 when a wait exceeds the spin limit
  double2* partial0;     // [n_chunks] warp sums of step 0
  double2* partial1;     // [n_chunks] warp sums of step 1
};

__device__ __forceinline__ int32_t ld_acquire(const int32_t* p) {
  int32_t v;
  asm volatile("ld.global.acquire.gpu.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ Vec<4> load_coherent(const double* p) {
  Vec<4> r;
  asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];"
               : "=d"(r.v[0]), "=d"(r.v[1]), "=d"(r.v[2]), "=d"(r.v[3])
               : "l"(p)
               : "memory");
  return r;
}

// rows [row0, row1) of one step by one warp; kCoherent: phi_n was written earlier in this launch
template <int LOG2T, bool kDiag, bool kCoherent>
__device__ __forceinline__ void sweep_rows(const StepArgs& a, const double* __restrict__ cur,
                                           double* __restrict__ io, int64_t row0, int64_t row1,
                                           int lane, double& s1, double& s2) {
  constexpr int VW = 4;
  constexpr int T = 1 << LOG2T;
  const int64_t n = a.n;
  const int width = a.width;
  const double scale = a.scale, b = a.b;
  const int64_t e_end = row1 * T;
  for (int64_t e = row0 * T + lane; e < e_end; e += 32) {
    const int64_t row = e >> LOG2T;
    const int64_t t = e - row * T;
    const double* xt = cur + t * VW;
    const int32_t* cp = a.cols + row;
    const double* vp = a.vals + row;
    const Vec<VW> prev = load_stream<VW>(io + e * VW);
    const Vec<VW> own = kCoherent ? load_coherent(cur + e * VW) : load_gather<VW>(cur + e * VW);
    Vec<VW> acc;
#pragma unroll
    for (int q = 0; q < VW; ++q) acc.v[q] = 0.0;
#pragma unroll 4
    for (int k = 0; k < width; ++k) {
      const int64_t c = __ldg(cp + (size_t)k * n);
      const double v = __ldg(vp + (size_t)k * n);
      const Vec<VW> x = kCoherent ? load_coherent(xt + c * T * VW) : load_gather<VW>(xt + c * T * VW);
#pragma unroll
      for (int q = 0; q < VW; ++q) acc.v[q] = fma(v, x.v[q], acc.v[q]);
    }
    if (kDiag) {
      const double d = __ldg(a.diag + row);
#pragma unroll
      for (int q = 0; q < VW; ++q) acc.v[q] = fma(d, own.v[q], acc.v[q]);
    }
    Vec<VW> y;
#pragma unroll
    for (int q = 0; q < VW; ++q) {
      y.v[q] = (acc.v[q] - b * own.v[q]) * scale - prev.v[q];
      s1 = fma(own.v[q], own.v[q], s1);
      s2 = fma(y.v[q], own.v[q], s2);
    }
    store_stream<VW>(io + e * VW, y);
  }
}

constexpr int kSpinLimit = 1 << 21;  // x 200 ns: ~0.4 s

template <int LOG2T, bool kDiag>
__global__ void __launch_bounds__(kBlock, 4) cheb_sweep_kernel(const SweepArgs a) {
  const int64_t n = a.s.n;
  const int nc = a.n_chunks, cr = a.chunk_rows;
  const int lane = threadIdx.x & 31;
  const int64_t halo = *a.halo_rows;
  const int ng = (int)((n + kGroupRows - 1) / kGroupRows);
  const int h = (int)min((int64_t)nc, (halo + cr - 1) / cr);   // halo in chunks
  const bool whole_ring = 2 * (halo + cr) + kGroupRows >= n;   // the wait range covers the ring
  const int seam = whole_ring ? nc : h;                        // chunks whose step 1 runs last
  const int skew = h + 1 + a.slack;
  // task list: keys t = 0 .. nc-1+skew, two slots per key: (j = t, l = 0) and (j = t - skew, l = 1)
  // for j >= seam; then (j, 1) for j = 0 .. seam-1.
  const int64_t main_slots = 2 * ((int64_t)nc + skew);
  const int64_t total = main_slots + seam;
  // an odd number of workers, so that a warp alternates between step-0 and step-1 slots (with an
  // even stride half of the warps would only ever see step-1 slots and wait on the other half)
  const int64_t W = ((int64_t)gridDim.x * (kBlock / 32) - 1) | 1;
  bool abort = false;
  const int64_t me = (int64_t)blockIdx.x * (kBlock / 32) + (threadIdx.x >> 5);
  for (int64_t task = me; task < total && !abort && me < W; task += W) {
    int j, l;
    if (task < main_slots) {
      l = (int)(task & 1);
      j = (int)(task >> 1) - (l ? skew : 0);
      if (j < (l ? seam : 0) || j >= nc) continue;
    } else {
      l = 1;
      j = (int)(task - main_slots);
    }
    const int64_t row0 = (int64_t)j * cr, row1 = min(n, row0 + cr);
    if (l == 1) {  // wait for step 0 on every group overlapping [row0 - halo, row1 + halo) (ring)
      int g0 = 0, cnt = ng;
      if (!whole_ring) {
        const int64_t lo = row0 - halo, hi = row1 + halo - 1;   // may leave [0, n): wraps
        g0 = (int)((lo + n) % n / kGroupRows);
        const int g1 = (int)(hi % n / kGroupRows);
        cnt = g1 >= g0 && hi - lo < n - kGroupRows ? g1 - g0 + 1 : g1 + ng - g0 + 1;
        if (cnt > ng) cnt = ng;
      }
      int spins = 0;
      for (;;) {
        bool ok = true;
        for (int q = lane; q < cnt; q += 32) {
          int g = g0 + q;
          if (g >= ng) g -= ng;
          const int64_t grows = min((int64_t)kGroupRows, n - (int64_t)g * kGroupRows);
          if (ld_acquire(a.group_done + g) < (int)((grows + cr - 1) / cr)) ok = false;
        }
        if (__all_sync(0xffffffffu, ok)) break;
        __nanosleep(200);
        if (++spins > kSpinLimit || ld_acquire(a.error) != 0) {
          if (lane == 0) atomicExch(a.error, 2);
          abort = true;
          break;
        }
      }
      if (abort) break;
    }
    double s1 = 0.0, s2 = 0.0;
    if (l == 0)
      sweep_rows<LOG2T, kDiag, false>(a.s, a.s.phi_cur, a.s.phi_io, row0, row1, lane, s1, s2);
    else
      sweep_rows<LOG2T, kDiag, true>(a.s, a.s.phi_io, const_cast<double*>(a.s.phi_cur), row0, row1,
                                     lane, s1, s2);
    s1 = warp_sum(s1);
    s2 = warp_sum(s2);
    __syncwarp();  // orders the lanes' phi stores before lane 0's fence below
    if (lane == 0) {
      (l ? a.partial1 : a.partial0)[j] = make_double2(s1, s2);
      if (l == 0) {
        __threadfence();  // cumulative: the warp's stores are visible device-wide before the count
        atomicAdd(a.group_done + row0 / kGroupRows, 1);
      }
    }
  }
}

// largest ring distance min(|c - i|, n - |c - i|) over the entries of H -> *out (zeroed before)
__global__ void __launch_bounds__(kBlock) halo_kernel(const int32_t* __restrict__ cols, int64_t n,
                                                      int32_t width, int32_t* out) {
  const int64_t total = n * width;
  int m = 0;
  for (int64_t e = (int64_t)blockIdx.x * kBlock + threadIdx.x; e < total;
       e += (int64_t)gridDim.x * kBlock) {
    const int64_t i = e % n;
    int64_t d = (int64_t)cols[e] - i;
    d = d < 0 ? -d : d;
    d = min(d, n - d);
    m = max(m, (int)d);
  }
  m = warp_max_i(m);
  if ((threadIdx.x & 31) == 0 && m > 0) atomicMax(out, m);
}

// K8s: the chunk sums of one sweep -> sums[0], sums[1], fixed order, two stages
constexpr int kSegs = 64;
__global__ void __launch_bounds__(kBlock) reduce_chunks_kernel(const double2* __restrict__ p0,
                                                               const double2* __restrict__ p1,
                                                               int n_chunks, double2* tmp) {
  const double2* p = blockIdx.y ? p1 : p0;
  const int per = (n_chunks + kSegs - 1) / kSegs;
  const int beg = blockIdx.x * per, end = min(n_chunks, beg + per);
  double s1 = 0.0, s2 = 0.0;
  for (int k = beg + threadIdx.x; k < end; k += kBlock) {
    s1 += p[k].x;
    s2 += p[k].y;
  }
  __shared__ double red[kBlock][2];
  red[threadIdx.x][0] = s1;
  red[threadIdx.x][1] = s2;
  __syncthreads();
  for (int o = kBlock / 2; o > 0; o >>= 1) {
    if (threadIdx.x < o) {
      red[threadIdx.x][0] += red[threadIdx.x + o][0];
      red[threadIdx.x][1] += red[threadIdx.x + o][1];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) tmp[blockIdx.y * kSegs + blockIdx.x] = make_double2(red[0][0], red[0][1]);
}
__global__ void reduce_segs_kernel(const double2* __restrict__ tmp, double2* sums) {
  const double2* t = tmp + threadIdx.x * kSegs;  // thread 0: step 0, thread 1: step 1
  double s1 = 0.0, s2 = 0.0;
  for (int k = 0; k < kSegs; ++k) {
    s1 += t[k].x;
    s2 += t[k].y;
  }
  double2 acc = sums[threadIdx.x];
  acc.x += s1;
  acc.y += s2;
  sums[threadIdx.x] = acc;
}

// K8a: sums[step] += sum over blocks of partial[step][block], in a fixed order
__global__ void __launch_bounds__(128) reduce_partials_kernel(const double2* __restrict__ partial,
                                                              int stride, int grid, double2* sums) {
  const double2* p = partial + (size_t)blockIdx.x * stride;
  double s1 = 0.0, s2 = 0.0;
  for (int k = threadIdx.x; k < grid; k += 128) {
    s1 += p[k].x;
    s2 += p[k].y;
  }
  __shared__ double red[128][2];
  red[threadIdx.x][0] = s1;
  red[threadIdx.x][1] = s2;
  __syncthreads();
  for (int o = 64; o > 0; o >>= 1) {
    if (threadIdx.x < o) {
      red[threadIdx.x][0] += red[threadIdx.x + o][0];
      red[threadIdx.x][1] += red[threadIdx.x + o][1];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    double2 acc = sums[blockIdx.x];
    acc.x += red[0][0];
    acc.y += red[0][1];
    sums[blockIdx.x] = acc;
  }
}

// K8b: doubling identities (reading C5); sums[k] = (sum_r <phi_k|phi_k>, sum_r Re<phi_{k+1}|phi_k>)
__global__ void __launch_bounds__(kBlock) finish_moments_kernel(const double2* __restrict__ sums,
                                                                int32_t M, double norm, double* mu,
                                                                int32_t* status) {
  const int n = blockIdx.x * kBlock + threadIdx.x;
  if (n >= M) return;
  const int k = n >> 1;
  const double2 s0 = sums[0];
  double m;
  if (n == 0) m = s0.x;
  else if (n == 1) m = s0.y;
  else if ((n & 1) == 0) m = 2.0 * sums[k].x - s0.x;
  else m = 2.0 * sums[k].y - s0.y;
  m /= norm;
  mu[n] = m;
  if (!isfinite(m)) atomicOr(status, 1);
}

__global__ void copy_sums_kernel(const double2* sums, double* out2) {
  out2[0] = sums[0].x;
  out2[1] = sums[0].y;
}

// ---- host side ---------------------------------------------------------------------------
template <int VW, int LOG2T, int CH, bool DOT>
void pick_ch(bool diag, StepPlan* p) {
  p->first = diag ? cheb_step_kernel<VW, LOG2T, true, true, CH, DOT> : cheb_step_kernel<VW, LOG2T, true, false, CH, DOT>;
  p->next = diag ? cheb_step_kernel<VW, LOG2T, false, true, CH, DOT> : cheb_step_kernel<VW, LOG2T, false, false, CH, DOT>;
}

template <int VW, int LOG2T>
void pick(bool diag, int ch, bool dot, StepPlan* p) {
  if (ch == 0) { if (dot) pick_ch<VW, LOG2T, 0, true>(diag, p); else pick_ch<VW, LOG2T, 0, false>(diag, p); }
  else { if (dot) pick_ch<VW, LOG2T, 8, true>(diag, p); else pick_ch<VW, LOG2T, 8, false>(diag, p); }
}

template <int LOG2T, int CH, bool DOT>
void pick_tile_ch(bool diag, StepPlan* p) {
  p->tfirst = diag ? cheb_tile_kernel<LOG2T, true, true, CH, DOT> : cheb_tile_kernel<LOG2T, true, false, CH, DOT>;
  p->tnext = diag ? cheb_tile_kernel<LOG2T, false, true, CH, DOT> : cheb_tile_kernel<LOG2T, false, false, CH, DOT>;
}

template <int LOG2T, bool DOT>
void pick_tile_dot(bool diag, int ch, StepPlan* p) {
  switch (ch) {
    case 3: pick_tile_ch<LOG2T, 3, DOT>(diag, p); break;
    case 4: pick_tile_ch<LOG2T, 4, DOT>(diag, p); break;
    case 6: pick_tile_ch<LOG2T, 6, DOT>(diag, p); break;
    case 8: pick_tile_ch<LOG2T, 8, DOT>(diag, p); break;
    default: pick_tile_ch<LOG2T, 10, DOT>(diag, p); break;
  }
}

template <int LOG2T>
void pick_tile(bool diag, int ch, bool dot, StepPlan* p) {
  if (dot) pick_tile_dot<LOG2T, true>(diag, ch, p);
  else pick_tile_dot<LOG2T, false>(diag, ch, p);
}

// gathers kept in flight per thread: the chunk that pads `width` least (ties: the larger)
int tile_chunk(int width) {
  if (width <= 3) return 3;
  if (width <= 4) return 4;
  int best = 10, waste = (width + 9) / 10 * 10 - width;
  for (int ch : {8, 6}) {
    const int w = (width + ch - 1) / ch * ch - width;
    if (w < waste) { best = ch; waste = w; }
  }
  return best;
}

int env_int(const char* name, int dflt) {
  const char* e = getenv(name);
  return e ? atoi(e) : dflt;
}

}  // namespace

template <int LOG2T, bool DOT>
void pick_orb_dot(int B, bool diag, StepPlan* p) {
  if (B == 4) {
    p->first = diag ? cheb_orb4_kernel<LOG2T, true, true, DOT> : cheb_orb4_kernel<LOG2T, true, false, DOT>;
    p->next = diag ? cheb_orb4_kernel<LOG2T, false, true, DOT> : cheb_orb4_kernel<LOG2T, false, false, DOT>;
  } else if (env_int("GTB_K7_ORB9_STAGE", 1)) {  // block columns through shared memory
    p->first = diag ? cheb_orb9_kernel<LOG2T, true, true, DOT, true> : cheb_orb9_kernel<LOG2T, true, false, DOT, true>;
    p->next = diag ? cheb_orb9_kernel<LOG2T, false, true, DOT, true> : cheb_orb9_kernel<LOG2T, false, false, DOT, true>;
  } else {
    p->first = diag ? cheb_orb9_kernel<LOG2T, true, true, DOT, false> : cheb_orb9_kernel<LOG2T, true, false, DOT, false>;
    p->next = diag ? cheb_orb9_kernel<LOG2T, false, true, DOT, false> : cheb_orb9_kernel<LOG2T, false, false, DOT, false>;
  }
}
template <int LOG2T>
void pick_orb(int B, bool diag, bool dot, StepPlan* p) {
  if (dot) pick_orb_dot<LOG2T, true>(B, diag, p);
  else pick_orb_dot<LOG2T, false>(B, diag, p);
}

// K7b plan (B = 4 or 9 orbitals per atom): one thread per (atom, 256-bit element); false when H or R
// does not fit and the scalar kernels must be used
bool make_plan_orb(const gtb_ell* H, int R, int B, bool dot, StepPlan* p) {
  if ((B != 4 && B != 9) || H->n % B || H->width % B || H->width == 0 || (R != 2 && R != 4 && R != 8) ||
      (B == 4 && ((reinterpret_cast<uintptr_t>(H->vals) & 31u) || (reinterpret_cast<uintptr_t>(H->diag) & 31u))))
    return false;
  const bool diag = H->diag != nullptr;
  if (R == 2) { pick_orb<0>(B, diag, dot, p); p->T = 1; }
  else if (R == 4) { pick_orb<1>(B, diag, dot, p); p->T = 2; }
  else { pick_orb<2>(B, diag, dot, p); p->T = 4; }
  p->vw = 4;
  p->stages = 0;
  int dev = 0, sms = kSmCount, per_sm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, p->next, kBlock, 0) != cudaSuccess)
    return false;
  per_sm = std::max(1, std::min(per_sm, kMaxBlocksPerSm));
  const int64_t total = H->n / B * p->T;
  p->grid = (int)std::max<int64_t>(1, std::min<int64_t>((total + kBlock - 1) / kBlock, (int64_t)sms * per_sm));
  return true;
}

template <int LOG2T, bool DOT>
void pick_grp_dot(bool diag, StepPlan* p) {
  p->first = diag ? cheb_grp4_kernel<LOG2T, true, true, DOT> : cheb_grp4_kernel<LOG2T, true, false, DOT>;
  p->next = diag ? cheb_grp4_kernel<LOG2T, false, true, DOT> : cheb_grp4_kernel<LOG2T, false, false, DOT>;
}

// K7g plan: H holds the grouped arrays of gtb_group_rows (cols [U][n/4], vals [U][n/4][4])
bool make_plan_grp4(const gtb_ell* H, int R, bool dot, StepPlan* p) {
  if (H->n % 4 || H->width == 0 || (R != 2 && R != 4 && R != 8) ||
      (reinterpret_cast<uintptr_t>(H->vals) & 31u) || (reinterpret_cast<uintptr_t>(H->diag) & 31u))
    return false;
  const bool diag = H->diag != nullptr;
  if (R == 2) { if (dot) pick_grp_dot<0, true>(diag, p); else pick_grp_dot<0, false>(diag, p); p->T = 1; }
  else if (R == 4) { if (dot) pick_grp_dot<1, true>(diag, p); else pick_grp_dot<1, false>(diag, p); p->T = 2; }
  else { if (dot) pick_grp_dot<2, true>(diag, p); else pick_grp_dot<2, false>(diag, p); p->T = 4; }
  p->vw = 4;
  p->stages = 0;
  p->block = kBlock;
  int dev = 0, sms = kSmCount, per_sm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return false;
  // K7gt: TMA-staged variant for R = 8 (one CTA of 256 threads per SM, 64 groups per tile)
  if (R == 8 && !dot && H->n % 16 == 0 && !(reinterpret_cast<uintptr_t>(H->cols) & 15u) &&
      env_int("GTB_K7_GROUP_TILE", 1) != 0) {
    int max_smem = 0;
    cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    const size_t stage_bytes = (size_t)H->width * 64 * 36;
    int stages = env_int("GTB_K7_STAGES", 2);
    while (stages > 1 && kBarBytes + stages * stage_bytes > (size_t)max_smem) --stages;
    const size_t smem = kBarBytes + stages * stage_bytes;
    if (smem <= (size_t)max_smem) {
      p->tfirst = diag ? cheb_grp4_tile_kernel<2, 256, true, true, false> : cheb_grp4_tile_kernel<2, 256, true, false, false>;
      p->tnext = diag ? cheb_grp4_tile_kernel<2, 256, false, true, false> : cheb_grp4_tile_kernel<2, 256, false, false, false>;
      if (cudaFuncSetAttribute(p->tfirst, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) == cudaSuccess &&
          cudaFuncSetAttribute(p->tnext, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) == cudaSuccess) {
        const int64_t n_tiles = (H->n / 4 + 63) / 64;
        p->grid = (int)std::max<int64_t>(1, std::min<int64_t>(n_tiles, sms));
        p->stages = stages;
        p->smem = smem;
        p->block = 256;
        return true;
      }
    }
  }
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, p->next, kBlock, 0) != cudaSuccess)
    return false;
  per_sm = std::max(1, std::min(per_sm, kMaxBlocksPerSm));
  const int64_t total = H->n / 4 * p->T;
  p->grid = (int)std::max<int64_t>(1, std::min<int64_t>((total + kBlock - 1) / kBlock, (int64_t)sms * per_sm));
  return true;
}

int make_plan(const gtb_ell* H, int R, bool dot, StepPlan* p) {
  const int64_t n = H->n;
  const int width = H->width;
  const bool diag = H->diag != nullptr;
  const int ch = width <= 4 ? 0 : 8;
  int log2t = -1;
  if (R == 2) { pick<4, 0>(diag, ch, dot, p); p->vw = 4; p->T = 1; log2t = 0; }
  else if (R == 4) { pick<4, 1>(diag, ch, dot, p); p->vw = 4; p->T = 2; log2t = 1; }
  else if (R == 8) { pick<4, 2>(diag, ch, dot, p); p->vw = 4; p->T = 4; log2t = 2; }
  else if (R == 1) { pick<2, 0>(diag, ch, dot, p); p->vw = 2; p->T = 1; }
  else { pick<2, -1>(diag, ch, dot, p); p->vw = 2; p->T = R; }
  // K7x2: narrow rows (K <= 4) take the two-elements-in-flight kernel for every pass but the first
  const bool x2 = env_int("GTB_K7_X2", 1) != 0 && log2t >= 0 && width >= 1 && width <= 4;
  if (x2) p->next = log2t == 0 ? pick_x2<0>(diag, width, dot) : log2t == 1 ? pick_x2<1>(diag, width, dot)
                                                                          : pick_x2<2>(diag, width, dot);
  int dev = 0, sms = kSmCount, per_sm = 0;
  GTB_CUDA_TRY(cudaGetDevice(&dev));
  GTB_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  // TMA-staged path: bulk copies need 16-byte aligned sources and sizes in every slot row
  const bool aligned = n % 4 == 0 && width >= 1 &&
                       !(reinterpret_cast<uintptr_t>(H->cols) & 15u) &&
                       !(reinterpret_cast<uintptr_t>(H->vals) & 15u) &&
                       !(reinterpret_cast<uintptr_t>(H->diag) & 15u);
  int stages = env_int("GTB_K7_TILE", width > 4 ? 1 : 0) ? env_int("GTB_K7_STAGES", 2) : 0;
  if (log2t < 0 || !aligned) stages = 0;
  p->stages = 0;
  if (stages > 0) {
    const int tch = tile_chunk(width);
    if (log2t == 0) pick_tile<0>(diag, tch, dot, p);
    else if (log2t == 1) pick_tile<1>(diag, tch, dot, p);
    else pick_tile<2>(diag, tch, dot, p);
    const int TR = kTileBlock / p->T;
    const size_t stage_bytes = tile_stage_bytes(width, TR, diag);
    int max_smem = 0;
    GTB_CUDA_TRY(cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    if (stages > 8) stages = 8;
    while (stages > 1 && kBarBytes + stages * stage_bytes > (size_t)max_smem) --stages;
    const size_t smem = kBarBytes + stages * stage_bytes;
    if (smem <= (size_t)max_smem) {
      GTB_CUDA_TRY(cudaFuncSetAttribute(p->tfirst, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      GTB_CUDA_TRY(cudaFuncSetAttribute(p->tnext, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      GTB_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, p->tnext, kTileBlock, smem));
      per_sm = std::max(1, std::min(per_sm, kMaxBlocksPerSm * kBlock / kTileBlock));
      const int64_t n_tiles = (n + TR - 1) / TR;
      p->grid = (int)std::max<int64_t>(1, std::min<int64_t>(n_tiles, (int64_t)sms * per_sm));
      p->grid = std::min(p->grid, kMaxGrid);
      p->stages = stages;
      p->smem = smem;
      return GTB_OK;
    }
  }
  GTB_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, p->next, kBlock, 0));
  per_sm = std::max(1, std::min(per_sm, kMaxBlocksPerSm));
  const int64_t total = n * p->T;
  int64_t grid = std::min<int64_t>((total + kBlock - 1) / kBlock, (int64_t)sms * per_sm);
  p->grid = (int)std::max<int64_t>(1, std::min<int64_t>(grid, kMaxGrid));
  return GTB_OK;
}

void launch_step(const StepPlan& p, bool first, const StepArgs& sa, cudaStream_t st) {
  if (p.stages > 0)
    (first ? p.tfirst : p.tnext)<<<p.grid, p.block ? p.block : kTileBlock, p.smem, st>>>(sa, p.stages);
  else
    (first ? p.first : p.next)<<<p.grid, kBlock, 0, st>>>(sa);
}

void launch_fill(int mode, uint64_t seed, int64_t r0, int R, int64_t n, double* phi, cudaStream_t st) {
  const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((n * R + kBlock - 1) / kBlock, kMaxGrid));
  if (mode == 0)
    random_phase_kernel<<<grid, kBlock, 0, st>>>(seed, (int32_t)r0, R, n, reinterpret_cast<double2*>(phi));
  else
    basis_fill_kernel<<<grid, kBlock, 0, st>>>(r0, R, n, reinterpret_cast<double2*>(phi));
}

void launch_reduce_partials(const double2* partial, int stride, int grid, double2* sums, int nslots,
                            cudaStream_t st) {
  reduce_partials_kernel<<<nslots, 128, 0, st>>>(partial, stride, grid, sums);
}

int check_ell(const gtb_ell* H) {
  if (!H || H->n <= 0 || H->width < 0 || (H->width > 0 && (!H->cols || !H->vals)))
    return GTB_ERR_INVALID_ARG;
  if (H->n > (int64_t)INT32_MAX - 64) return GTB_ERR_INDEX_RANGE;
  return GTB_OK;
}

int check_ws(const void* ws, size_t ws_bytes, size_t need) {
  if (!ws || (reinterpret_cast<uintptr_t>(ws) & 255u) || ws_bytes < need) return GTB_ERR_WORKSPACE;
  return GTB_OK;
}

namespace {

struct KpmWs {
  double* phi_a;
  double* phi_b;
  double2* partial;  // [S][kMaxGrid]
  double2* sums;     // [S]
  int32_t* status;   // [0] = non-finite flag, [1] = sweep error, [2] = halo of H in rows
  int32_t* sync;     // [n/kGroupRows + 1]: step-0 chunks finished per row group   (K7s)
  double2* cpartial; // [2][n/kMinChunk + 1] chunk sums of one sweep            (K7s)
  double2* ctmp;     // [2][kSegs]
  size_t chunk_cap;
  size_t bytes;
};

constexpr int kMinChunk = 64;  // smallest chunk_rows the workspace is sized for

KpmWs carve_kpm(void* ws, int64_t n, int32_t M, int32_t R) {
  const size_t S = (size_t)(M + 1) / 2;
  Carver c(ws);
  KpmWs w;
  w.status = c.take<int32_t>(64);
  w.phi_a = c.take<double>((size_t)n * R * 2);
  w.phi_b = c.take<double>((size_t)n * R * 2);
  w.partial = c.take<double2>(S * kMaxGrid);
  w.sums = c.take<double2>(S);
  w.chunk_cap = (size_t)n / kMinChunk + 1;
  w.sync = c.take<int32_t>((size_t)n / kGroupRows + 1);
  w.cpartial = c.take<double2>(2 * w.chunk_cap);
  w.ctmp = c.take<double2>(2 * kSegs);
  w.bytes = c.off;
  return w;
}

int fill_grid(int64_t total) {
  return (int)std::max<int64_t>(1, std::min<int64_t>((total + kBlock - 1) / kBlock, kMaxGrid));
}

using SweepFn = void (*)(const SweepArgs);
SweepFn sweep_fn(int T, bool diag) {
  if (T == 1) return diag ? cheb_sweep_kernel<0, true> : cheb_sweep_kernel<0, false>;
  if (T == 2) return diag ? cheb_sweep_kernel<1, true> : cheb_sweep_kernel<1, false>;
  return diag ? cheb_sweep_kernel<2, true> : cheb_sweep_kernel<2, false>;
}

struct LoopTimer {
  cudaEvent_t beg = nullptr, end = nullptr;
  int passes = 0;
  bool armed = false;
};
thread_local LoopTimer g_timer;

}  // namespace
}  // namespace gtb

using namespace gtb;

extern "C" int gtb_random_phase_fill(uint64_t seed, int32_t r0, int32_t R, int64_t n, double* phi,
                                     void* stream) {
  if (R <= 0 || n < 0 || r0 < 0) return GTB_ERR_INVALID_ARG;
  if (n == 0) return GTB_OK;
  if (!phi) return GTB_ERR_INVALID_ARG;
  random_phase_kernel<<<fill_grid(n * R), kBlock, 0, static_cast<cudaStream_t>(stream)>>>(
      seed, r0, R, n, reinterpret_cast<double2*>(phi));
  GTB_LAUNCHED();
  return GTB_OK;
}

extern "C" size_t gtb_kpm_workspace_bytes(int64_t n, int32_t M, int32_t R_batch) {
  if (n <= 0 || M <= 0 || R_batch <= 0) return 0;
  return carve_kpm(nullptr, n, M, R_batch).bytes;
}

extern "C" int gtb_kpm_moments(const gtb_ell* H, double a, double b, int32_t M, int32_t R_total,
                               int32_t R_batch, uint64_t seed, int32_t mode_flags, double* mu, void* ws,
                               size_t ws_bytes, void* stream) {
  int rc = check_ell(H);
  if (rc != GTB_OK) return rc;
  if ((mode_flags & ~(1 | GTB_MODE_ORB4 | GTB_MODE_ORB9 | GTB_MODE_GROUP4)) ||
      ((mode_flags & GTB_MODE_ORB4) != 0) + ((mode_flags & GTB_MODE_ORB9) != 0) +
              ((mode_flags & GTB_MODE_GROUP4) != 0) > 1)
    return GTB_ERR_INVALID_ARG;
  const int32_t mode = mode_flags & 1;
  const int orb = (mode_flags & GTB_MODE_ORB4) ? 4 : (mode_flags & GTB_MODE_ORB9) ? 9 : 0;
  const bool grouped = (mode_flags & GTB_MODE_GROUP4) != 0;
  if (!mu || M <= 0 || !(a > 0.0) || !std::isfinite(b) || R_batch <= 0 || R_batch > 64 ||
      (mode != 0 && mode != 1) || (mode == 0 && R_total <= 0))
    return GTB_ERR_INVALID_ARG;
  rc = check_ws(ws, ws_bytes, gtb_kpm_workspace_bytes(H->n, M, R_batch));
  if (rc != GTB_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int64_t n = H->n;
  const KpmWs w = carve_kpm(ws, n, M, R_batch);
  const int S = (M + 1) / 2;  // fused passes: phi_1 .. phi_S
  const int64_t n_vec = mode == 0 ? (int64_t)R_total : n;
  GTB_CUDA_TRY(cudaMemsetAsync(w.sums, 0, sizeof(double2) * (size_t)S, st));
  GTB_CUDA_TRY(cudaMemsetAsync(w.status, 0, sizeof(int32_t) * 64, st));
  if (!g_timer.beg) {
    GTB_CUDA_TRY(cudaEventCreate(&g_timer.beg));
    GTB_CUDA_TRY(cudaEventCreate(&g_timer.end));
  }
  g_timer.armed = false;
  for (int64_t r0 = 0; r0 < n_vec; r0 += R_batch) {
    const int R = (int)std::min<int64_t>(R_batch, n_vec - r0);
    const bool last_batch = r0 + R_batch >= n_vec;
    StepPlan plan;
    if (grouped && !make_plan_grp4(H, R, false, &plan)) return GTB_ERR_INVALID_ARG;  // no scalar reading
    const bool blocked = grouped || (orb && env_int("GTB_K7_ORB4", 1) != 0 && make_plan_orb(H, R, orb, false, &plan));
    if (!blocked) {
      rc = make_plan(H, R, false, &plan);
      if (rc != GTB_OK) return rc;
    }
    // K7s (two steps per HBM sweep): opt-in (GTB_K7_SWEEP=1).  It moves 35 % fewer HBM bytes but
    // measures 2.60 ms per step at config 5 against K7's 2.20 ms, so K7 stays.
    int chunk_rows = env_int("GTB_K7_CHUNK", 128);
    if (chunk_rows != 64 && chunk_rows != 128 && chunk_rows != 256 && chunk_rows != 512 &&
        chunk_rows != 1024)
      chunk_rows = 128;
    const int n_chunks = (int)((n + chunk_rows - 1) / chunk_rows);
    const bool sweep = !blocked && env_int("GTB_K7_SWEEP", 0) != 0 && H->width >= 1 && H->width <= 4 &&
                       (R == 2 || R == 4 || R == 8) && n >= 2 * kGroupRows;
    int sweep_grid = 0, sweep_slack = 0;
    if (sweep) {
      int dev = 0, sms = kSmCount, per_sm = 0;
      GTB_CUDA_TRY(cudaGetDevice(&dev));
      GTB_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
      GTB_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(
          &per_sm, sweep_fn(plan.T, H->diag != nullptr), kBlock, 0));
      per_sm = std::max(1, std::min(per_sm, env_int("GTB_K7_SWEEP_BPS", kMaxBlocksPerSm)));
      sweep_grid = sms * per_sm;
      sweep_slack = env_int("GTB_K7_SLACK", sweep_grid * (kBlock / 32) / 2);  // chunks: one round of all warps
      GTB_CUDA_TRY(cudaMemsetAsync(w.status + 2, 0, sizeof(int32_t), st));
      halo_kernel<<<fill_grid(n * H->width), kBlock, 0, st>>>(H->cols, n, H->width, w.status + 2);
      GTB_LAUNCHED();
    }
    // K7p: every element of phi on its own resident thread -> all passes in one cooperative launch
    int small_grid = 0;
    void* small_fn = nullptr;
    if (!blocked && !sweep && plan.vw == 4 && S >= 2 && env_int("GTB_K7_SMALL", 1) != 0) {
      const bool dg = H->diag != nullptr;
      small_fn = plan.T == 1 ? (dg ? (void*)cheb_small_kernel<0, true> : (void*)cheb_small_kernel<0, false>)
               : plan.T == 2 ? (dg ? (void*)cheb_small_kernel<1, true> : (void*)cheb_small_kernel<1, false>)
                             : (dg ? (void*)cheb_small_kernel<2, true> : (void*)cheb_small_kernel<2, false>);
      int dev = 0, sms = kSmCount, per_sm = 0, coop = 0;
      GTB_CUDA_TRY(cudaGetDevice(&dev));
      GTB_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
      GTB_CUDA_TRY(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
      GTB_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, small_fn, kBlock, 0));
      const int64_t blocks = (n * plan.T + kBlock - 1) / kBlock;
      if (coop && blocks <= (int64_t)sms * per_sm && blocks <= kMaxGrid) small_grid = (int)blocks;
    }
    double* cur = w.phi_a;   // phi_k
    double* io = w.phi_b;    // phi_{k-1} -> phi_{k+1}
    if (mode == 0) {
      random_phase_kernel<<<fill_grid(n * R), kBlock, 0, st>>>(seed, (int32_t)r0, R, n,
                                                               reinterpret_cast<double2*>(cur));
    } else {
      basis_fill_kernel<<<fill_grid(n * R), kBlock, 0, st>>>(r0, R, n,
                                                             reinterpret_cast<double2*>(cur));
    }
    GTB_LAUNCHED();
    StepArgs sa{H->cols, H->vals, H->diag, n, H->width, plan.T, cur, io, 1.0 / a, b, w.partial};
    if (small_grid > 0) {  // K7p: K6 and all K7 passes in one launch
      if (last_batch) GTB_CUDA_TRY(cudaEventRecord(g_timer.beg, st));
      int S_arg = S;
      double inv_a = 1.0 / a;
      void* args[] = {&sa, &S_arg, &inv_a};
      GTB_CUDA_TRY(cudaLaunchCooperativeKernel(small_fn, dim3(small_grid), dim3(kBlock), args, 0, st));
      count_launch();
      if (last_batch) {
        GTB_CUDA_TRY(cudaEventRecord(g_timer.end, st));
        g_timer.passes = S;
        g_timer.armed = true;
      }
      reduce_partials_kernel<<<S, 128, 0, st>>>(w.partial, kMaxGrid, small_grid, w.sums);
      GTB_LAUNCHED();
      continue;
    }
    launch_step(plan, true, sa, st);  // K6: phi_1, <phi_0|phi_0>, Re<phi_1|phi_0>
    GTB_LAUNCHED();
    if (last_batch) GTB_CUDA_TRY(cudaEventRecord(g_timer.beg, st));
    int k = 1;
    if (sweep) {  // K7s: two steps per launch while at least two remain
      SweepFn fn = sweep_fn(plan.T, H->diag != nullptr);
      SweepArgs wa;
      wa.s = sa;
      wa.s.scale = 2.0 / a;
      wa.chunk_rows = chunk_rows;
      wa.n_chunks = n_chunks;
      wa.halo_rows = w.status + 2;
      wa.slack = sweep_slack;
      wa.group_done = w.sync;
      wa.error = w.status + 1;
      wa.partial0 = w.cpartial;
      wa.partial1 = w.cpartial + w.chunk_cap;
      for (; k + 1 < S; k += 2) {  // phi_{k+1}, phi_{k+2} from phi_k (cur after the swap), phi_{k-1}
        std::swap(cur, io);
        wa.s.phi_cur = cur;
        wa.s.phi_io = io;
        GTB_CUDA_TRY(cudaMemsetAsync(w.sync, 0, sizeof(int32_t) * ((size_t)n / kGroupRows + 1), st));
        fn<<<sweep_grid, kBlock, 0, st>>>(wa);
        GTB_LAUNCHED();
        reduce_chunks_kernel<<<dim3(kSegs, 2), kBlock, 0, st>>>(wa.partial0, wa.partial1, n_chunks,
                                                                w.ctmp);
        GTB_LAUNCHED();
        reduce_segs_kernel<<<1, 2, 0, st>>>(w.ctmp, w.sums + k);
        GTB_LAUNCHED();
        std::swap(cur, io);  // the sweep leaves phi_{k+2} in `cur`'s buffer and phi_{k+1} in `io`'s
      }
    }
    const int k_single = k;
    for (; k < S; ++k) {  // K7: phi_{k+1} from phi_k (cur) and phi_{k-1} (io)
      std::swap(cur, io);
      sa.phi_cur = cur;
      sa.phi_io = io;
      sa.scale = 2.0 / a;
      sa.partial = w.partial + (size_t)k * kMaxGrid;
      launch_step(plan, false, sa, st);
      GTB_LAUNCHED();
    }
    if (last_batch) {
      GTB_CUDA_TRY(cudaEventRecord(g_timer.end, st));
      g_timer.passes = S - 1;
      g_timer.armed = true;
    }
    // partial rows are kMaxGrid apart; only the first plan.grid entries of each are live
    reduce_partials_kernel<<<1, 128, 0, st>>>(w.partial, kMaxGrid, plan.grid, w.sums);
    GTB_LAUNCHED();
    if (k_single < S) {
      reduce_partials_kernel<<<S - k_single, 128, 0, st>>>(w.partial + (size_t)k_single * kMaxGrid,
                                                           kMaxGrid, plan.grid, w.sums + k_single);
      GTB_LAUNCHED();
    }
  }
  const double norm = mode == 0 ? (double)n * (double)R_total : (double)n;
  finish_moments_kernel<<<(M + kBlock - 1) / kBlock, kBlock, 0, st>>>(w.sums, M, norm, mu, w.status);
  GTB_LAUNCHED();
  return GTB_OK;
}

extern "C" int gtb_group_width(const gtb_ell* H, int32_t* scratch, void* stream, int32_t* width_out) {
  int rc = check_ell(H);
  if (rc != GTB_OK) return rc;
  if (!scratch || !width_out || H->n % 4 || H->width == 0) return GTB_ERR_INVALID_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  GTB_CUDA_TRY(cudaMemsetAsync(scratch, 0, sizeof(int32_t), st));
  group_rows_kernel<false><<<fill_grid(H->n / 4), kBlock, 0, st>>>(H->cols, H->vals, H->n, H->width, 0,
                                                                   nullptr, nullptr, scratch);
  GTB_LAUNCHED();
  GTB_CUDA_TRY(cudaMemcpyAsync(width_out, scratch, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  GTB_CUDA_TRY(cudaStreamSynchronize(st));
  if (*width_out < 1) *width_out = 1;  // a matrix without off-diagonal entries still gets one (zero) slot
  return GTB_OK;
}

extern "C" int gtb_group_rows(const gtb_ell* H, gtb_ell* G, int32_t* scratch, void* stream) {
  int rc = check_ell(H);
  if (rc != GTB_OK) return rc;
  if (!G || !scratch || H->n % 4 || H->width == 0 || G->n != H->n || G->width < 1 || !G->cols ||
      !G->vals || (reinterpret_cast<uintptr_t>(G->vals) & 31u))
    return GTB_ERR_INVALID_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  GTB_CUDA_TRY(cudaMemsetAsync(scratch, 0, sizeof(int32_t), st));
  group_rows_kernel<true><<<fill_grid(H->n / 4), kBlock, 0, st>>>(H->cols, H->vals, H->n, H->width,
                                                                  G->width, G->cols, G->vals, scratch);
  GTB_LAUNCHED();
  int32_t needed = 0;
  GTB_CUDA_TRY(cudaMemcpyAsync(&needed, scratch, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  GTB_CUDA_TRY(cudaStreamSynchronize(st));
  return needed > G->width ? GTB_ERR_ELL_OVERFLOW : GTB_OK;
}

extern "C" int gtb_kpm_status(const void* ws, void* stream) {
  if (!ws) return GTB_ERR_INVALID_ARG;
  int32_t flag[2] = {0, 0};
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  GTB_CUDA_TRY(cudaMemcpyAsync(flag, ws, sizeof(flag), cudaMemcpyDeviceToHost, st));
  GTB_CUDA_TRY(cudaStreamSynchronize(st));
  if (flag[1]) {  // a K7s dependency wait ran into its spin limit: the result is not valid
    note_cuda_error(cudaErrorLaunchTimeout, "cheb_sweep_kernel dependency wait");
    return GTB_ERR_CUDA;
  }
  return flag[0] ? GTB_ERR_DIVERGED : GTB_OK;
}

extern "C" int gtb_kpm_step(const gtb_ell* H, double a, double b, int32_t first, int32_t R,
                            const double* phi_cur, double* phi_io, double* sums, void* ws,
                            size_t ws_bytes, void* stream) {
  int rc = check_ell(H);
  if (rc != GTB_OK) return rc;
  if (!phi_cur || !phi_io || !sums || !(a > 0.0) || R <= 0 || R > 64 ||
      (reinterpret_cast<uintptr_t>(phi_cur) & 31u) || (reinterpret_cast<uintptr_t>(phi_io) & 31u))
    return GTB_ERR_INVALID_ARG;
  rc = check_ws(ws, ws_bytes, gtb_kpm_workspace_bytes(H->n, 2, R));
  if (rc != GTB_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const KpmWs w = carve_kpm(ws, H->n, 2, R);
  StepPlan plan;
  rc = make_plan(H, R, false, &plan);
  if (rc != GTB_OK) return rc;
  GTB_CUDA_TRY(cudaMemsetAsync(w.sums, 0, sizeof(double2), st));
  StepArgs sa{H->cols, H->vals, H->diag, H->n, H->width, plan.T, phi_cur, phi_io,
              (first ? 1.0 : 2.0) / a, b, w.partial};
  launch_step(plan, first != 0, sa, st);
  GTB_LAUNCHED();
  reduce_partials_kernel<<<1, 128, 0, st>>>(w.partial, kMaxGrid, plan.grid, w.sums);
  GTB_LAUNCHED();
  copy_sums_kernel<<<1, 1, 0, st>>>(w.sums, sums);
  GTB_LAUNCHED();
  return GTB_OK;
}

extern "C" int gtb_kpm_last_loop_ms(double* ms, int32_t* passes) {
  if (!ms || !passes) return GTB_ERR_INVALID_ARG;
  if (!g_timer.armed) return GTB_ERR_INVALID_ARG;
  GTB_CUDA_TRY(cudaEventSynchronize(g_timer.end));
  float t = 0.f;
  GTB_CUDA_TRY(cudaEventElapsedTime(&t, g_timer.beg, g_timer.end));
  *ms = (double)t;
  *passes = g_timer.passes;
  return GTB_OK;
}
