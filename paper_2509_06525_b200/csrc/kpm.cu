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
#include <mutex>

#include "tma.cuh"
#include "vecload.cuh"

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
                                                              int64_t n, double2* __restrict__ phi,
                                                              int64_t row_offset = 0) {
  const int64_t total = n * R;
  for (int64_t e = (int64_t)blockIdx.x * kBlock + threadIdx.x; e < total;
       e += (int64_t)gridDim.x * kBlock) {
    const int64_t i = e / R;
    const int32_t k = (int32_t)(e - i * R);
    const uint64_t key = mix64(seed + ((uint64_t)(uint32_t)(r0 + k) + 1ull) * kGamma);
    const uint64_t h = mix64(key + ((uint64_t)(i + row_offset) + 1ull) * kGamma);   // row_offset: a strip's first row
    const double u = (double)(h >> 11) * 0x1.0p-53;
    const double theta = 6.283185307179586 * u;
    double s, c;
    sincos(theta, &s, &c);
    phi[e] = make_double2(c, s);
  }
}

// exact-trace mode: phi[i][k] = delta(i, r0 + k)   (basis vectors e_{r0} .. e_{r0+R-1})
__global__ void __launch_bounds__(kBlock) basis_fill_kernel(int64_t r0, int32_t R, int64_t n,
                                                            double2* __restrict__ phi, int64_t row_offset = 0) {
  const int64_t total = n * R;
  for (int64_t e = (int64_t)blockIdx.x * kBlock + threadIdx.x; e < total;
       e += (int64_t)gridDim.x * kBlock) {
    const int64_t i = e / R;
    const int64_t k = e - i * R;
    phi[e] = make_double2(i + row_offset == r0 + k ? 1.0 : 0.0, 0.0);
  }
}


// K6 / K7.  Thread e handles element e of phi viewed as an array of Vec<VW>: row = e / T, vector
// group t = e % T, so a warp touches one contiguous 32*VW*8-byte span of phi_{n-1}/phi_{n+1}, and
// every gather of a row's neighbour is T consecutive threads reading R*16 contiguous bytes.
template <int VW, int LOG2T, bool kFirst, bool kDiag, int CH, int kMode>
__global__ void __launch_bounds__(kBlock) cheb_step_kernel(const StepArgs a) {
  constexpr bool kDotL = kMode == 1, kAxpy = kMode == 2;
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
    if (kAxpy) with = load_stream<VW>(a.axpy_acc + e * VW);
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
      if (!kAxpy) {
        s1 = fma(own.v[q], kDotL ? with.v[q] : own.v[q], s1);
        s2 = fma(y.v[q], kDotL ? with.v[q] : own.v[q], s2);
      }
    }
    store_stream<VW>(a.phi_io + e * VW, y);
    if (kAxpy) {
      axpy_into<VW>(with, y, a.axpy_cr, a.axpy_ci);
      store_stream<VW>(a.axpy_acc + e * VW, with);
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


// ---- K7x2: K7 for narrow rows with two independent elements in flight per thread --------------------
// K7 above is latency-bound at K = 3 (ncu: 94 % of the stall cycles on long_scoreboard, DRAM at 76 %):
// per element a thread issues its two streamed loads and the K column/hopping loads, and only then the K
// gathers that depend on the columns.  Here every thread works on TWO elements per iteration, one grid
// stride apart: all 2 x (2 + 2W) independent loads are issued first, then the 2 x W gathers, then the FMAs
// and the two stores.  W (3 or 4) is a compile-time bound on the row width, so everything is unrolled and
// lives in registers (64 registers: still 4 blocks per SM).  Same arithmetic order per element as K7.
// Config 5: 2.20 -> 1.99 ms per pass.
template <int LOG2T, bool kDiag, int W, int kMode>
__global__ void __launch_bounds__(kBlock) cheb_step_x2_kernel(const StepArgs a) {
  constexpr bool kDotL = kMode == 1, kAxpy = kMode == 2;
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
      if (kAxpy) with[r] = load_stream<VW>(a.axpy_acc + e[r] * VW);
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
          if (!kAxpy) {
            s1 = fma(own[r].v[q], kDotL ? with[r].v[q] : own[r].v[q], s1);
            s2 = fma(y.v[q], kDotL ? with[r].v[q] : own[r].v[q], s2);
          }
        }
        store_stream<VW>(a.phi_io + e[r] * VW, y);
        if (kAxpy) {
          axpy_into<VW>(with[r], y, a.axpy_cr, a.axpy_ci);
          store_stream<VW>(a.axpy_acc + e[r] * VW, with[r]);
        }
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

template <int LOG2T, int W, int DOT>
StepFn pick_x2(bool diag) {
  return diag ? cheb_step_x2_kernel<LOG2T, true, W, DOT> : cheb_step_x2_kernel<LOG2T, false, W, DOT>;
}
template <int LOG2T>
StepFn pick_x2(bool diag, int width, int mode) {
  if (width <= 3) return mode == 2 ? pick_x2<LOG2T, 3, 2>(diag) : mode == 1 ? pick_x2<LOG2T, 3, 1>(diag) : pick_x2<LOG2T, 3, 0>(diag);
  return mode == 2 ? pick_x2<LOG2T, 4, 2>(diag) : mode == 1 ? pick_x2<LOG2T, 4, 1>(diag) : pick_x2<LOG2T, 4, 0>(diag);
}

// ---- K7t: the same pass with the Hamiltonian stream staged by TMA ------------------------------
// With wide rows (K ~ 10-20) the register path above is latency-bound: every gather waits for a
// column index that itself comes from HBM.  Here one lane-parallel producer (warp 0) copies the
// next tiles' ELL slots (cols, vals, diag) into a ring of shared-memory stages with
// cp.async.bulk (TMA, completion on an mbarrier) and bulk-prefetches the tiles' phi_{n-1}/phi_n
// lines into L2, so the consumers' dependent chain is  LDS column -> gather  only.
constexpr int kBarBytes = 128;  // mbarrier ring at the start of dynamic shared memory

// stage layout (TR rows): vals [width][TR] f64 | diag [TR] f64 | cols [width][TR] i32
__host__ __device__ inline uint32_t tile_stage_bytes(int width, int TR, bool diag) {
  return (uint32_t)((width * TR * 12 + (diag ? TR * 8 : 0) + 127) / 128 * 128);
}

#ifndef GTB_TILE_BLOCK
#define GTB_TILE_BLOCK 256
#endif
constexpr int kTileBlock = GTB_TILE_BLOCK;  // threads per CTA of K7t

// Warp-specialised: warps 0 .. kTileBlock/32 - 1 consume, one more warp produces; a stage goes round on two
// mbarriers, full[s] (the copies' bytes) and empty[s] (one arrival per consumer warp), so consumer warps never
// wait for one another (with a __syncthreads per tile and warp 0 doubling as producer ncu showed 3-4 stall
// cycles per issue on `barrier`).
constexpr int kTileCta = kTileBlock + 32;
constexpr int kTileConsumers = kTileBlock / 32;

template <int LOG2T, bool kFirst, bool kDiag, int CH, int kMode>
__global__ void __launch_bounds__(kTileCta, 3) cheb_tile_kernel(const StepArgs a, const int nstages) {
  constexpr bool kDotL = kMode == 1, kAxpy = kMode == 2;
  constexpr int VW = 4;
  constexpr int T = 1 << LOG2T;
  constexpr int TR = kTileBlock / T;  // rows per tile: one consumer thread per 256-bit element
  extern __shared__ __align__(128) unsigned char smem[];
  const int64_t n = a.n;
  const int width = a.width;
  const double scale = a.scale, b = a.b;
  const uint32_t stage_bytes = tile_stage_bytes(width, TR, kDiag);
  const uint32_t vals_off = 0, diag_off = (uint32_t)width * TR * 8;
  const uint32_t cols_off = diag_off + (kDiag ? TR * 8 : 0);
  const uint32_t bar0 = smem_u32(smem);
  const uint32_t empty0 = bar0 + 64;   // full[s] at bar0 + 8 s, empty[s] at bar0 + 64 + 8 s (s < 8)
  unsigned char* const stage0 = smem + kBarBytes;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int64_t n_tiles = (n + TR - 1) / TR;
  const int64_t my_tiles = blockIdx.x < n_tiles ? (n_tiles - 1 - blockIdx.x) / gridDim.x + 1 : 0;

  if (tid == 0) {
    for (int s = 0; s < nstages; ++s) {
      mbar_init(bar0 + 8 * s, 1);
      mbar_init(empty0 + 8 * s, kTileConsumers);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  double s1 = 0.0, s2 = 0.0;
  if (wid == kTileConsumers) {   // ---- producer warp, lane-parallel
    for (int64_t i = 0; i < my_tiles; ++i) {
      const int s = (int)(i % nstages);
      if (i >= nstages) mbar_wait(empty0 + 8 * s, (uint32_t)(((i / nstages) - 1) & 1));
      const int64_t row0 = (blockIdx.x + i * gridDim.x) * TR;
      const uint32_t rows = (uint32_t)min((int64_t)TR, n - row0);
      const uint32_t bar = bar0 + 8 * s;
      const uint32_t base = smem_u32(stage0 + (size_t)s * stage_bytes);
      if (lane == 0) mbar_expect_tx(bar, rows * (uint32_t)(width * 12 + (kDiag ? 8 : 0)));
      __syncwarp();
      for (int j = lane; j < 2 * width + (kDotL || kAxpy ? 4 : 3); j += 32) {
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
          if (kAxpy) bulk_prefetch_l2(a.axpy_acc + row0 * (T * VW), rows * (T * VW * 8));
        }
      }
    }
    block_store_sums<kTileCta>(s1, s2, a.partial + blockIdx.x);
    return;
  }

  const int rl = tid >> LOG2T;             // row within the tile
  const int t = tid & (T - 1);             // 256-bit element within the row
  const double* xt = a.phi_cur + t * VW;
  // (loading the thread's own phi_{n-1} / phi_n elements one tile ahead was measured: no gain for K7w, and K7t
  // loses a third at its 72-register cap)
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
    __syncwarp();     // this warp has read stage s: one arrival hands its share back to the producer
    if (lane == 0) mbar_arrive(empty0 + 8 * s);
    if (live) {
      if (kDotL) with = load_stream<VW>(a.dot_with + e * VW);  // prefetched into L2 by the producer
      if (kAxpy) with = load_stream<VW>(a.axpy_acc + e * VW);
      Vec<VW> y;
#pragma unroll
      for (int q = 0; q < VW; ++q) {
        y.v[q] = (acc.v[q] - b * own.v[q]) * scale;
        if (!kFirst) y.v[q] -= prev.v[q];
        if (!kAxpy) {
          s1 = fma(own.v[q], kDotL ? with.v[q] : own.v[q], s1);
          s2 = fma(y.v[q], kDotL ? with.v[q] : own.v[q], s2);
        }
      }
      store_stream<VW>(a.phi_io + e * VW, y);
      if (kAxpy) {
        axpy_into<VW>(with, y, a.axpy_cr, a.axpy_ci);
        store_stream<VW>(a.axpy_acc + e * VW, with);
      }
    }
  }
  block_store_sums<kTileCta>(s1, s2, a.partial + blockIdx.x);
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


// ---- K7c: all passes of a TINY system inside one thread-block cluster, phi in distributed shared memory -----
// Config 1 (2 304 atoms, R = 4: 4 608 elements of 32 bytes) fits the shared memory of one cluster of 8 CTAs with
// one thread per element.  Each CTA keeps its slice of both vector sets in its own shared memory for the whole
// run, a thread keeps its row's <= 4 columns and hoppings in registers, gathers go to the owning CTA's shared
// memory (mapa + ld.shared::cluster), and the passes are separated by a cluster barrier (arrive.release /
// wait.acquire) instead of K7p's grid-wide barrier: no global-memory traffic per pass but the block sums.
// Same arithmetic order per element and the same per-(pass, block) sums layout as K7p.
constexpr int kClusterSize = 8;

__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ uint32_t map_to_cta(uint32_t local_addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local_addr), "r"(rank));
  return r;
}
__device__ __forceinline__ Vec<4> ld_cluster(uint32_t addr) {
  Vec<4> r;
  asm volatile("ld.shared::cluster.v2.f64 {%0,%1}, [%2];" : "=d"(r.v[0]), "=d"(r.v[1]) : "r"(addr) : "memory");
  asm volatile("ld.shared::cluster.v2.f64 {%0,%1}, [%2];" : "=d"(r.v[2]), "=d"(r.v[3]) : "r"(addr + 16) : "memory");
  return r;
}
__device__ __forceinline__ void cluster_sync() {
  asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
  asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}

template <int LOG2T, bool kDiag>
__global__ void __cluster_dims__(kClusterSize, 1, 1) __launch_bounds__(1024)
    cheb_cluster_kernel(const StepArgs a, const int S, const double inv_a, const int per_cta) {
  constexpr int VW = 4;
  constexpr int T = 1 << LOG2T;
  constexpr int W = 4;   // width bound: columns and hoppings live in registers
  extern __shared__ __align__(16) unsigned char s_phi[];   // [2][per_cta] elements of 32 bytes
  const int64_t n = a.n;
  const int64_t total = n * T;
  const uint32_t rank = cluster_ctarank();
  const int tid = threadIdx.x;
  const int64_t e = (int64_t)rank * per_cta + tid;
  const bool live = tid < per_cta && e < total;
  const int64_t row = live ? (e >> LOG2T) : 0;
  const int t = (int)(e & (T - 1));
  const uint32_t base = smem_u32(s_phi);
  const uint32_t buf_bytes = (uint32_t)per_cta * 32;
  double* mine = reinterpret_cast<double*>(s_phi) + (size_t)tid * VW;   // + buffer * per_cta * VW
  // phi_0 (written by the fill kernel) -> buffer 0
  if (live) {
    const Vec<VW> x0 = load_gather<VW>(a.phi_cur + e * VW);
#pragma unroll
    for (int q = 0; q < VW; ++q) mine[q] = x0.v[q];
  }
  // the row's slots: remote addresses of the gathered elements in buffer 0 (buffer 1: + buf_bytes)
  uint32_t gaddr[W];
  double v[W];
#pragma unroll
  for (int k = 0; k < W; ++k) {
    const bool ok = live && k < a.width;
    const int64_t c = ok ? (int64_t)__ldg(a.cols + (size_t)k * n + row) : row;
    v[k] = ok ? __ldg(a.vals + (size_t)k * n + row) : 0.0;
    const int64_t ce = c * T + t;
    gaddr[k] = map_to_cta(base + (uint32_t)(ce % per_cta) * 32, (uint32_t)(ce / per_cta));
  }
  const double dg = kDiag && live ? __ldg(a.diag + row) : 0.0;
  const double b = a.b;
  const int nwarps = (int)(blockDim.x >> 5);
  double2* s_sums = reinterpret_cast<double2*>(s_phi + 2 * (size_t)buf_bytes);   // [S][nwarps]
  cluster_sync();   // every CTA's slice of phi_0 is in place
  int cur = 0;
  for (int k = 0; k < S; ++k) {
    const double scale = k == 0 ? inv_a : 2.0 * inv_a;
    double s1 = 0.0, s2 = 0.0;
    if (live) {
      const uint32_t off = cur ? buf_bytes : 0u;
      Vec<VW> acc;
#pragma unroll
      for (int q = 0; q < VW; ++q) acc.v[q] = 0.0;
#pragma unroll
      for (int s = 0; s < W; ++s) {
        const Vec<VW> x = ld_cluster(gaddr[s] + off);
#pragma unroll
        for (int q = 0; q < VW; ++q) acc.v[q] = fma(v[s], x.v[q], acc.v[q]);
      }
      const double* own_p = mine + (size_t)cur * per_cta * VW;
      double* io_p = mine + (size_t)(cur ^ 1) * per_cta * VW;
#pragma unroll
      for (int q = 0; q < VW; ++q) {
        const double own = own_p[q];
        double hx = acc.v[q];
        if (kDiag) hx = fma(dg, own, hx);
        double y = (hx - b * own) * scale;
        if (k > 0) y -= io_p[q];
        s1 = fma(own, own, s1);
        s2 = fma(y, own, s2);
        io_p[q] = y;
      }
    }
    // warp sums parked in shared memory, [pass][warp]: no block barrier and no serial block sum inside a pass
    s1 = warp_sum(s1);
    s2 = warp_sum(s2);
    if ((tid & 31) == 0) s_sums[(size_t)k * nwarps + (tid >> 5)] = make_double2(s1, s2);
    cluster_sync();   // phi_{k+1} complete in every CTA before anyone gathers it
    cur ^= 1;
  }
  for (int k = tid; k < S; k += (int)blockDim.x) {   // block sums in warp order, as K7p's
    double2 acc = s_sums[(size_t)k * nwarps];
    for (int w = 1; w < nwarps; ++w) {
      acc.x += s_sums[(size_t)k * nwarps + w].x;
      acc.y += s_sums[(size_t)k * nwarps + w].y;
    }
    a.partial[(size_t)k * kMaxGrid + blockIdx.x] = acc;
  }
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
template <int VW, int LOG2T, int CH, int DOT>
void pick_ch(bool diag, StepPlan* p) {
  p->first = diag ? cheb_step_kernel<VW, LOG2T, true, true, CH, DOT> : cheb_step_kernel<VW, LOG2T, true, false, CH, DOT>;
  p->next = diag ? cheb_step_kernel<VW, LOG2T, false, true, CH, DOT> : cheb_step_kernel<VW, LOG2T, false, false, CH, DOT>;
}

template <int VW, int LOG2T>
void pick(bool diag, int ch, int mode, StepPlan* p) {
  if (ch == 0) { if (mode == 2) pick_ch<VW, LOG2T, 0, 2>(diag, p); else if (mode == 1) pick_ch<VW, LOG2T, 0, 1>(diag, p); else pick_ch<VW, LOG2T, 0, 0>(diag, p); }
  else { if (mode == 2) pick_ch<VW, LOG2T, 8, 2>(diag, p); else if (mode == 1) pick_ch<VW, LOG2T, 8, 1>(diag, p); else pick_ch<VW, LOG2T, 8, 0>(diag, p); }
}

template <int LOG2T, int CH, int DOT>
void pick_tile_ch(bool diag, StepPlan* p) {
  p->tfirst = diag ? cheb_tile_kernel<LOG2T, true, true, CH, DOT> : cheb_tile_kernel<LOG2T, true, false, CH, DOT>;
  p->tnext = diag ? cheb_tile_kernel<LOG2T, false, true, CH, DOT> : cheb_tile_kernel<LOG2T, false, false, CH, DOT>;
}

template <int LOG2T, int DOT>
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
void pick_tile(bool diag, int ch, int mode, StepPlan* p) {
  if (mode == 2) pick_tile_dot<LOG2T, 2>(diag, ch, p);
  else if (mode == 1) pick_tile_dot<LOG2T, 1>(diag, ch, p);
  else pick_tile_dot<LOG2T, 0>(diag, ch, p);
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


}  // namespace

// Picks the kernels and the launch shape of the fused pass for (H, R).  opt (may be NULL) pins a
// kernel; a pinned kernel that cannot take this matrix is GTB_ERR_INVALID_ARG, never a silent detour.
int make_plan(const gtb_ell* H, int R, int dot, const gtb_kpm_options* opt, StepPlan* p) {
  if (dot < 0 || dot > 2) return GTB_ERR_INVALID_ARG;
  const int64_t n = H->n;
  const int width = H->width;
  const bool diag = H->diag != nullptr;
  const int want = opt ? opt->kernel : GTB_KERNEL_AUTO;
  if (want < GTB_KERNEL_AUTO || want > GTB_KERNEL_TILE || (opt && (opt->tile_stages < 0 || opt->tile_stages > 8)))
    return GTB_ERR_INVALID_ARG;
  const int ch = width <= 4 ? 0 : 8;
  int log2t = -1;
  if (R == 2) { pick<4, 0>(diag, ch, dot, p); p->vw = 4; p->T = 1; log2t = 0; }
  else if (R == 4) { pick<4, 1>(diag, ch, dot, p); p->vw = 4; p->T = 2; log2t = 1; }
  else if (R == 8) { pick<4, 2>(diag, ch, dot, p); p->vw = 4; p->T = 4; log2t = 2; }
  else if (R == 1) { pick<2, 0>(diag, ch, dot, p); p->vw = 2; p->T = 1; }
  else { pick<2, -1>(diag, ch, dot, p); p->vw = 2; p->T = R; }
  // K7x2: narrow rows (K <= 4) take the two-elements-in-flight kernel for every pass but the first
  const bool x2_ok = log2t >= 0 && width >= 1 && width <= 4;
  if (want == GTB_KERNEL_ROW_X2 && !x2_ok) return GTB_ERR_INVALID_ARG;
  if (x2_ok && (want == GTB_KERNEL_AUTO || want == GTB_KERNEL_ROW_X2))
    p->next = log2t == 0 ? pick_x2<0>(diag, width, dot) : log2t == 1 ? pick_x2<1>(diag, width, dot)
                                                                    : pick_x2<2>(diag, width, dot);
  int dev = 0, sms = kSmCount, per_sm = 0;
  GTB_CUDA_TRY(cudaGetDevice(&dev));
  GTB_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  // TMA-staged path: bulk copies need 16-byte aligned sources and sizes in every slot row
  const bool tile_ok = log2t >= 0 && n % 4 == 0 && width >= 1 &&
                       !(reinterpret_cast<uintptr_t>(H->cols) & 15u) &&
                       !(reinterpret_cast<uintptr_t>(H->vals) & 15u) &&
                       !(reinterpret_cast<uintptr_t>(H->diag) & 15u);
  if (want == GTB_KERNEL_TILE && !tile_ok) return GTB_ERR_INVALID_ARG;
  int stages = 0;
  // wide rows, and narrow rows with a full 128-byte line per gathered neighbour (R = 8: c4 0.93 against K7x2's
  // 0.88 of the measured peak); at R = 2, 4 narrow rows stay on K7x2 (c5: 2.00 against 2.07 ms)
  if (tile_ok && (want == GTB_KERNEL_TILE || (want == GTB_KERNEL_AUTO && (width > 4 || R == 8))))
    stages = opt && opt->tile_stages ? opt->tile_stages : 2;
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
    while (stages > 1 && kBarBytes + stages * stage_bytes > (size_t)max_smem) --stages;
    const size_t smem = kBarBytes + stages * stage_bytes;
    if (smem <= (size_t)max_smem) {
      GTB_CUDA_TRY(cudaFuncSetAttribute(p->tfirst, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      GTB_CUDA_TRY(cudaFuncSetAttribute(p->tnext, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      GTB_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, p->tnext, kTileCta, smem));
      per_sm = std::max(1, std::min(per_sm, kMaxBlocksPerSm * kBlock / kTileBlock));
      const int64_t n_tiles = (n + TR - 1) / TR;
      p->grid = (int)std::max<int64_t>(1, std::min<int64_t>(n_tiles, (int64_t)sms * per_sm));
      p->grid = std::min(p->grid, kMaxGrid);
      p->stages = stages;
      p->smem = smem;
      return GTB_OK;
    }
    if (want == GTB_KERNEL_TILE) return GTB_ERR_INVALID_ARG;   // one stage does not fit in shared memory
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
    (first ? p.tfirst : p.tnext)<<<p.grid, p.block ? p.block : kTileCta, p.smem, st>>>(sa, p.stages);
  else
    (first ? p.first : p.next)<<<p.grid, p.block ? p.block : kBlock, p.smem, st>>>(sa);
}

void launch_fill(int mode, uint64_t seed, int64_t r0, int R, int64_t n, double* phi, cudaStream_t st,
                 int64_t row_offset) {
  const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((n * R + kBlock - 1) / kBlock, kMaxGrid));
  if (mode == 0)
    random_phase_kernel<<<grid, kBlock, 0, st>>>(seed, (int32_t)r0, R, n, reinterpret_cast<double2*>(phi), row_offset);
  else
    basis_fill_kernel<<<grid, kBlock, 0, st>>>(r0, R, n, reinterpret_cast<double2*>(phi), row_offset);
}

void launch_finish_moments(const double2* sums, int M, double norm, double* mu, int32_t* status, cudaStream_t st) {
  finish_moments_kernel<<<(M + kBlock - 1) / kBlock, kBlock, 0, st>>>(sums, M, norm, mu, status);
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

int check_options(const gtb_kpm_options* opt) {
  if (!opt) return GTB_OK;
  if (opt->kernel < GTB_KERNEL_AUTO || opt->kernel > GTB_KERNEL_TILE || opt->tile_stages < 0 ||
      opt->tile_stages > 8 ||
      (opt->flags & ~(GTB_OPT_PER_PASS_LAUNCH | GTB_OPT_SCALAR_BLOCKS | GTB_OPT_BLOCK_DIRECT |
                      GTB_OPT_SEPARATE_AXPY | GTB_OPT_GRID_SYNC)) ||
      ((opt->loop_begin == nullptr) != (opt->loop_end == nullptr)) ||
      (opt->alt && opt->alt_mode != GTB_MODE_PACKED && opt->alt_mode != GTB_MODE_WINDOW))
    return GTB_ERR_INVALID_ARG;
  return GTB_OK;
}

namespace {

struct KpmWs {
  double* phi_a;
  double* phi_b;
  double2* partial;  // [S][kMaxGrid]
  double2* sums;     // [S]
  int32_t* status;   // [0] = non-finite flag
  size_t bytes;
};

KpmWs carve_kpm(void* ws, int64_t n, int32_t M, int32_t R) {
  const size_t S = (size_t)(M + 1) / 2;
  Carver c(ws);
  KpmWs w;
  w.status = c.take<int32_t>(64);
  w.phi_a = c.take<double>((size_t)n * R * 2);
  w.phi_b = c.take<double>((size_t)n * R * 2);
  w.partial = c.take<double2>(S * kMaxGrid);
  w.sums = c.take<double2>(S);
  w.bytes = c.off;
  return w;
}

int fill_grid(int64_t total) {
  return (int)std::max<int64_t>(1, std::min<int64_t>((total + kBlock - 1) / kBlock, kMaxGrid));
}

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
                               size_t ws_bytes, void* stream, const gtb_kpm_options* opt) {
  int rc = check_ell(H);
  if (rc != GTB_OK) return rc;
  rc = check_options(opt);
  if (rc != GTB_OK) return rc;
  if ((mode_flags & ~(1 | GTB_MODE_ORB4 | GTB_MODE_ORB9 | GTB_MODE_BLOCK9 | GTB_MODE_BOND9 | GTB_MODE_PACKED |
                     GTB_MODE_WINDOW)) ||
      ((mode_flags & GTB_MODE_ORB4) != 0) + ((mode_flags & GTB_MODE_ORB9) != 0) +
              ((mode_flags & GTB_MODE_BLOCK9) != 0) + ((mode_flags & GTB_MODE_BOND9) != 0) +
              ((mode_flags & GTB_MODE_PACKED) != 0) + ((mode_flags & GTB_MODE_WINDOW) != 0) > 1)
    return GTB_ERR_INVALID_ARG;
  const int32_t mode = mode_flags & 1;
  const bool packed = (mode_flags & GTB_MODE_PACKED) != 0;
  const bool windowed = (mode_flags & GTB_MODE_WINDOW) != 0;
  const int opt_flags = opt ? opt->flags : 0;
  const int orb = (mode_flags & GTB_MODE_ORB4) ? 4 : (mode_flags & GTB_MODE_ORB9) ? 9 : 0;
  const int rep = (mode_flags & GTB_MODE_BLOCK9) ? 1 : (mode_flags & GTB_MODE_BOND9) ? 2 : 0;
  if (!mu || M <= 0 || !(a > 0.0) || !std::isfinite(b) || R_batch <= 0 || R_batch > 64 ||
      (mode != 0 && mode != 1) || (mode == 0 && R_total <= 0))
    return GTB_ERR_INVALID_ARG;
  // vector rows: in the block / bond representations H->n counts atoms, 9 orbitals each
  const int64_t n = rep ? 9 * H->n : H->n;
  if (n > (int64_t)INT32_MAX - 64) return GTB_ERR_INDEX_RANGE;
  rc = check_ws(ws, ws_bytes, gtb_kpm_workspace_bytes(n, M, R_batch));
  if (rc != GTB_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const KpmWs w = carve_kpm(ws, n, M, R_batch);
  const int S = (M + 1) / 2;  // fused passes: phi_1 .. phi_S
  const int64_t n_vec = mode == 0 ? (int64_t)R_total : n;
  cudaEvent_t ev_beg = opt ? static_cast<cudaEvent_t>(opt->loop_begin) : nullptr;
  cudaEvent_t ev_end = opt ? static_cast<cudaEvent_t>(opt->loop_end) : nullptr;
  GTB_CUDA_TRY(cudaMemsetAsync(w.sums, 0, sizeof(double2) * (size_t)S, st));
  GTB_CUDA_TRY(cudaMemsetAsync(w.status, 0, sizeof(int32_t) * 64, st));
  for (int64_t r0 = 0; r0 < n_vec; r0 += R_batch) {
    const int R = (int)std::min<int64_t>(R_batch, n_vec - r0);
    const bool last_batch = r0 + R_batch >= n_vec;
    StepPlan plan;
    bool blocked = false;
    if (packed) {  // packed rows: no plain reading exists
      if (!make_plan_packed(H, R, 0, &plan)) return GTB_ERR_INVALID_ARG;
      blocked = true;
    } else if (windowed) {  // windowed tiles, built for R_batch vectors: every batch must be full
      if (R != R_batch || !make_plan_window(H, R, 0, opt ? opt->tile_stages : 0, &plan)) return GTB_ERR_INVALID_ARG;
      blocked = true;
    } else if (rep) {  // block / bond representation: no scalar reading exists
      if (!make_plan_rep9(H, R, rep, &plan)) return GTB_ERR_INVALID_ARG;
      blocked = true;
    } else if (orb && !(opt_flags & GTB_OPT_SCALAR_BLOCKS)) {
      blocked = make_plan_orb(H, R, orb, false, (opt_flags & GTB_OPT_BLOCK_DIRECT) != 0, &plan);
    }
    if (!blocked) {
      rc = make_plan(H, R, false, opt, &plan);
      if (rc != GTB_OK) return rc;
    }
    // K7c: a tiny system inside one cluster of 8 CTAs, phi in distributed shared memory
    int cluster_threads = 0;
    if (!blocked && plan.vw == 4 && S >= 2 && H->width <= 4 && n * plan.T <= kClusterSize * 1024 &&
        !(opt_flags & (GTB_OPT_PER_PASS_LAUNCH | GTB_OPT_GRID_SYNC)) && (!opt || opt->kernel == GTB_KERNEL_AUTO))
      cluster_threads = (int)(((n * plan.T + kClusterSize - 1) / kClusterSize + 31) / 32 * 32);
    if (cluster_threads > 0 && (size_t)2 * cluster_threads * 32 + (size_t)S * (cluster_threads / 32) * 16 > 200 * 1024)
      cluster_threads = 0;   // the per-pass warp sums must fit beside the vectors
    // K7p: every element of phi on its own resident thread -> all passes in one cooperative launch
    int small_grid = 0;
    void* small_fn = nullptr;
    if (!blocked && plan.vw == 4 && S >= 2 && !(opt_flags & GTB_OPT_PER_PASS_LAUNCH) &&
        (!opt || opt->kernel == GTB_KERNEL_AUTO)) {
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
    launch_fill(mode, seed, r0, R, n, cur, st);
    GTB_LAUNCHED();
    StepArgs sa{H->cols, H->vals, H->diag, n, windowed ? (H->width & 0xffff) : H->width, plan.T, cur, io, 1.0 / a, b,
                w.partial};
    sa.aux = windowed ? ((H->width >> 16) & 0xff) : 0;
    if (cluster_threads > 0) {  // K7c: K6 and all K7 passes in one cluster launch
      const bool dg = H->diag != nullptr;
      using ClusterFn = void (*)(const StepArgs, const int, const double, const int);
      ClusterFn fn = plan.T == 1 ? (dg ? cheb_cluster_kernel<0, true> : cheb_cluster_kernel<0, false>)
                   : plan.T == 2 ? (dg ? cheb_cluster_kernel<1, true> : cheb_cluster_kernel<1, false>)
                                 : (dg ? cheb_cluster_kernel<2, true> : cheb_cluster_kernel<2, false>);
      const size_t smem = (size_t)2 * cluster_threads * 32 + (size_t)S * (cluster_threads / 32) * 16;
      GTB_CUDA_TRY(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      if (last_batch && ev_beg) GTB_CUDA_TRY(cudaEventRecord(ev_beg, st));
      fn<<<kClusterSize, cluster_threads, smem, st>>>(sa, S, 1.0 / a, cluster_threads);
      GTB_LAUNCHED();
      if (last_batch && ev_end) {
        GTB_CUDA_TRY(cudaEventRecord(ev_end, st));
        if (opt->loop_passes) *opt->loop_passes = S;
      }
      reduce_partials_kernel<<<S, 128, 0, st>>>(w.partial, kMaxGrid, kClusterSize, w.sums);
      GTB_LAUNCHED();
      continue;
    }
    if (small_grid > 0) {  // K7p: K6 and all K7 passes in one launch
      if (last_batch && ev_beg) GTB_CUDA_TRY(cudaEventRecord(ev_beg, st));
      int S_arg = S;
      double inv_a = 1.0 / a;
      void* args[] = {&sa, &S_arg, &inv_a};
      GTB_CUDA_TRY(cudaLaunchCooperativeKernel(small_fn, dim3(small_grid), dim3(kBlock), args, 0, st));
      count_launch();
      if (last_batch && ev_end) {
        GTB_CUDA_TRY(cudaEventRecord(ev_end, st));
        if (opt->loop_passes) *opt->loop_passes = S;
      }
      reduce_partials_kernel<<<S, 128, 0, st>>>(w.partial, kMaxGrid, small_grid, w.sums);
      GTB_LAUNCHED();
      continue;
    }
    launch_step(plan, true, sa, st);  // K6: phi_1, <phi_0|phi_0>, Re<phi_1|phi_0>
    GTB_LAUNCHED();
    if (last_batch && ev_beg) GTB_CUDA_TRY(cudaEventRecord(ev_beg, st));
    for (int k = 1; k < S; ++k) {  // K7: phi_{k+1} from phi_k (cur) and phi_{k-1} (io)
      std::swap(cur, io);
      sa.phi_cur = cur;
      sa.phi_io = io;
      sa.scale = 2.0 / a;
      sa.partial = w.partial + (size_t)k * kMaxGrid;
      launch_step(plan, false, sa, st);
      GTB_LAUNCHED();
    }
    if (last_batch && ev_end) {
      GTB_CUDA_TRY(cudaEventRecord(ev_end, st));
      if (opt->loop_passes) *opt->loop_passes = S - 1;
    }
    // partial rows are kMaxGrid apart; only the first plan.grid entries of each are live
    reduce_partials_kernel<<<S, 128, 0, st>>>(w.partial, kMaxGrid, plan.grid, w.sums);
    GTB_LAUNCHED();
  }
  const double norm = mode == 0 ? (double)n * (double)R_total : (double)n;
  finish_moments_kernel<<<(M + kBlock - 1) / kBlock, kBlock, 0, st>>>(w.sums, M, norm, mu, w.status);
  GTB_LAUNCHED();
  return GTB_OK;
}

extern "C" int gtb_kpm_status(const void* ws, void* stream) {
  if (!ws) return GTB_ERR_INVALID_ARG;
  int32_t flag = 0;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  GTB_CUDA_TRY(cudaMemcpyAsync(&flag, ws, sizeof(flag), cudaMemcpyDeviceToHost, st));
  GTB_CUDA_TRY(cudaStreamSynchronize(st));
  return flag ? GTB_ERR_DIVERGED : GTB_OK;
}

// ---- gtb_kpm_moments_static: the same run with its scratch in a static device array -------------------------
// For callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc): the
// workspace of gtb_kpm_moments lives in g_static_ws below, GTB_STATIC_WS_BYTES per GPU that loads the library,
// held until the process exits.  In host code the NAME g_static_ws is a host-side stand-in, not a device
// address -- a kernel handed &g_static_ws[0] from the host faults (or, where the GPU reaches host memory,
// silently uses the wrong memory) -- so the device address is asked for once per device, with that device
// current, by cudaGetSymbolAddress, and that pointer is what goes down as the workspace.
static __device__ __align__(256) unsigned char g_static_ws[GTB_STATIC_WS_BYTES];

namespace {
constexpr int kMaxDevices = 64;
std::mutex g_static_mutex;
void* g_static_addr[kMaxDevices] = {};   // device address of g_static_ws on device d, once asked for
}  // namespace

extern "C" int gtb_kpm_moments_static(const gtb_ell* H, double a, double b, int32_t M, int32_t R_total,
                                      int32_t R_batch, uint64_t seed, int32_t mode_flags, double* mu,
                                      void* stream, const gtb_kpm_options* opt) {
  int rc = check_ell(H);
  if (rc != GTB_OK) return rc;
  if (M <= 0 || R_batch <= 0 || R_batch > 64) return GTB_ERR_INVALID_ARG;
  const bool rep = (mode_flags & (GTB_MODE_BLOCK9 | GTB_MODE_BOND9)) != 0;
  const int64_t rows = rep ? 9 * H->n : H->n;
  // the size is checked before anything is launched: nothing beyond the array is ever carved
  if (rows > (int64_t)GTB_STATIC_WS_BYTES || gtb_kpm_workspace_bytes(rows, M, R_batch) > (size_t)GTB_STATIC_WS_BYTES)
    return GTB_ERR_STATIC_LIMIT;
  int dev = 0;
  GTB_CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return GTB_ERR_INVALID_ARG;
  void* ws = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_addr[dev]) {
      void* p = nullptr;
      GTB_CUDA_TRY(cudaGetSymbolAddress(&p, g_static_ws));
      g_static_addr[dev] = p;
    }
    ws = g_static_addr[dev];
  }
  // gtb_kpm_moments clears what must start at zero (the per-pass sums and the status word) on the stream and
  // overwrites every other word it later reads; it calls no allocating routine
  return gtb_kpm_moments(H, a, b, M, R_total, R_batch, seed, mode_flags, mu, ws, (size_t)GTB_STATIC_WS_BYTES, stream,
                         opt);
}

extern "C" int gtb_kpm_step(const gtb_ell* H, double a, double b, int32_t first, int32_t R,
                            const double* phi_cur, double* phi_io, double* sums, int32_t mode_flags,
                            void* ws, size_t ws_bytes, void* stream, const gtb_kpm_options* opt) {
  int rc = check_ell(H);
  if (rc != GTB_OK) return rc;
  rc = check_options(opt);
  if (rc != GTB_OK) return rc;
  const int orb = (mode_flags & GTB_MODE_ORB4) ? 4 : (mode_flags & GTB_MODE_ORB9) ? 9 : 0;
  const int rep = (mode_flags & GTB_MODE_BLOCK9) ? 1 : (mode_flags & GTB_MODE_BOND9) ? 2 : 0;
  const bool packed = (mode_flags & GTB_MODE_PACKED) != 0;
  const bool windowed = (mode_flags & GTB_MODE_WINDOW) != 0;
  if ((mode_flags & ~(GTB_MODE_ORB4 | GTB_MODE_ORB9 | GTB_MODE_BLOCK9 | GTB_MODE_BOND9 | GTB_MODE_PACKED |
                      GTB_MODE_WINDOW)) ||
      (orb != 0) + (rep != 0) + (packed ? 1 : 0) + (windowed ? 1 : 0) > 1 || ((mode_flags & GTB_MODE_ORB4) && (mode_flags & GTB_MODE_ORB9)) ||
      ((mode_flags & GTB_MODE_BLOCK9) && (mode_flags & GTB_MODE_BOND9)))
    return GTB_ERR_INVALID_ARG;
  if (!phi_cur || !phi_io || !sums || !(a > 0.0) || R <= 0 || R > 64 ||
      (reinterpret_cast<uintptr_t>(phi_cur) & 31u) || (reinterpret_cast<uintptr_t>(phi_io) & 31u))
    return GTB_ERR_INVALID_ARG;
  const int64_t n = rep ? 9 * H->n : H->n;   // vector rows
  if (n > (int64_t)INT32_MAX - 64) return GTB_ERR_INDEX_RANGE;
  rc = check_ws(ws, ws_bytes, gtb_kpm_workspace_bytes(n, 2, R));
  if (rc != GTB_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const KpmWs w = carve_kpm(ws, n, 2, R);
  StepPlan plan;
  const int opt_flags = opt ? opt->flags : 0;
  bool blocked = false;
  if (packed) {
    if (!make_plan_packed(H, R, 0, &plan)) return GTB_ERR_INVALID_ARG;
    blocked = true;
  } else if (windowed) {
    if (!make_plan_window(H, R, 0, opt ? opt->tile_stages : 0, &plan)) return GTB_ERR_INVALID_ARG;
    blocked = true;
  } else if (rep) {
    if (!make_plan_rep9(H, R, rep, &plan)) return GTB_ERR_INVALID_ARG;
    blocked = true;
  } else if (orb && !(opt_flags & GTB_OPT_SCALAR_BLOCKS)) {
    blocked = make_plan_orb(H, R, orb, false, (opt_flags & GTB_OPT_BLOCK_DIRECT) != 0, &plan);
  }
  if (!blocked) {
    rc = make_plan(H, R, false, opt, &plan);
    if (rc != GTB_OK) return rc;
  }
  GTB_CUDA_TRY(cudaMemsetAsync(w.sums, 0, sizeof(double2), st));
  StepArgs sa{H->cols, H->vals, H->diag, n, windowed ? (H->width & 0xffff) : H->width, plan.T, phi_cur, phi_io,
              (first ? 1.0 : 2.0) / a, b, w.partial};
  sa.aux = windowed ? ((H->width >> 16) & 0xff) : 0;
  launch_step(plan, first != 0, sa, st);
  GTB_LAUNCHED();
  reduce_partials_kernel<<<1, 128, 0, st>>>(w.partial, kMaxGrid, plan.grid, w.sums);
  GTB_LAUNCHED();
  copy_sums_kernel<<<1, 1, 0, st>>>(w.sums, sums);
  GTB_LAUNCHED();
  return GTB_OK;
}
