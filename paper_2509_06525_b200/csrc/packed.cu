// Compressed Hamiltonian stream for narrow rows (fewer bytes per pass than the
// sec. 8(d) bound 12 K + 8 [diag] + 48 R).  For K <= 4 a row of the ELL matrix is packed into ONE 16-byte
// word: per slot a 16-bit column offset relative to the row (ring distance, so periodic wrap-around stays
// small) and a 16-bit index into a dictionary of the distinct hopping values -- lossless, the fp64 values
// themselves are read from the dictionary.  Models with beta = 0 (configs 1, 4, 5: t_ij = t0[s_i][s_j]) have
// a handful of distinct values; config 5 has one.  With K <= 3 the fourth slot carries the dictionary index
// of the onsite energy, so the diagonal array is not streamed either.
//   config 5:  12*3 + 96 = 132  ->  16 + 96 = 112 bytes per atom and pass  (-15 %)
//   config 4:  12*3 + 8 + 384 = 428  ->  16 + 384 = 400                      (-6.5 %)
// A matrix that does not fit (an offset beyond +-32767 rows, more than 65535 distinct values -- any beta != 0
// model) is reported as GTB_ERR_NOT_PACKABLE and stays on the plain path.
// SHORT rows: with K <= 3 and at most 16 distinct values (hoppings and onsite energies together) the row is ONE
// 8-byte word -- three 16-bit offsets and four 4-bit dictionary indices (slot 3: the onsite energy):
//   config 5:  132  ->  8 + 96 = 104 bytes per atom and pass  (-21 %)
// gtb_pack_ell picks the format and says so in P->width (bit 8).
//
// K7x2p is K7x2 (two elements in flight per thread) reading this word: same values, same slot order, same
// arithmetic per element, so the vectors are bit-identical to the plain path's.
#include <algorithm>

#include "vecload.cuh"

namespace gtb {
namespace {

constexpr uint64_t kEmpty = 0xFFFFFFFFFFFFFFFFull;   // a NaN pattern no hopping can carry
constexpr int kHashBits = 17;
constexpr int kHashSize = 1 << kHashBits;            // 2 x the largest dictionary
constexpr int kMaxValues = 65535;
constexpr int kHeaderWords = 32;                     // blob: 32 words of header, then the dictionary
constexpr uint64_t kMagic = 0x4754425041434B31ull;   // "GTBPACK1"
constexpr int kSmemValues = 1024;
constexpr int kShortFlag = 0x100;                   // in P->width: 8-byte rows
constexpr int kShortValues = 16;                    // ... need 4-bit dictionary indices

__device__ __forceinline__ uint32_t hash_slot(uint64_t key) {
  key ^= key >> 33;
  key *= 0xff51afd7ed558ccdull;
  key ^= key >> 33;
  return (uint32_t)key & (kHashSize - 1);
}

// inserts the bit pattern; returns false when the table is full
__device__ bool hash_insert(unsigned long long* table, uint64_t key, int32_t* count) {
  uint32_t s = hash_slot(key);
  for (int probe = 0; probe < kHashSize; ++probe) {
    const unsigned long long cur = table[s];
    if (cur == key) return true;
    if (cur == kEmpty) {
      const unsigned long long old = atomicCAS(table + s, (unsigned long long)kEmpty, (unsigned long long)key);
      if (old == kEmpty) {
        atomicAdd(count, 1);
        return true;
      }
      if (old == key) return true;
    }
    s = (s + 1) & (kHashSize - 1);
  }
  return false;
}

__device__ __forceinline__ int32_t hash_find(const unsigned long long* table, const int32_t* index, uint64_t key) {
  uint32_t s = hash_slot(key);
  for (int probe = 0; probe < kHashSize; ++probe) {
    const unsigned long long cur = table[s];
    if (cur == key) return index[s];
    if (cur == kEmpty) return -1;
    s = (s + 1) & (kHashSize - 1);
  }
  return -1;
}

__global__ void __launch_bounds__(kBlock) hash_init_kernel(unsigned long long* table, int32_t* flags) {
  const int i = blockIdx.x * kBlock + threadIdx.x;
  if (i < kHashSize) table[i] = kEmpty;
  if (i == 0) {
    table[hash_slot(0)] = 0ull;   // +0.0 (the padding value) is always entry 0
    flags[0] = 1;                 // distinct values so far
    flags[1] = 0;                 // 1: offset out of range, 2: too many values
  }
}

// flags[0] = number of distinct bit patterns (until it exceeds the limit), flags[1] |= 2 on overflow
__global__ void __launch_bounds__(kBlock) hash_values_kernel(const double* __restrict__ vals, int64_t count,
                                                             unsigned long long* table, int32_t* flags) {
  for (int64_t e = (int64_t)blockIdx.x * kBlock + threadIdx.x; e < count; e += (int64_t)gridDim.x * kBlock) {
    if (flags[1] & 2) return;
    const uint64_t key = (uint64_t)__double_as_longlong(vals[e]);
    if (key == kEmpty || !hash_insert(table, key, flags) || flags[0] > kMaxValues) atomicOr(flags + 1, 2);
  }
}

// dictionary index per occupied slot; +0.0 gets index 0, the rest in slot order (deterministic): one block,
// each thread counts its run of slots, a block scan places the runs
constexpr int kIndexThreads = 1024;
__global__ void __launch_bounds__(kIndexThreads) hash_index_kernel(const unsigned long long* table, int32_t* index,
                                                                    double* dict) {
  constexpr int kRun = kHashSize / kIndexThreads;
  __shared__ int s_scan[kIndexThreads];
  const int s0 = threadIdx.x * kRun;
  int mine = 0;
  for (int s = s0; s < s0 + kRun; ++s) {
    const unsigned long long key = table[s];
    mine += key != kEmpty && key != 0ull;
  }
  s_scan[threadIdx.x] = mine;
  __syncthreads();
  for (int o = 1; o < kIndexThreads; o <<= 1) {   // inclusive Hillis-Steele scan
    const int v = threadIdx.x >= o ? s_scan[threadIdx.x - o] : 0;
    __syncthreads();
    s_scan[threadIdx.x] += v;
    __syncthreads();
  }
  int next = 1 + s_scan[threadIdx.x] - mine;
  for (int s = s0; s < s0 + kRun; ++s) {
    const unsigned long long key = table[s];
    if (key == kEmpty) continue;
    const int id = key == 0ull ? 0 : next++;
    index[s] = id;
    if (id <= kMaxValues) dict[id] = __longlong_as_double((long long)key);
  }
}

// one thread per row: four (offset, index) pairs; kShort: three offsets and four 4-bit indices in 8 bytes
template <bool kShort>
__global__ void __launch_bounds__(kBlock) pack_rows_kernel(const int32_t* __restrict__ cols,
                                                           const double* __restrict__ vals,
                                                           const double* __restrict__ diag, int64_t n, int32_t K,
                                                           const unsigned long long* __restrict__ table,
                                                           const int32_t* __restrict__ index,
                                                           uint4* __restrict__ rows, int32_t* flags) {
  for (int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x; i < n; i += (int64_t)gridDim.x * kBlock) {
    uint32_t w[4] = {0u, 0u, 0u, 0u};
    for (int k = 0; k < K; ++k) {
      int64_t d = (int64_t)cols[(size_t)k * n + i] - i;   // ring distance in (-n/2, n/2]
      if (2 * d > n) d -= n;
      if (2 * d <= -n) d += n;
      const int32_t id = hash_find(table, index, (uint64_t)__double_as_longlong(vals[(size_t)k * n + i]));
      if (d < -32768 || d > 32767) atomicOr(flags + 1, 1);
      if (id < 0 || id > kMaxValues || (kShort && id >= kShortValues)) atomicOr(flags + 1, 2);
      w[k] = ((uint32_t)id << 16) | ((uint32_t)d & 0xffffu);
    }
    if (diag && K <= 3) {
      const int32_t id = hash_find(table, index, (uint64_t)__double_as_longlong(diag[i]));
      if (id < 0 || id > kMaxValues || (kShort && id >= kShortValues)) atomicOr(flags + 1, 2);
      w[3] = (uint32_t)id << 16;
    }
    if (kShort) {
      const uint32_t ids = (w[0] >> 16) | ((w[1] >> 16) << 4) | ((w[2] >> 16) << 8) | ((w[3] >> 16) << 12);
      reinterpret_cast<uint2*>(rows)[i] = make_uint2((w[0] & 0xffffu) | (w[1] << 16), (w[2] & 0xffffu) | (ids << 16));
    } else {
      rows[i] = make_uint4(w[0], w[1], w[2], w[3]);
    }
  }
}

__global__ void pack_header_kernel(const int32_t* flags, int32_t diag_in_slot, double* blob) {
  unsigned long long* h = reinterpret_cast<unsigned long long*>(blob);
  h[0] = kMagic;
  h[1] = (unsigned long long)flags[0];
  h[2] = (unsigned long long)diag_in_slot;
}

__device__ __forceinline__ uint2 ld_stream_u2(const uint2* p) {
  uint2 v;
  asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
  return v;
}
__device__ __forceinline__ uint4 ld_stream_u4(const uint4* p) {
  uint4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
               : "l"(p));
  return v;
}

// ---- K7x2p ------------------------------------------------------------------------------------------
// kDiagArr: the diagonal is a separate fp64 array (K = 4 with a diagonal); otherwise header word 2 says
// whether slot 3 carries the dictionary index of the onsite energy (K <= 3) or there is no diagonal
// kShort: 8-byte rows (W = 3, no diagonal array)
template <int LOG2T, bool kFirst, bool kDiagArr, int W, int kMode, bool kShort = false>
__global__ void __launch_bounds__(kBlock) cheb_packed_kernel(const StepArgs a) {
  static_assert(!kShort || (W == 3 && !kDiagArr), "short rows: K <= 3, diagonal folded");
  constexpr int VW = 4;
  constexpr int T = 1 << LOG2T;
  constexpr int NE = 2;
  constexpr bool kDotL = kMode == 1, kAxpy = kMode == 2;
  __shared__ double s_dict[kSmemValues];
  const unsigned long long* head = reinterpret_cast<const unsigned long long*>(a.vals);
  const int n_values = (int)head[1];
  const bool folded = W <= 3 && head[2] != 0;
  const double* dict = a.vals + kHeaderWords;
  const bool in_smem = n_values <= kSmemValues;
  if (in_smem)
    for (int q = threadIdx.x; q < n_values; q += kBlock) s_dict[q] = dict[q];
  __syncthreads();
  const int64_t n = a.n;
  const int64_t total = n * T;
  const uint4* rows = reinterpret_cast<const uint4*>(a.cols);
  const double scale = a.scale, b = a.b;
  const int64_t stride = (int64_t)gridDim.x * kBlock;
  double s1 = 0.0, s2 = 0.0;
  for (int64_t e0 = (int64_t)blockIdx.x * kBlock + threadIdx.x; e0 < total; e0 += NE * stride) {
    int64_t e[NE], row[NE];
    bool live[NE];
    Vec<VW> prev[NE], own[NE], with[NE];
    uint4 pk[NE];
#pragma unroll
    for (int r = 0; r < NE; ++r) {
      e[r] = e0 + r * stride;
      live[r] = e[r] < total;
      if (!live[r]) e[r] = e0;   // a harmless duplicate: loaded, never stored or summed
      row[r] = e[r] >> LOG2T;
      if (!kFirst) prev[r] = load_stream<VW>(a.phi_io + e[r] * VW);
      own[r] = load_gather<VW>(a.phi_cur + e[r] * VW);
      if (kDotL) with[r] = load_stream<VW>(a.dot_with + e[r] * VW);
      if (kAxpy) with[r] = load_stream<VW>(a.axpy_acc + e[r] * VW);
      if (kShort) {   // expanded to the long form's four words: the decode below is shared
        const uint2 q = ld_stream_u2(reinterpret_cast<const uint2*>(rows) + row[r]);
        const uint32_t ids = q.y >> 16;
        pk[r] = make_uint4((q.x & 0xffffu) | ((ids & 15u) << 16), (q.x >> 16) | (((ids >> 4) & 15u) << 16),
                           (q.y & 0xffffu) | (((ids >> 8) & 15u) << 16), (ids >> 12) << 16);
      } else {
        pk[r] = ld_stream_u4(rows + row[r]);
      }
    }
    double dg[NE];
#pragma unroll
    for (int r = 0; r < NE; ++r) dg[r] = kDiagArr ? ld_stream_f64(a.diag + row[r]) : 0.0;
    Vec<VW> x[NE][W];
    double v[NE][W];
#pragma unroll
    for (int r = 0; r < NE; ++r) {
      const uint32_t w[4] = {pk[r].x, pk[r].y, pk[r].z, pk[r].w};
      const double* xt = a.phi_cur + (e[r] - row[r] * T) * VW;
#pragma unroll
      for (int k = 0; k < W; ++k) {
        int64_t c = row[r] + (int64_t)(int16_t)(w[k] & 0xffffu);
        c += c < 0 ? n : 0;
        c -= c >= n ? n : 0;
        x[r][k] = load_gather<VW>(xt + c * (T * VW));
        const uint32_t id = w[k] >> 16;
        v[r][k] = in_smem ? s_dict[id] : __ldg(dict + id);
      }
      if (!kDiagArr && folded) {
        const uint32_t id = w[3] >> 16;
        dg[r] = in_smem ? s_dict[id] : __ldg(dict + id);
      }
    }
#pragma unroll
    for (int r = 0; r < NE; ++r) {
      Vec<VW> acc;
#pragma unroll
      for (int q = 0; q < VW; ++q) acc.v[q] = 0.0;
#pragma unroll
      for (int k = 0; k < W; ++k)
#pragma unroll
        for (int q = 0; q < VW; ++q) acc.v[q] = fma(v[r][k], x[r][k].v[q], acc.v[q]);
      if (kDiagArr || folded) {
#pragma unroll
        for (int q = 0; q < VW; ++q) acc.v[q] = fma(dg[r], own[r].v[q], acc.v[q]);
      }
      if (live[r]) {
        Vec<VW> y;
#pragma unroll
        for (int q = 0; q < VW; ++q) {
          y.v[q] = (acc.v[q] - b * own[r].v[q]) * scale;
          if (!kFirst) y.v[q] -= prev[r].v[q];
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
  block_store_sums<kBlock>(s1, s2, a.partial + blockIdx.x);
}

template <int LOG2T, bool DIAG, int W, bool SHORT = false>
void pick_packed_mode(int mode, StepPlan* p) {
  if (mode == 2) {
    p->first = cheb_packed_kernel<LOG2T, true, DIAG, W, 2, SHORT>;
    p->next = cheb_packed_kernel<LOG2T, false, DIAG, W, 2, SHORT>;
  } else if (mode == 1) {
    p->first = cheb_packed_kernel<LOG2T, true, DIAG, W, 1, SHORT>;
    p->next = cheb_packed_kernel<LOG2T, false, DIAG, W, 1, SHORT>;
  } else {
    p->first = cheb_packed_kernel<LOG2T, true, DIAG, W, 0, SHORT>;
    p->next = cheb_packed_kernel<LOG2T, false, DIAG, W, 0, SHORT>;
  }
}

template <int LOG2T>
void pick_packed(bool diag_array, int width, bool short_rows, int mode, StepPlan* p) {
  if (short_rows) pick_packed_mode<LOG2T, false, 3, true>(mode, p);
  else if (width <= 3) pick_packed_mode<LOG2T, false, 3>(mode, p);
  else if (diag_array) pick_packed_mode<LOG2T, true, 4>(mode, p);
  else pick_packed_mode<LOG2T, false, 4>(mode, p);
}

struct PackWs {
  unsigned long long* table;
  int32_t* index;
  int32_t* flags;
  size_t bytes;
};

PackWs carve_pack(void* ws) {
  Carver c(ws);
  PackWs w;
  w.table = c.take<unsigned long long>(kHashSize);
  w.index = c.take<int32_t>(kHashSize);
  w.flags = c.take<int32_t>(16);
  w.bytes = c.off;
  return w;
}

int grid_for(int64_t total) {
  return (int)std::max<int64_t>(1, std::min<int64_t>((total + kBlock - 1) / kBlock, kMaxGrid));
}

}  // namespace

// plan of the packed pass; P->width = K (1..4) | kShortFlag for 8-byte rows, P->diag != NULL only for K = 4 with a
// diagonal
bool make_plan_packed(const gtb_ell* P, int R, int mode, StepPlan* p) {
  const int K = P->width & 0xff;
  const bool short_rows = (P->width & kShortFlag) != 0;
  if ((P->width & ~(0xff | kShortFlag)) || K < 1 || K > 4 || (short_rows && K > 3) || (R != 2 && R != 4 && R != 8) ||
      !P->cols || !P->vals || (reinterpret_cast<uintptr_t>(P->cols) & 15u) || mode < 0 || mode > 2)
    return false;
  if (P->diag && K <= 3) return false;   // gtb_pack_ell folds the diagonal into slot 3 for K <= 3
  const bool diag = P->diag != nullptr;
  if (R == 2) { pick_packed<0>(diag, K, short_rows, mode, p); p->T = 1; }
  else if (R == 4) { pick_packed<1>(diag, K, short_rows, mode, p); p->T = 2; }
  else { pick_packed<2>(diag, K, short_rows, mode, p); p->T = 4; }
  p->vw = 4;
  p->stages = 0;
  p->block = 0;
  p->smem = 0;
  int dev = 0, sms = kSmCount, per_sm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, p->next, kBlock, 0) != cudaSuccess)
    return false;
  per_sm = std::max(1, std::min(per_sm, kMaxBlocksPerSm));
  const int64_t total = P->n * p->T;
  p->grid = (int)std::max<int64_t>(1, std::min<int64_t>((total + kBlock - 1) / kBlock, (int64_t)sms * per_sm));
  p->grid = std::min(p->grid, kMaxGrid);
  return true;
}

}  // namespace gtb

using namespace gtb;

extern "C" size_t gtb_pack_workspace_bytes(void) { return carve_pack(nullptr).bytes; }
extern "C" size_t gtb_packed_rows_bytes(int64_t n) { return n > 0 ? align_up((size_t)n * 16) : 0; }
extern "C" size_t gtb_packed_dict_bytes(void) { return align_up((size_t)(kHeaderWords + kMaxValues + 1) * 8); }

extern "C" int gtb_pack_ell(const gtb_ell* H, gtb_ell* P, void* ws, size_t ws_bytes, void* stream,
                            int32_t* n_values) {
  int rc = check_ell(H);
  if (rc != GTB_OK) return rc;
  if (!P || P->n != H->n || P->width != H->width || !P->cols || !P->vals ||
      (reinterpret_cast<uintptr_t>(P->cols) & 15u) || (reinterpret_cast<uintptr_t>(P->vals) & 15u))
    return GTB_ERR_INVALID_ARG;
  if (H->width < 1 || H->width > 4) return GTB_ERR_NOT_PACKABLE;
  rc = check_ws(ws, ws_bytes, gtb_pack_workspace_bytes());
  if (rc != GTB_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const PackWs w = carve_pack(ws);
  const int64_t n = H->n;
  const bool fold_diag = H->diag && H->width <= 3;
  hash_init_kernel<<<kHashSize / kBlock, kBlock, 0, st>>>(w.table, w.flags);
  GTB_LAUNCHED();
  hash_values_kernel<<<grid_for(n * H->width), kBlock, 0, st>>>(H->vals, n * H->width, w.table, w.flags);
  GTB_LAUNCHED();
  if (fold_diag) {
    hash_values_kernel<<<grid_for(n), kBlock, 0, st>>>(H->diag, n, w.table, w.flags);
    GTB_LAUNCHED();
  }
  int32_t flags[2] = {0, 0};
  GTB_CUDA_TRY(cudaMemcpyAsync(flags, w.flags, sizeof(flags), cudaMemcpyDeviceToHost, st));
  GTB_CUDA_TRY(cudaStreamSynchronize(st));
  if (flags[1] || flags[0] > kMaxValues) return GTB_ERR_NOT_PACKABLE;
  const bool short_rows = H->width <= 3 && flags[0] <= kShortValues;
  hash_index_kernel<<<1, kIndexThreads, 0, st>>>(w.table, w.index, P->vals + kHeaderWords);
  GTB_LAUNCHED();
  if (short_rows)
    pack_rows_kernel<true><<<grid_for(n), kBlock, 0, st>>>(H->cols, H->vals, fold_diag ? H->diag : nullptr, n, H->width,
                                                          w.table, w.index, reinterpret_cast<uint4*>(P->cols), w.flags);
  else
    pack_rows_kernel<false><<<grid_for(n), kBlock, 0, st>>>(H->cols, H->vals, fold_diag ? H->diag : nullptr, n, H->width,
                                                           w.table, w.index, reinterpret_cast<uint4*>(P->cols), w.flags);
  GTB_LAUNCHED();
  pack_header_kernel<<<1, 1, 0, st>>>(w.flags, fold_diag ? 1 : 0, P->vals);
  GTB_LAUNCHED();
  GTB_CUDA_TRY(cudaMemcpyAsync(flags, w.flags, sizeof(flags), cudaMemcpyDeviceToHost, st));
  GTB_CUDA_TRY(cudaStreamSynchronize(st));
  if (flags[1]) return GTB_ERR_NOT_PACKABLE;
  P->diag = fold_diag ? nullptr : H->diag;
  P->width = H->width | (short_rows ? kShortFlag : 0);
  if (n_values) *n_values = flags[0];
  return GTB_OK;
}
