// K7w: the fused Chebyshev pass for WIDE rows with the gathered vector staged in shared memory
// (sliced ELL, 16-bit relative columns decoded in the kernel).
//
// K7t (kpm.cu) stages the ELL slots by TMA but gathers phi_n from global memory: at K = 20 it sits on the L1
// data pipe and on the latency of the gathers that miss L1 (profiles/r01_wide_k7_full.md).  Lattices are
// numbered so that the neighbours of a tile of consecutive rows fall into a few short runs of rows (the tile's
// own row of cells and the two next to it).  gtb_window_ell therefore re-arranges H once, tile by tile
// (T = R / 2 threads per row; TR = 256 / T rows, at R = 8 TR = 128 / T = 32 rows -- tile_threads below):
//   * the distinct row BLOCKS (G rows = 1 KB of phi each) the tile's columns touch, ascending: its window;
//   * every column as a 16-bit index into that window (position of its block x G + row within the block);
//   * the tile's own slot count K_t = longest row of the tile (sliced ELL: padding slots beyond it are dropped);
//   * hoppings, diagonal and the 16-bit columns of the tile contiguous, so a stage is THREE bulk copies
//     instead of 2 K + 1, and H costs 10 bytes per slot instead of 12.
// The pass copies each window block with one cp.async.bulk (1 KB, from L2 after the first tile that needs it)
// next to the tile's H part into a shared-memory stage; the consumers then gather with LDS only -- no tag
// lookup, no miss, ~30 cycles -- in the ELL's own slot order (R = 4: see the builder), so the vectors equal K7's bit for bit wherever
// no padding slot is involved.
// A tile whose columns need more than kMaxBlocks blocks makes the matrix GTB_ERR_NOT_PACKABLE: K7t stays.
#include <algorithm>
#include <type_traits>

#include "tma.cuh"
#include "vecload.cuh"

namespace gtb {
namespace {

constexpr int kWinThreads = 256;
constexpr int kMaxBlocks = 40;          // window blocks per tile (40 KB of phi_n per stage)
constexpr int kBlockBytes = 1024;       // one window block = G rows of phi
constexpr int kHeadBytes = 256;         // per tile: n_blocks, K_t, then the block ids
constexpr int kGlobalHead = 256;        // blob header
constexpr int kWinBarBytes = 128;

struct WinLayout {
  int T, TR, G;              // threads per row, rows per tile, rows per window block
  uint32_t vals_off, diag_off, cols_off, tile_bytes;   // within a tile record (after nothing: head at 0)
  int64_t n_tiles;
};

// Consumer threads per tile and CTAs per SM.  R = 8 takes 32-row tiles (128 consumer threads, four CTAs per SM):
// ncu had the 64-row pass waiting for its stages to fill (profiles/r02_wide_k7w.md), and eight 27 KB stages in
// flight per SM fill more evenly than four 50 KB ones although a smaller tile brings more window per row:
// c2 0.148 -> 0.143 ms.  Measured around it: 128-row tiles (one CTA per SM) 0.186 ms, 16-row tiles (six CTAs)
// 0.159 ms; R = 4 with 64-row tiles 0.96 instead of 0.92 ms at c3 (that pass sits on the shared-memory pipe).
__host__ __device__ constexpr int tile_threads(int R) { return R == 8 ? 128 : kWinThreads; }
__host__ __device__ constexpr int tile_ctas(int R) { return R == 8 ? 4 : 2; }

__host__ __device__ inline WinLayout win_layout(int64_t n, int K, int R, bool diag) {
  WinLayout L;
  L.T = R / 2;
  L.TR = tile_threads(R) / L.T;
  L.G = kBlockBytes / (R * 16);
  L.vals_off = kHeadBytes;
  L.diag_off = L.vals_off + (uint32_t)K * L.TR * 8;
  L.cols_off = L.diag_off + (diag ? L.TR * 8 : 0);
  L.tile_bytes = (L.cols_off + (uint32_t)K * L.TR * 2 + 127) / 128 * 128;
  L.n_tiles = (n + L.TR - 1) / L.TR;
  return L;
}

// ---- build: one CTA per tile ---------------------------------------------------------------------------
constexpr int kSetSize = 2048;
constexpr int kSwapWord = 44;     // tile header word of the swap bits (after n_blocks, K_t, 2 spare words, 40 block ids)
constexpr int kPairSlots = 48;   // widest matrix whose slots are re-ordered for R = 4 (local arrays of the builder)

__global__ void __launch_bounds__(kWinThreads) window_build_kernel(const int32_t* __restrict__ cols,
                                                                   const double* __restrict__ vals,
                                                                   const double* __restrict__ diag, int64_t n,
                                                                   int32_t K, int32_t R,
                                                                   unsigned char* __restrict__ blob,
                                                                   int32_t* __restrict__ flags) {
  const WinLayout L = win_layout(n, K, R, diag != nullptr);
  __shared__ int32_t s_set[kSetSize];
  __shared__ int32_t s_list[kMaxBlocks], s_sorted[kMaxBlocks];
  __shared__ int32_t s_count, s_kt;
  __shared__ uint32_t s_swap[8];   // bit per row of the tile: the row reads the halves of its elements in swapped order
  for (int64_t tile = blockIdx.x; tile < L.n_tiles; tile += gridDim.x) {
    const int64_t row0 = tile * L.TR;
    const int rows = (int)min((int64_t)L.TR, n - row0);
    for (int q = threadIdx.x; q < kSetSize; q += kWinThreads) s_set[q] = -1;
    if (threadIdx.x == 0) {
      s_count = 0;
      s_kt = 0;
    }
    __syncthreads();
    for (int e = threadIdx.x; e < L.TR * K; e += kWinThreads) {
      const int k = e / L.TR, rl = e - k * L.TR;
      if (rl >= rows) continue;
      const int32_t c = cols[(size_t)k * n + row0 + rl];
      if (c == row0 + rl) continue;   // padding slot (a genuine entry never has col = row)
      atomicMax(&s_kt, k + 1);
      const int32_t id = c / L.G;
      uint32_t h = ((uint32_t)id * 2654435761u) & (kSetSize - 1);
      for (int probe = 0; probe < kSetSize; ++probe) {
        const int32_t old = atomicCAS(&s_set[h], -1, id);
        if (old == -1 || old == id) break;
        h = (h + 1) & (kSetSize - 1);
      }
    }
    __syncthreads();
    for (int q = threadIdx.x; q < kSetSize; q += kWinThreads)
      if (s_set[q] >= 0) {
        const int pos = atomicAdd(&s_count, 1);
        if (pos < kMaxBlocks) s_list[pos] = s_set[q];
      }
    __syncthreads();
    const int nb = s_count;
    if (threadIdx.x == 0) atomicMax(flags, nb);   // the largest window sizes the shared-memory stage
    if (nb > kMaxBlocks) {   // the tile's neighbours are too scattered for a window: the matrix stays on K7t
      __syncthreads();
      continue;
    }
    if (threadIdx.x < nb) {  // rank sort (ids are distinct)
      const int32_t mine = s_list[threadIdx.x];
      int rank = 0;
      for (int j = 0; j < nb; ++j) rank += s_list[j] < mine;
      s_sorted[rank] = mine;
    }
    __syncthreads();
    unsigned char* rec = blob + kGlobalHead + (size_t)tile * L.tile_bytes;
    int32_t* head = reinterpret_cast<int32_t*>(rec);
    const int kt = s_kt;
    if (threadIdx.x == 0) {
      head[0] = nb;
      head[1] = kt;
    }
    if (threadIdx.x < kMaxBlocks) head[4 + threadIdx.x] = threadIdx.x < nb ? s_sorted[threadIdx.x] : 0;
    double* tv = reinterpret_cast<double*>(rec + L.vals_off);
    uint16_t* tc = reinterpret_cast<uint16_t*>(rec + L.cols_off);
    for (int e = threadIdx.x; e < L.TR * K; e += kWinThreads) {
      const int k = e / L.TR, rl = e - k * L.TR;
      double v = 0.0;
      uint32_t idx = 0;
      if (rl < rows) {
        const int32_t c = cols[(size_t)k * n + row0 + rl];
        if (c != row0 + rl) {
          v = vals[(size_t)k * n + row0 + rl];
          const int32_t id = c / L.G;
          int lo = 0, hi = nb - 1;
          while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (s_sorted[mid] < id) lo = mid + 1; else hi = mid;
          }
          idx = (uint32_t)(lo * L.G + (c - id * L.G));
        }
      }
      tv[e] = v;
      tc[e] = (uint16_t)idx;
    }
    if (diag) {
      double* td = reinterpret_cast<double*>(rec + L.diag_off);
      for (int rl = threadIdx.x; rl < L.TR; rl += kWinThreads) td[rl] = rl < rows ? diag[row0 + rl] : 0.0;
    }
    __syncthreads();
    // R = 4: a gathered neighbour is 64 bytes = half of the 32 banks, read by the row's two threads with two
    // LDS.128, and a quarter-warp holds four rows.  Two rows that read the same halves of their elements in the
    // same step (the same swap bit) collide whenever their window indices have the same parity: with the fixed
    // pattern "odd rows swap" 45 % of the shared-memory wavefronts of the pass at c3 were such conflicts
    // (profiles/r02_wide_k7w.md).  The order of a row's slots is free, so the two rows sharing a swap bit get their
    // slots re-ordered here until, position by position, one index is even and the other odd; what cannot be
    // matched meets a padding slot (value 0) of the opposite parity while the tile's slot count allows, and only
    // the rest stays same-parity.  The sum over a row's slots then runs in another order than the ELL's: the
    // vectors equal K7t's to rounding, no longer bit for bit.
    // Which two rows of a quarter-warp read the same halves in the same step is the tile's choice (one bit per
    // row in the header, read by the pass): of the three ways to pair four rows the builder takes the one whose
    // slot counts leave the fewest same-parity meetings -- on a lattice the even / odd counts of a row follow its
    // sublattice, and the fixed pairing (rl, rl + 2) met its like in a third of the positions at c3.
    if (threadIdx.x < 8) s_swap[threadIdx.x] = 0xAAAAAAAAu;   // default: odd rows swap (what R = 2 and R = 8 use)
    __syncthreads();
    if (R == 4 && K <= kPairSlots && kt > 0) {
      for (int quad = threadIdx.x; quad < L.TR / 4; quad += kWinThreads) {
        double v4[4][kPairSlots];
        uint16_t i4[4][kPairSlots];
        int ne[4] = {0, 0, 0, 0}, no[4] = {0, 0, 0, 0};
        for (int r = 0; r < 4; ++r)
          for (int k = 0; k < K; ++k) {
            v4[r][k] = tv[k * L.TR + 4 * quad + r];
            i4[r][k] = tc[k * L.TR + 4 * quad + r];
            if (v4[r][k] != 0.0) { if (i4[r][k] & 1) ++no[r]; else ++ne[r]; }
          }
        auto meetings = [&](int x, int y) {   // same-parity positions the slot count forces on the pair (x, y)
          const int n1 = min(ne[x], no[y]), n2 = min(no[x], ne[y]);
          return max(0, (ne[x] + no[x] - n1 - n2) + (ne[y] + no[y] - n1 - n2) - (kt - n1 - n2));
        };
        const int cost0 = meetings(0, 2) + meetings(1, 3), cost1 = meetings(0, 1) + meetings(2, 3),
                  cost2 = meetings(0, 3) + meetings(1, 2);
        int pa[2], pb[2];
        uint32_t bits;   // bit r: row r of the quad swaps its halves; partners share the bit
        if (cost0 <= cost1 && cost0 <= cost2) { pa[0] = 0; pb[0] = 2; pa[1] = 1; pb[1] = 3; bits = 0xAu; }
        else if (cost1 <= cost2) { pa[0] = 0; pb[0] = 1; pa[1] = 2; pb[1] = 3; bits = 0xCu; }
        else { pa[0] = 0; pb[0] = 3; pa[1] = 1; pb[1] = 2; bits = 0x6u; }
        const int word = (4 * quad) >> 5, shift = (4 * quad) & 31;
        atomicAnd(&s_swap[word], ~(0xFu << shift));
        atomicOr(&s_swap[word], bits << shift);
        for (int h = 0; h < 2; ++h) {
          const int ra = pa[h], rb = pb[h];
          const int a = 4 * quad + ra, b = 4 * quad + rb;
          const double *va = v4[ra], *vb = v4[rb];
          const uint16_t *ia = i4[ra], *ib = i4[rb];
          unsigned char ae[kPairSlots], ao[kPairSlots], be[kPairSlots], bo[kPairSlots];
          int nae = 0, nao = 0, nbe = 0, nbo = 0;
          for (int k = 0; k < K; ++k) {
            if (va[k] != 0.0) { if (ia[k] & 1) ao[nao++] = (unsigned char)k; else ae[nae++] = (unsigned char)k; }
            if (vb[k] != 0.0) { if (ib[k] & 1) bo[nbo++] = (unsigned char)k; else be[nbe++] = (unsigned char)k; }
          }
          int pos = 0;
          auto put = [&](int ka, int kb, int pad_a, int pad_b) {   // k < 0: a padding slot of the given parity
            tv[pos * L.TR + a] = ka >= 0 ? va[ka] : 0.0;
            tc[pos * L.TR + a] = ka >= 0 ? ia[ka] : (uint16_t)pad_a;
            tv[pos * L.TR + b] = kb >= 0 ? vb[kb] : 0.0;
            tc[pos * L.TR + b] = kb >= 0 ? ib[kb] : (uint16_t)pad_b;
            ++pos;
          };
          const int n1 = min(nae, nbo), n2 = min(nao, nbe);
          for (int i2 = 0; i2 < n1; ++i2) put(ae[i2], bo[i2], 0, 0);
          for (int i2 = 0; i2 < n2; ++i2) put(ao[i2], be[i2], 0, 0);
          // leftovers: A's (even ones first), B's (even ones first): like meets like only when the count forces it
          unsigned char la[kPairSlots], lb[kPairSlots];
          int nla = 0, nlb = 0;
          for (int i2 = n1; i2 < nae; ++i2) la[nla++] = ae[i2];
          for (int i2 = n2; i2 < nao; ++i2) la[nla++] = ao[i2];
          for (int i2 = n2; i2 < nbe; ++i2) lb[nlb++] = be[i2];
          for (int i2 = n1; i2 < nbo; ++i2) lb[nlb++] = bo[i2];
          const int merges = max(0, nla + nlb - (kt - pos));
          for (int i2 = 0; i2 < merges; ++i2) put(la[i2], lb[i2], 0, 0);
          for (int i2 = merges; i2 < nla; ++i2) put(la[i2], -1, 0, (ia[la[i2]] & 1) ^ 1);
          for (int i2 = merges; i2 < nlb; ++i2) put(-1, lb[i2], (ib[lb[i2]] & 1) ^ 1, 0);
          while (pos < kt) put(-1, -1, 0, 1);
        }
      }
    }
    __syncthreads();
    if (threadIdx.x < 8) head[kSwapWord + threadIdx.x] = (int32_t)s_swap[threadIdx.x];
    __syncthreads();
  }
}


// ---- the pass ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double2 lds_f64x2(uint32_t addr) {
  double2 v;
  asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
  return v;
}

// Rows whose swap bit is set (tile header; the odd rows unless gtb_window_ell chose otherwise at R = 4) keep the
// two complex numbers of their 256-bit element in swapped order in registers:
// the two 16-byte halves of a gathered element are read with two LDS.128, and when the row pair sharing a
// quarter-warp reads opposite halves first, the eight lanes cover all 32 banks (without it: 2-way conflicts,
// twice the shared-memory wavefronts).  The sums over the element do not depend on the order.
template <int VW>
__device__ __forceinline__ Vec<VW> swap_halves(const Vec<VW>& x, bool odd) {
  Vec<VW> r;
  r.v[0] = odd ? x.v[2] : x.v[0];
  r.v[1] = odd ? x.v[3] : x.v[1];
  r.v[2] = odd ? x.v[0] : x.v[2];
  r.v[3] = odd ? x.v[1] : x.v[3];
  return r;
}

// Warp-specialised: the first CT / 32 warps consume (one thread per 256-bit element of the tile), the last warp
// produces.  A stage
// goes round on two mbarriers: full[s] (the copies' bytes) and empty[s] (one arrival per consumer warp once it
// has read the stage), so the consumer warps never wait for one another -- with a __syncthreads per tile and
// warp 0 doubling as producer, ncu showed 5.9 stall cycles per issue on `barrier` and nothing else.
template <int LOG2T, bool kFirst, bool kDiag, int kMode>
__global__ void __launch_bounds__(tile_threads(2 << LOG2T) + 32, tile_ctas(2 << LOG2T))
cheb_window_kernel(const StepArgs a, const int nstages) {
  constexpr int VW = 4;
  constexpr int T = 1 << LOG2T;
  constexpr int R = 2 * T;
  constexpr int CT = tile_threads(R);
  constexpr int kWinCtaThreads = CT + 32;
  constexpr int kConsumerWarps = CT / 32;
  constexpr int TR = CT / T;
  constexpr int G = kBlockBytes / (R * 16);
  constexpr uint32_t kRowBytes = R * 16;
  constexpr int CH = R == 8 ? 4 : 6;   // gathers in flight per chunk (A/B on one box at c2, R = 8: 4 / 5 / 6 / 7 -> 0.138 / 0.141 / 0.141 / 0.141 ms; at c3, R = 4, after the slot re-ordering: 5 / 6 / 9 -> 0.834 / 0.822 / 0.832 ms)
  constexpr bool kDotL = kMode == 1, kAxpy = kMode == 2;
  extern __shared__ __align__(128) unsigned char smem[];
  const int64_t n = a.n;
  const int K = a.width;
  const WinLayout L = win_layout(n, K, R, kDiag);
  const double scale = a.scale, b = a.b;
  const uint32_t stage_bytes = L.tile_bytes + (uint32_t)a.aux * kBlockBytes;   // aux: blocks of the largest window
  const uint32_t bar0 = smem_u32(smem);
  unsigned char* const stage0 = smem + kWinBarBytes;
  const unsigned char* blob = reinterpret_cast<const unsigned char*>(a.vals) + kGlobalHead;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int64_t my_tiles = blockIdx.x < L.n_tiles ? (L.n_tiles - 1 - blockIdx.x) / gridDim.x + 1 : 0;
  const uint32_t empty0 = bar0 + 64;   // full[s] at bar0 + 8 s, empty[s] at bar0 + 64 + 8 s (s < 8)
  if (tid == 0) {
    for (int s = 0; s < nstages; ++s) {
      mbar_init(bar0 + 8 * s, 1);
      mbar_init(empty0 + 8 * s, kConsumerWarps);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // producer state (warp 8): header of the next tile to issue, loaded one tile ahead
  int32_t h_nb = 0, h_kt = 0, h_id0 = 0, h_id1 = 0;
  auto load_head = [&](int64_t i) {
    const int32_t* head = reinterpret_cast<const int32_t*>(blob + (size_t)(blockIdx.x + i * gridDim.x) * L.tile_bytes);
    h_nb = __ldg(head);
    h_kt = __ldg(head + 1);
    h_id0 = lane < kMaxBlocks ? __ldg(head + 4 + lane) : 0;
    h_id1 = lane + 32 < kMaxBlocks ? __ldg(head + 4 + lane + 32) : 0;
  };
  auto issue = [&](int64_t i) {   // all lanes of the producer warp
    const int s = (int)(i % nstages);
    const int64_t tile = blockIdx.x + i * gridDim.x;
    const int64_t row0 = tile * TR;
    const uint32_t rows = (uint32_t)min((int64_t)TR, n - row0);
    const uint32_t bar = bar0 + 8 * s;
    const uint32_t base = smem_u32(stage0 + (size_t)s * stage_bytes);
    const unsigned char* rec = blob + (size_t)tile * L.tile_bytes;
    const int nb = h_nb, kt = h_kt;
    auto block_bytes = [&](int32_t id) { return (uint32_t)min((int64_t)G, n - (int64_t)id * G) * kRowBytes; };
    uint32_t mine = (lane < nb ? block_bytes(h_id0) : 0u) + (lane + 32 < nb ? block_bytes(h_id1) : 0u);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mine += __shfl_xor_sync(0xffffffffu, mine, o);
    const uint32_t head_vals = L.vals_off + (uint32_t)kt * TR * 8;
    const uint32_t cols_bytes = (uint32_t)kt * TR * 2;
    if (lane == 0) mbar_expect_tx(bar, mine + head_vals + (kDiag ? TR * 8 : 0) + cols_bytes);
    __syncwarp();
    if (lane == 0) bulk_g2s(base, rec, head_vals, bar);
    if (lane == 1 && kDiag) bulk_g2s(base + L.diag_off, rec + L.diag_off, TR * 8, bar);
    if (lane == 2 && cols_bytes) bulk_g2s(base + L.cols_off, rec + L.cols_off, cols_bytes, bar);
    if (lane == 3) bulk_prefetch_l2(a.phi_cur + row0 * (T * VW), rows * (T * VW * 8));
    if (lane == 4 && !kFirst) bulk_prefetch_l2(a.phi_io + row0 * (T * VW), rows * (T * VW * 8));
    if (lane == 5 && kDotL) bulk_prefetch_l2(a.dot_with + row0 * (T * VW), rows * (T * VW * 8));
    if (lane == 5 && kAxpy) bulk_prefetch_l2(a.axpy_acc + row0 * (T * VW), rows * (T * VW * 8));
    const uint32_t win = base + L.tile_bytes;
    if (lane < nb)
      bulk_g2s(win + (uint32_t)lane * kBlockBytes, a.phi_cur + (int64_t)h_id0 * G * (T * VW), block_bytes(h_id0), bar);
    if (lane + 32 < nb)
      bulk_g2s(win + (uint32_t)(lane + 32) * kBlockBytes, a.phi_cur + (int64_t)h_id1 * G * (T * VW),
               block_bytes(h_id1), bar);
    if (i + 1 < my_tiles) load_head(i + 1);
  };
  double s1 = 0.0, s2 = 0.0;
  if (wid == kConsumerWarps) {   // ---- producer warp
    if (my_tiles > 0) load_head(0);
    for (int64_t i = 0; i < my_tiles; ++i) {
      if (i >= nstages) mbar_wait(empty0 + 8 * (int)(i % nstages), (uint32_t)(((i / nstages) - 1) & 1));
      issue(i);
    }
    block_store_sums<kWinCtaThreads>(s1, s2, a.partial + blockIdx.x);
    return;
  }
  const int rl = tid >> LOG2T;
  const int t = tid & (T - 1);
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
    const int kt = reinterpret_cast<const int32_t*>(st)[1];
    // the row's swap bit of this tile (gtb_window_ell: rows sharing the bit read the same halves in the same step)
    const bool odd = ((reinterpret_cast<const uint32_t*>(st)[kSwapWord + (rl >> 5)] >> (rl & 31)) & 1u) != 0;
    const uint32_t first_half = odd ? 16u : 0u, second_half = odd ? 0u : 16u;
    const uint16_t* sc = reinterpret_cast<const uint16_t*>(st + L.cols_off) + rl;
    const double* sv = reinterpret_cast<const double*>(st + L.vals_off) + rl;
    const uint32_t win = smem_u32(st) + L.tile_bytes + (uint32_t)t * 32;
    if (live) {
      // kt is the tile's own slot count (uniform over the CTA): whole chunks of CH gathers in flight, then the
      // remainder in chunks of 4, 2, 1 -- no gather is issued for a slot beyond kt (with every chunk padded to CH,
      // kt = 20 cost 24 gathers: a sixth of the shared-memory wavefronts of the pass)
      auto chunk = [&](auto width, int k0) {
        constexpr int N = decltype(width)::value;
        double v[N];
        Vec<VW> x[N];
#pragma unroll
        for (int j = 0; j < N; ++j) {
          const uint32_t c = sc[(k0 + j) * TR];
          v[j] = sv[(k0 + j) * TR];
          const uint32_t at = win + c * kRowBytes;
          const double2 p = lds_f64x2(at + first_half), q2 = lds_f64x2(at + second_half);
          x[j].v[0] = p.x; x[j].v[1] = p.y; x[j].v[2] = q2.x; x[j].v[3] = q2.y;
        }
#pragma unroll
        for (int j = 0; j < N; ++j)
#pragma unroll
          for (int q = 0; q < VW; ++q) acc.v[q] = fma(v[j], x[j].v[q], acc.v[q]);
      };
      int k0 = 0;
      for (; k0 + CH <= kt; k0 += CH) chunk(std::integral_constant<int, CH>{}, k0);
      if (kt - k0 >= 4) { chunk(std::integral_constant<int, 4>{}, k0); k0 += 4; }
      if (kt - k0 >= 2) { chunk(std::integral_constant<int, 2>{}, k0); k0 += 2; }
      if (kt - k0 >= 1) chunk(std::integral_constant<int, 1>{}, k0);
    }
    double dg = 0.0;
    if (kDiag) dg = reinterpret_cast<const double*>(st + L.diag_off)[rl];
    __syncwarp();     // this warp has read stage s: one arrival hands its share back to the producer
    if (lane == 0) mbar_arrive(empty0 + 8 * s);
    if (live) {
      acc = swap_halves<VW>(acc, odd);   // back to memory order
      if (kDiag) {
#pragma unroll
        for (int q = 0; q < VW; ++q) acc.v[q] = fma(dg, own.v[q], acc.v[q]);
      }
      if (kDotL) with = load_stream<VW>(a.dot_with + e * VW);
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
  block_store_sums<kWinCtaThreads>(s1, s2, a.partial + blockIdx.x);
}

template <int LOG2T, int MODE>
void pick_window_mode(bool diag, StepPlan* p) {
  p->tfirst = diag ? cheb_window_kernel<LOG2T, true, true, MODE> : cheb_window_kernel<LOG2T, true, false, MODE>;
  p->tnext = diag ? cheb_window_kernel<LOG2T, false, true, MODE> : cheb_window_kernel<LOG2T, false, false, MODE>;
}
template <int LOG2T>
void pick_window(bool diag, int mode, StepPlan* p) {
  if (mode == 2) pick_window_mode<LOG2T, 2>(diag, p);
  else if (mode == 1) pick_window_mode<LOG2T, 1>(diag, p);
  else pick_window_mode<LOG2T, 0>(diag, p);
}

}  // namespace

// plan of the windowed pass: Wd->n rows, Wd->width = K | blocks of the largest window << 16 | R << 24, Wd->vals =
// the blob of gtb_window_ell built for THIS R (checked), Wd->diag != NULL iff the tiles carry a diagonal.  stages: 0 = default
bool make_plan_window(const gtb_ell* Wd, int R, int mode, int want_stages, StepPlan* p) {
  const int K = Wd->width & 0xffff, blocks = (Wd->width >> 16) & 0xff, built_for = Wd->width >> 24;
  if ((R != 2 && R != 4 && R != 8) || built_for != R || K < 1 || blocks < 0 || blocks > kMaxBlocks || !Wd->vals || mode < 0 ||
      mode > 2 || (reinterpret_cast<uintptr_t>(Wd->vals) & 127u))
    return false;
  const bool diag = Wd->diag != nullptr;
  if (R == 2) { pick_window<0>(diag, mode, p); p->T = 1; }
  else if (R == 4) { pick_window<1>(diag, mode, p); p->T = 2; }
  else { pick_window<2>(diag, mode, p); p->T = 4; }
  p->vw = 4;
  p->block = tile_threads(R) + 32;
  const WinLayout L = win_layout(Wd->n, K, R, diag);
  const size_t stage_bytes = (size_t)L.tile_bytes + (size_t)blocks * kBlockBytes;
  int dev = 0, sms = kSmCount, per_sm = 0, max_smem = 0;
  if (cudaGetDevice(&dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess)
    return false;
  int stages = want_stages > 0 ? std::min(want_stages, 4) : 2;
  while (stages > 1 && kWinBarBytes + stages * stage_bytes > (size_t)max_smem) --stages;
  const size_t smem = kWinBarBytes + stages * stage_bytes;
  if (smem > (size_t)max_smem) return false;
  if (cudaFuncSetAttribute(p->tfirst, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
      cudaFuncSetAttribute(p->tnext, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, p->tnext, p->block, smem) != cudaSuccess)
    return false;
  per_sm = std::max(1, std::min(per_sm, kMaxBlocksPerSm));
  p->grid = (int)std::max<int64_t>(1, std::min<int64_t>(L.n_tiles, (int64_t)sms * per_sm));
  p->grid = std::min(p->grid, kMaxGrid);
  p->stages = stages;
  p->smem = smem;
  return true;
}

}  // namespace gtb

using namespace gtb;

extern "C" size_t gtb_window_bytes(int64_t n, int32_t width, int32_t R, int32_t with_diag) {
  if (n <= 0 || width < 1 || (R != 2 && R != 4 && R != 8)) return 0;
  const WinLayout L = win_layout(n, width, R, with_diag != 0);
  return align_up(kGlobalHead + (size_t)L.n_tiles * L.tile_bytes);
}

extern "C" int gtb_window_ell(const gtb_ell* H, int32_t R, gtb_ell* Wd, int32_t* scratch, void* stream,
                              int32_t* blocks_needed) {
  int rc = check_ell(H);
  if (rc != GTB_OK) return rc;
  if ((R != 2 && R != 4 && R != 8) || !Wd || !scratch || Wd->n != H->n || Wd->width != H->width || !Wd->vals ||
      (reinterpret_cast<uintptr_t>(Wd->vals) & 127u) || H->width < 1)
    return GTB_ERR_INVALID_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const WinLayout L = win_layout(H->n, H->width, R, H->diag != nullptr);
  GTB_CUDA_TRY(cudaMemsetAsync(scratch, 0, sizeof(int32_t), st));
  const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(L.n_tiles, kMaxGrid));
  window_build_kernel<<<grid, kWinThreads, 0, st>>>(H->cols, H->vals, H->diag, H->n, H->width, R,
                                                    reinterpret_cast<unsigned char*>(Wd->vals), scratch);
  GTB_LAUNCHED();
  int32_t worst = 0;
  GTB_CUDA_TRY(cudaMemcpyAsync(&worst, scratch, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  GTB_CUDA_TRY(cudaStreamSynchronize(st));
  if (blocks_needed) *blocks_needed = worst;
  if (worst > kMaxBlocks) return GTB_ERR_NOT_PACKABLE;
  Wd->width = H->width | (worst << 16) | (R << 24);
  Wd->cols = H->cols;   // unused by the pass; kept non-NULL for the argument checks
  Wd->diag = H->diag;
  return GTB_OK;
}
