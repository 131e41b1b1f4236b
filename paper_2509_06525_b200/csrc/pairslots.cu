// gtb_pair_slots: the SAME matrix as a plain ELL whose rows keep their entries in another slot order.
//
// With R = 4 vectors per pass a gathered neighbour is 64 bytes: half of a 128-byte L1 line.  The fused passes
// that gather from global memory (K7, K7x2, K7t) give a row to two threads (32 bytes each), and the L1 data stage
// serves 128 bytes per wavefront: the gathers of rows 2q and 2q + 1 go out together when the two columns differ
// in parity (address bit 6) and one after the other when they do not.  ncu on K7t at config 3b (K = 11, R = 4):
// 14.6 L1 wavefronts per 256-bit gather request where 8 are needed, l1tex__data_pipe_lsu_wavefronts at 82 %
// (profiles/r02_k7t.md).  The order of a row's slots is free, so this pass re-orders the slots of each such pair
// of rows until, position by position, one column is even and the other odd; padding slots keep (column = the row
// itself, value 0), so row 2q pads even and row 2q + 1 pads odd.  The result is an ordinary gtb_ell of the same
// matrix: every kernel takes it, the sums over a row run in the new order (equal to the plain order's to rounding).
// The windowed form (window.cu) does the same for its shared-memory gathers.
#include <algorithm>

#include "cheb.cuh"

namespace gtb {
namespace {

constexpr int kPairMaxSlots = 48;   // local arrays of the kernel; wider matrices are copied unchanged

__global__ void __launch_bounds__(kBlock) pair_slots_kernel(const int32_t* __restrict__ cols,
                                                            const double* __restrict__ vals, int64_t n, int32_t K,
                                                            int32_t* __restrict__ ocols, double* __restrict__ ovals) {
  const int64_t pairs = (n + 1) / 2;
  for (int64_t p = (int64_t)blockIdx.x * kBlock + threadIdx.x; p < pairs; p += (int64_t)gridDim.x * kBlock) {
    const int64_t a = 2 * p, b = 2 * p + 1;
    const bool has_b = b < n;
    int32_t ca[kPairMaxSlots], cb[kPairMaxSlots];
    double va[kPairMaxSlots], vb[kPairMaxSlots];
    unsigned char ae[kPairMaxSlots], ao[kPairMaxSlots], be[kPairMaxSlots], bo[kPairMaxSlots];
    int nae = 0, nao = 0, nbe = 0, nbo = 0;
    for (int k = 0; k < K; ++k) {
      ca[k] = cols[(size_t)k * n + a];
      va[k] = vals[(size_t)k * n + a];
      if (ca[k] != (int32_t)a) { if (ca[k] & 1) ao[nao++] = (unsigned char)k; else ae[nae++] = (unsigned char)k; }
      if (has_b) {
        cb[k] = cols[(size_t)k * n + b];
        vb[k] = vals[(size_t)k * n + b];
        if (cb[k] != (int32_t)b) { if (cb[k] & 1) bo[nbo++] = (unsigned char)k; else be[nbe++] = (unsigned char)k; }
      }
    }
    int pos = 0;
    auto put = [&](int ka, int kb) {   // k < 0: a padding slot
      ocols[(size_t)pos * n + a] = ka >= 0 ? ca[ka] : (int32_t)a;
      ovals[(size_t)pos * n + a] = ka >= 0 ? va[ka] : 0.0;
      if (has_b) {
        ocols[(size_t)pos * n + b] = kb >= 0 ? cb[kb] : (int32_t)b;
        ovals[(size_t)pos * n + b] = kb >= 0 ? vb[kb] : 0.0;
      }
      ++pos;
    };
    // a is an even row (its padding column is even), b an odd one
    const int n1 = min(nae, nbo), n2 = min(nao, nbe);
    for (int i = 0; i < n1; ++i) put(ae[i], bo[i]);
    for (int i = 0; i < n2; ++i) put(ao[i], be[i]);
    // What is left on both sides has found no partner of the other parity.  A's even ones and B's odd ones are
    // harmless against the other row's padding (B pads odd, A pads even); A's odd ones and B's even ones meet
    // their like whatever stands opposite (the count of such positions is fixed by the rows, not by the order).
    unsigned char la[kPairMaxSlots], lb[kPairMaxSlots];
    int nla = 0, nlb = 0;
    for (int i = n1; i < nae; ++i) la[nla++] = ae[i];
    for (int i = n2; i < nao; ++i) la[nla++] = ao[i];
    for (int i = n1; i < nbo; ++i) lb[nlb++] = bo[i];
    for (int i = n2; i < nbe; ++i) lb[nlb++] = be[i];
    const int m = max(nla, nlb);
    for (int i = 0; i < m; ++i) put(i < nla ? la[i] : -1, i < nlb ? lb[i] : -1);
    while (pos < K) put(-1, -1);
  }
}

// R = 2: a gathered neighbour is 32 bytes, a quarter of a line, and a row has one thread: the gathers of rows
// 4q .. 4q + 3 share one L1 wavefront when their columns differ in the two low bits (address bits 5 and 6).  In the
// sorted slot order of a honeycomb lattice they almost never do (2.4 % of the positions at config 5); one
// permutation of each row's slots, chosen row by row, makes them all differ.  K <= 4: every permutation is tried.
constexpr int kQuadMaxSlots = 4;

__device__ __forceinline__ void unrank_permutation(int rank, int K, int* perm) {   // lexicographic, K <= 4
  int pool[kQuadMaxSlots] = {0, 1, 2, 3};
  int f = 1;
  for (int i = 2; i < K; ++i) f *= i;   // (K - 1)!
  for (int i = 0; i < K; ++i) {
    const int pick = rank / f;
    rank -= pick * f;
    perm[i] = pool[pick];
    for (int j = pick; j < K - 1 - i; ++j) pool[j] = pool[j + 1];
    if (K - 1 - i > 0) f /= (K - 1 - i);
  }
}

__global__ void __launch_bounds__(kBlock) quad_slots_kernel(const int32_t* __restrict__ cols,
                                                            const double* __restrict__ vals, int64_t n, int32_t K,
                                                            int32_t* __restrict__ ocols, double* __restrict__ ovals) {
  const int64_t quads = (n + 3) / 4;
  int nperm = 1;
  for (int i = 2; i <= K; ++i) nperm *= i;
  for (int64_t q = (int64_t)blockIdx.x * kBlock + threadIdx.x; q < quads; q += (int64_t)gridDim.x * kBlock) {
    int32_t c[4][kQuadMaxSlots];
    double v[4][kQuadMaxSlots];
    int chosen[4][kQuadMaxSlots];
    const int rows = (int)min((int64_t)4, n - 4 * q);
    for (int r = 0; r < rows; ++r)
      for (int k = 0; k < K; ++k) {
        c[r][k] = cols[(size_t)k * n + 4 * q + r];
        v[r][k] = vals[(size_t)k * n + 4 * q + r];
      }
    for (int k = 0; k < K; ++k) chosen[0][k] = k;
    for (int r = 1; r < rows; ++r) {   // the permutation of row r that clashes least with the rows before it
      int best = 1 << 30, best_rank = 0;
      for (int rank = 0; rank < nperm; ++rank) {
        int perm[kQuadMaxSlots];
        unrank_permutation(rank, K, perm);
        int clashes = 0;
        for (int k = 0; k < K; ++k) {
          const int mine = c[r][perm[k]] & 3;
          for (int j = 0; j < r; ++j) clashes += (c[j][chosen[j][k]] & 3) == mine;
        }
        if (clashes < best) { best = clashes; best_rank = rank; }
      }
      unrank_permutation(best_rank, K, chosen[r]);
    }
    for (int r = 0; r < rows; ++r)
      for (int k = 0; k < K; ++k) {
        ocols[(size_t)k * n + 4 * q + r] = c[r][chosen[r][k]];
        ovals[(size_t)k * n + 4 * q + r] = v[r][chosen[r][k]];
      }
  }
}

// R = 2, wider rows (neighbour lists of the s,p,d bond form: K = 12): position by position the four rows of a quad
// take entries whose columns differ in their two low bits -- of the 24 ways to hand the four residues to the four
// rows the one that most rows can serve (ties: from the fullest piles); a row that cannot serve takes what it has.
__global__ void __launch_bounds__(kBlock) quad_greedy_kernel(const int32_t* __restrict__ cols,
                                                             const double* __restrict__ vals, int64_t n, int32_t K,
                                                             int32_t* __restrict__ ocols, double* __restrict__ ovals) {
  const int64_t quads = (n + 3) / 4;
  for (int64_t q = (int64_t)blockIdx.x * kBlock + threadIdx.x; q < quads; q += (int64_t)gridDim.x * kBlock) {
    int32_t c[4][kPairMaxSlots];
    unsigned long long used[4] = {0ull, 0ull, 0ull, 0ull};
    int count[4][4];
    const int rows = (int)min((int64_t)4, n - 4 * q);
    for (int r = 0; r < 4; ++r)
      for (int m = 0; m < 4; ++m) count[r][m] = 0;
    for (int r = 0; r < rows; ++r)
      for (int k = 0; k < K; ++k) {
        c[r][k] = cols[(size_t)k * n + 4 * q + r];
        ++count[r][c[r][k] & 3];
      }
    for (int pos = 0; pos < K; ++pos) {
      int best_served = -1, best_pile = -1, best_rank = 0;
      for (int rank = 0; rank < 24; ++rank) {
        int perm[4];
        unrank_permutation(rank, 4, perm);
        int served = 0, pile = 0;
        for (int r = 0; r < rows; ++r) {
          const int have = count[r][perm[r]];
          served += have > 0;
          pile += have;
        }
        if (served > best_served || (served == best_served && pile > best_pile)) {
          best_served = served; best_pile = pile; best_rank = rank;
        }
      }
      int perm[4];
      unrank_permutation(best_rank, 4, perm);
      for (int r = 0; r < rows; ++r) {
        int pick = -1;
        for (int k = 0; k < K && pick < 0; ++k)
          if (!((used[r] >> k) & 1ull) && (c[r][k] & 3) == perm[r]) pick = k;
        for (int k = 0; k < K && pick < 0; ++k)
          if (!((used[r] >> k) & 1ull)) pick = k;
        used[r] |= 1ull << pick;
        --count[r][c[r][pick] & 3];
        ocols[(size_t)pos * n + 4 * q + r] = c[r][pick];
        ovals[(size_t)pos * n + 4 * q + r] = vals[(size_t)pick * n + 4 * q + r];
      }
    }
  }
}

__global__ void __launch_bounds__(kBlock) copy_slots_kernel(const int32_t* __restrict__ cols,
                                                            const double* __restrict__ vals, int64_t count,
                                                            int32_t* __restrict__ ocols, double* __restrict__ ovals) {
  for (int64_t e = (int64_t)blockIdx.x * kBlock + threadIdx.x; e < count; e += (int64_t)gridDim.x * kBlock) {
    ocols[e] = cols[e];
    ovals[e] = vals[e];
  }
}

}  // namespace
}  // namespace gtb

using namespace gtb;

extern "C" int gtb_pair_slots(const gtb_ell* H, int32_t R, gtb_ell* Hp, void* stream) {
  int rc = check_ell(H);
  if (rc != GTB_OK) return rc;
  if (!Hp || Hp->n != H->n || Hp->width != H->width || R < 1 || (H->width > 0 && (!Hp->cols || !Hp->vals)) ||
      Hp->cols == H->cols || Hp->vals == H->vals)
    return GTB_ERR_INVALID_ARG;
  Hp->diag = H->diag;
  if (H->width == 0) return GTB_OK;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int64_t n = H->n;
  if (R == 4 && H->width <= kPairMaxSlots) {
    const int64_t pairs = (n + 1) / 2;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((pairs + kBlock - 1) / kBlock, kMaxGrid));
    pair_slots_kernel<<<grid, kBlock, 0, st>>>(H->cols, H->vals, n, H->width, Hp->cols, Hp->vals);
  } else if (R == 2 && H->width <= kQuadMaxSlots) {
    const int64_t quads = (n + 3) / 4;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((quads + kBlock - 1) / kBlock, kMaxGrid));
    quad_slots_kernel<<<grid, kBlock, 0, st>>>(H->cols, H->vals, n, H->width, Hp->cols, Hp->vals);
  } else if (R == 2 && H->width <= kPairMaxSlots) {
    const int64_t quads = (n + 3) / 4;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((quads + kBlock - 1) / kBlock, kMaxGrid));
    quad_greedy_kernel<<<grid, kBlock, 0, st>>>(H->cols, H->vals, n, H->width, Hp->cols, Hp->vals);
  } else {   // nothing to gain (R = 8 gathers whole lines) or too wide for the kernel's local arrays: a copy
    const int64_t count = n * H->width;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((count + kBlock - 1) / kBlock, kMaxGrid));
    copy_slots_kernel<<<grid, kBlock, 0, st>>>(H->cols, H->vals, count, Hp->cols, Hp->vals);
  }
  GTB_LAUNCHED();
  return GTB_OK;
}
