// Blocked fused passes for multi-orbital Slater-Koster Hamiltonians (
// DESIGN.md sec. 13): K7b (4 orbitals per atom) and K7b9 (9 orbitals) on the scalar ELL expansion.
#include <algorithm>

#include "vecload.cuh"

namespace gtb {
namespace {

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
    // the next column is carried as loaded: any arithmetic on it here would wait for the load at once
    // (ncu on K7m: a quarter of the stall samples sat on the sign extension of the "prefetched" column)
    int32_t craw = K > 0 ? __ldg(cp) : 0;
    for (int k = 0; k < K; ++k) {
      const int64_t j = (int64_t)(craw >> 2);
      const int32_t cnext = k + 1 < K ? __ldg(cp + (size_t)(4 * (k + 1)) * N) : 0;
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
      craw = cnext;
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
    int32_t craw = K > 0 ? __ldg(cp) : 0;   // carried as loaded (see K7b)
    for (int k = 0; k < K; ++k) {
      const int64_t j = (int64_t)(craw / B);
      const int32_t cnext = k + 1 < K ? __ldg(cp + (size_t)(B * (k + 1)) * N) : 0;
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
      craw = cnext;
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

}  // namespace

template <int LOG2T, bool DOT>
void pick_orb_dot(int B, bool diag, bool direct, StepPlan* p) {
  if (B == 4) {
    p->first = diag ? cheb_orb4_kernel<LOG2T, true, true, DOT> : cheb_orb4_kernel<LOG2T, true, false, DOT>;
    p->next = diag ? cheb_orb4_kernel<LOG2T, false, true, DOT> : cheb_orb4_kernel<LOG2T, false, false, DOT>;
  } else if (!direct) {  // block columns through shared memory
    p->first = diag ? cheb_orb9_kernel<LOG2T, true, true, DOT, true> : cheb_orb9_kernel<LOG2T, true, false, DOT, true>;
    p->next = diag ? cheb_orb9_kernel<LOG2T, false, true, DOT, true> : cheb_orb9_kernel<LOG2T, false, false, DOT, true>;
  } else {
    p->first = diag ? cheb_orb9_kernel<LOG2T, true, true, DOT, false> : cheb_orb9_kernel<LOG2T, true, false, DOT, false>;
    p->next = diag ? cheb_orb9_kernel<LOG2T, false, true, DOT, false> : cheb_orb9_kernel<LOG2T, false, false, DOT, false>;
  }
}
template <int LOG2T>
void pick_orb(int B, bool diag, bool dot, bool direct, StepPlan* p) {
  if (dot) pick_orb_dot<LOG2T, true>(B, diag, direct, p);
  else pick_orb_dot<LOG2T, false>(B, diag, direct, p);
}

// K7b plan (B = 4 or 9 orbitals per atom): one thread per (atom, 256-bit element); false when H or R
// does not fit and the scalar kernels must be used
bool make_plan_orb(const gtb_ell* H, int R, int B, bool dot, bool direct, StepPlan* p) {
  if ((B != 4 && B != 9) || H->n % B || H->width % B || H->width == 0 || (R != 2 && R != 4 && R != 8) ||
      (B == 4 && ((reinterpret_cast<uintptr_t>(H->vals) & 31u) || (reinterpret_cast<uintptr_t>(H->diag) & 31u))))
    return false;
  const bool diag = H->diag != nullptr;
  if (R == 2) { pick_orb<0>(B, diag, dot, direct, p); p->T = 1; }
  else if (R == 4) { pick_orb<1>(B, diag, dot, direct, p); p->T = 2; }
  else { pick_orb<2>(B, diag, dot, direct, p); p->T = 4; }
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
  p->grid = std::min(p->grid, kMaxGrid);   // partial-sum rows are kMaxGrid apart
  return true;
}

}  // namespace gtb

