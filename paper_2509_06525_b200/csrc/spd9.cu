// s,p,d Slater-Koster Hamiltonians at the paper's scale (PAPER.md:96 "s, p, d orbital basis", :106 "over
// 100 million atoms (approximately 1 billion orbitals)", Fig. 4a :192): two representations of the same
// operator that gtb_spd_hamiltonian writes as a scalar ELL matrix, and the fused Chebyshev pass on each.
//
//   blocks (GTB_MODE_BLOCK9, K7bb):  cols int32 [K][n], blocks double [K][81][n] (entry 9 nu + mu, atom
//       fastest: a warp's loads of one entry are one contiguous run), onsite double [9][n].  652 K bytes
//       per atom instead of the scalar form's 972 K, no dead column copies, every load coalesced.
//   bonds  (GTB_MODE_BOND9, K7m):    cols int32 [K][n] and one record (x, y, z, species) per atom; the pass
//       rebuilds each pair's action from the bond vector and the species pair's integrals in registers:
//       H costs 4 K + 40 bytes per atom, so 10^8 atoms x 9 orbitals fit one 180 GB B200.
//
// The two-centre integrals are diagonal in the bond frame (reading S4).  Summing the
// frame out in closed form gives, with u = (l, m, n) the bond direction, D_a = u^T A_a u and G_a = A_a u
// for the five d orbitals (A_a the quadratic forms of reading S4):
//   E_ss = V_ss;   E_{s,pb} = V_sp u_b;   E_{s,db} = V_sd D_b;
//   E_{pa,s} = -V'_sp u_a;   E_{pa,pb} = V_ppp d_ab + (V_pps - V_ppp) u_a u_b;
//   E_{pa,db} = (V_pds - k V_pdp) u_a D_b + k V_pdp G_{b,a},   k = 2/sqrt3;
//   E_{da,s} = V'_sd D_a;   E_{da,pb} = -(V'_pds - k V'_pdp) D_a u_b - k V'_pdp G_{a,b};
//   E_{da,db} = V_ddd d_ab + (V_dds - 4/3 V_ddp + 1/3 V_ddd) D_a D_b + 4/3 (V_ddp - V_ddd) G_a . G_b,
// V of the pair (s_i, s_j), V' of (s_j, s_i) (the l_a > l_b elements belong to the (j, i)
// block).  Applied to a vector these are 64 FMAs per real component instead of 81 for a stored block.
#include <algorithm>
#include <cmath>

#include "spd_pair.cuh"
#include "vecload.cuh"

namespace gtb {
namespace {

constexpr size_t kBondHeaderBytes = 8192;

struct BondHeader {
  double box[3];
  double r0, beta;
  int32_t pbc[3];
  int32_t n_species;
  int64_t n;
  double onsite[3][GTB_MAX_SPECIES];                        // s, p, d
  double coef[GTB_MAX_SPECIES * GTB_MAX_SPECIES][kNc];      // see pair_coefficients
};
static_assert(sizeof(BondHeader) <= kBondHeaderBytes, "bond header");

// bond i -> j with the minimum image; the same evaluation order as the assembly kernels
__device__ __forceinline__ Geometry bond_geometry(const double pi[3], const double pj[3],
                                                  const double* box, const int32_t* pbc, double r0,
                                                  double beta) {
  double d[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    d[a] = __dsub_rn(pj[a], pi[a]);
    if (pbc[a]) d[a] = __dsub_rn(d[a], __dmul_rn(box[a], rint(__ddiv_rn(d[a], box[a]))));
  }
  const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2]));
  const double r = sqrt(r2);
  const double inv = 1.0 / r;
  Geometry g;
  g.l = d[0] * inv;
  g.m = d[1] * inv;
  g.n = d[2] * inv;
  g.f = beta == 0.0 ? 1.0 : exp(-beta * (r / r0 - 1.0));
  return g;
}

__device__ __forceinline__ Vec<4> ld_rec(const double* p) {   // 32-byte atom record, read-only path
  return load_gather<4>(p);
}

// ---- assembly ---------------------------------------------------------------------------------------
// bond records: posw[i] = (x, y, z, species), shift[i]
__global__ void __launch_bounds__(kBlock) bond_record_kernel(int64_t n, const double* __restrict__ pos,
                                                             const int32_t* __restrict__ species,
                                                             const double* __restrict__ shift_in,
                                                             int32_t n_species, double* __restrict__ posw,
                                                             double* __restrict__ shift,
                                                             int32_t* __restrict__ status) {
  for (int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x; i < n; i += (int64_t)gridDim.x * kBlock) {
    const int s = species[i];
    if (s < 0 || s >= n_species) atomicOr(status, 1);
    posw[4 * i + 0] = pos[3 * i + 0];
    posw[4 * i + 1] = pos[3 * i + 1];
    posw[4 * i + 2] = pos[3 * i + 2];
    posw[4 * i + 3] = (double)min(max(s, 0), n_species - 1);
    shift[i] = shift_in ? shift_in[i] : 0.0;
  }
}

// one thread per (atom, neighbour slot): the block of the pair into blocks[k][9 nu + mu][i]
__global__ void __launch_bounds__(128) block9_assemble_kernel(const int32_t* __restrict__ cols, int64_t n,
                                                              int32_t K, const double* __restrict__ bond,
                                                              double* __restrict__ blocks) {
  const BondHeader& h = *reinterpret_cast<const BondHeader*>(bond);
  const double* posw = bond + kBondHeaderBytes / 8;
  const int64_t total = n * K;
  for (int64_t e = (int64_t)blockIdx.x * 128 + threadIdx.x; e < total; e += (int64_t)gridDim.x * 128) {
    const int64_t k = e / n;
    const int64_t i = e - k * n;
    const int64_t j = cols[e];
    double E[9][9];
    if (j == i) {   // padding slot
      for (int mu = 0; mu < 9; ++mu)
        for (int nu = 0; nu < 9; ++nu) E[mu][nu] = 0.0;
    } else {
      const Vec<4> pi = ld_rec(posw + 4 * i), pj = ld_rec(posw + 4 * j);
      const Geometry g = bond_geometry(pi.v, pj.v, h.box, h.pbc, h.r0, h.beta);
      const double* c0 = h.coef[(int)pi.v[3] * h.n_species + (int)pj.v[3]];
      double c[kNc];
      for (int q = 0; q < kNc; ++q) c[q] = c0[q] * g.f;
      pair_block(g, c, E);
    }
    double* out = blocks + (size_t)k * 81 * n + i;
    for (int nu = 0; nu < 9; ++nu)
      for (int mu = 0; mu < 9; ++mu) out[(size_t)(9 * nu + mu) * n] = E[mu][nu];
  }
}

// onsite[mu][i] = eps_{l(mu)}[s_i] + shift_i
__global__ void __launch_bounds__(kBlock) onsite9_kernel(int64_t n, const double* __restrict__ bond,
                                                         double* __restrict__ onsite) {
  const BondHeader& h = *reinterpret_cast<const BondHeader*>(bond);
  const double* posw = bond + kBondHeaderBytes / 8;
  const double* shift = posw + 4 * n;
  for (int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x; i < n; i += (int64_t)gridDim.x * kBlock) {
    const int s = (int)posw[4 * i + 3];
    const double sh = shift[i];
    for (int mu = 0; mu < 9; ++mu) onsite[(size_t)mu * n + i] = h.onsite[mu == 0 ? 0 : (mu < 4 ? 1 : 2)][s] + sh;
  }
}

// Gershgorin interval of the orbital matrix from either representation (rows = atoms x 9):
// kBond: blocks rebuilt from the bond records; else read from the stored blocks
template <bool kBond>
__global__ void __launch_bounds__(128) bounds9_kernel(const int32_t* __restrict__ cols, int64_t n, int32_t K,
                                                      const double* __restrict__ bond_or_blocks,
                                                      const double* __restrict__ onsite,
                                                      double* __restrict__ partial) {
  double lo = INFINITY, hi = -INFINITY;
  for (int64_t i = (int64_t)blockIdx.x * 128 + threadIdx.x; i < n; i += (int64_t)gridDim.x * 128) {
    double off[9];
    for (int mu = 0; mu < 9; ++mu) off[mu] = 0.0;
    double eps[9];
    if (kBond) {
      const BondHeader& h = *reinterpret_cast<const BondHeader*>(bond_or_blocks);
      const double* posw = bond_or_blocks + kBondHeaderBytes / 8;
      const Vec<4> pi = ld_rec(posw + 4 * i);
      for (int k = 0; k < K; ++k) {
        const int64_t j = cols[(size_t)k * n + i];
        if (j == i) continue;
        const Vec<4> pj = ld_rec(posw + 4 * j);
        const Geometry g = bond_geometry(pi.v, pj.v, h.box, h.pbc, h.r0, h.beta);
        const double* c0 = h.coef[(int)pi.v[3] * h.n_species + (int)pj.v[3]];
        double c[kNc];
        for (int q = 0; q < kNc; ++q) c[q] = c0[q] * g.f;
        double E[9][9];
        pair_block(g, c, E);
        for (int mu = 0; mu < 9; ++mu)
          for (int nu = 0; nu < 9; ++nu) off[mu] += fabs(E[mu][nu]);
      }
      const double sh = posw[4 * n + i];
      for (int mu = 0; mu < 9; ++mu) eps[mu] = h.onsite[mu == 0 ? 0 : (mu < 4 ? 1 : 2)][(int)pi.v[3]] + sh;
    } else {
      for (int k = 0; k < K; ++k)
        for (int nu = 0; nu < 9; ++nu)
          for (int mu = 0; mu < 9; ++mu)
            off[mu] += fabs(bond_or_blocks[((size_t)k * 81 + 9 * nu + mu) * n + i]);
      for (int mu = 0; mu < 9; ++mu) eps[mu] = onsite ? onsite[(size_t)mu * n + i] : 0.0;
    }
    for (int mu = 0; mu < 9; ++mu) {
      lo = fmin(lo, eps[mu] - off[mu]);
      hi = fmax(hi, eps[mu] + off[mu]);
    }
  }
  __shared__ double s[4][2];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  lo = warp_min(lo);
  hi = warp_max(hi);
  if (lane == 0) {
    s[wid][0] = lo;
    s[wid][1] = hi;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 4; ++w) {
      lo = fmin(lo, s[w][0]);
      hi = fmax(hi, s[w][1]);
    }
    partial[2 * blockIdx.x + 0] = lo;
    partial[2 * blockIdx.x + 1] = hi;
  }
}

__global__ void bounds9_final_kernel(const double* partial, int blocks, double* lo_hi) {
  if (threadIdx.x == 0) {
    double lo = partial[0], hi = partial[1];
    for (int b = 1; b < blocks; ++b) {
      lo = fmin(lo, partial[2 * b]);
      hi = fmax(hi, partial[2 * b + 1]);
    }
    lo_hi[0] = lo;
    lo_hi[1] = hi;
  }
}

// ---- the fused pass, shared epilogue -------------------------------------------------------------------
// thread = (atom i, one 256-bit element t); the vectors are orbital rows 9 i + mu, [9 n][R][2], as everywhere.
// (An orbital-major layout [9][n][R][2] for the library's own vectors was built and measured: the gathers of
// consecutive atoms do not share cache lines on these lattices -- same-sublattice atoms are 4 apart -- and
// nine separate row streams per array cost more than they save: 2.44 -> 3.20 ms at K = 3, 6.27 -> 6.92 ms
// at K = 12 for 1.02e7 atoms, R = 2; removed.)
template <int LOG2T>
__device__ __forceinline__ int64_t vec_off(int64_t i, int mu) {   // in 256-bit elements, before t
  return (9 * i + mu) << LOG2T;
}

template <int VW, int LOG2T, bool kFirst, bool kDotL>
__device__ __forceinline__ void epilogue9(const StepArgs& a, int64_t i, int64_t t,
                                          const Vec<VW> (&acc)[9], const double (&eps)[9], double& s1,
                                          double& s2) {
  const double scale = a.scale, b = a.b;
#pragma unroll
  for (int mu = 0; mu < 9; ++mu) {
    const int64_t at = (vec_off<LOG2T>(i, mu) + t) * VW;
    const Vec<VW> own = load_gather<VW>(a.phi_cur + at);
    Vec<VW> prev, with;
    if (!kFirst) prev = load_stream<VW>(a.phi_io + at);
    if (kDotL) with = load_stream<VW>(a.dot_with + at);
    Vec<VW> y;
#pragma unroll
    for (int q = 0; q < VW; ++q) {
      const double hx = fma(eps[mu], own.v[q], acc[mu].v[q]);
      y.v[q] = (hx - b * own.v[q]) * scale;
      if (!kFirst) y.v[q] -= prev.v[q];
      s1 = fma(own.v[q], kDotL ? with.v[q] : own.v[q], s1);
      s2 = fma(y.v[q], kDotL ? with.v[q] : own.v[q], s2);
    }
    store_stream<VW>(a.phi_io + at, y);
  }
}

// ---- K7bb: stored blocks [K][81][n] ----------------------------------------------------------------------
constexpr int kBlock9Threads = 256;

template <int LOG2T, bool kFirst, bool kDotL>
__global__ void __launch_bounds__(kBlock9Threads, 2) cheb_block9_kernel(const StepArgs a) {
  constexpr int VW = 4;
  constexpr int T = 1 << LOG2T;
  const int64_t n = a.n / 9;   // atoms
  const int K = a.width;
  const int64_t total = n * T;
  double s1 = 0.0, s2 = 0.0;
  for (int64_t e = (int64_t)blockIdx.x * kBlock9Threads + threadIdx.x; e < total;
       e += (int64_t)gridDim.x * kBlock9Threads) {
    const int64_t i = e >> LOG2T;
    const int64_t t = e - i * T;
    const double* xt = a.phi_cur + t * VW;
    Vec<VW> acc[9];
#pragma unroll
    for (int mu = 0; mu < 9; ++mu)
#pragma unroll
      for (int q = 0; q < VW; ++q) acc[mu].v[q] = 0.0;
    int32_t craw = K > 0 ? ld_stream_i32(a.cols + i) : 0;   // carried as loaded (see K7m below)
    for (int k = 0; k < K; ++k) {
      const int64_t j = craw;
      const int32_t cnext = k + 1 < K ? ld_stream_i32(a.cols + (size_t)(k + 1) * n + i) : 0;
      const double* blk = a.vals + (size_t)k * 81 * n + i;
#pragma unroll 3
      for (int nu = 0; nu < 9; ++nu) {
        double hcol[9];
#pragma unroll
        for (int mu = 0; mu < 9; ++mu) hcol[mu] = ld_stream_f64(blk + (size_t)(9 * nu + mu) * n);
        const Vec<VW> x = load_gather<VW>(xt + vec_off<LOG2T>(j, nu) * VW);
#pragma unroll
        for (int mu = 0; mu < 9; ++mu)
#pragma unroll
          for (int q = 0; q < VW; ++q) acc[mu].v[q] = fma(hcol[mu], x.v[q], acc[mu].v[q]);
      }
      craw = cnext;
    }
    double eps[9];
#pragma unroll
    for (int mu = 0; mu < 9; ++mu) eps[mu] = a.diag ? ld_stream_f64(a.diag + (size_t)mu * n + i) : 0.0;
    epilogue9<VW, LOG2T, kFirst, kDotL>(a, i, t, acc, eps, s1, s2);
  }
  block_store_sums<kBlock9Threads>(s1, s2, a.partial + blockIdx.x);
}

// ---- K7m: matrix-free, from the bond records ---------------------------------------------------------------
// Per (atom, neighbour): one column index, the neighbour's record (32 B) and its 9 orbital elements as
// 256-bit gathers (issued before the geometry, whose ~100 dependent fp64 instructions cover their latency),
// then 64 FMAs per real component.  (Staging the gathers through shared memory with cp.async one neighbour
// ahead measured 20 % SLOWER: the pass is bound by L1 wavefronts -- one per 32-byte gather of a lane --
// not by latency: ncu of that variant, l1tex data pipe 94 %, fp64 pipe 25 %.)
constexpr int kBond9Threads = 128;

// (Also measured and removed: one complex number per thread, 160 registers and 12 instead of 8 warps per
// SM for a second copy of the geometry -- the same 6.24 ms at K = 12; an L2 prefetch of the rows two grid
// strides ahead -- 5 % slower.  ncu at 10^8 atoms, K = 12: fp64 pipe 35 %, L1 data pipe 57 %, DRAM 24 % with
// traffic = 1.006 x the algorithmic bytes, 5.3 stall cycles per issue on long_scoreboard.  And at R = 2, where a
// neighbour's nine elements are 288 contiguous bytes: one cp.async.bulk per lane and neighbour into a per-lane
// shared-memory slot, one neighbour ahead, per-warp mbarriers -- bit-identical, 8.52 ms against 6.25 at K = 12:
// 1.2e8 small bulk copies per pass are one per ~20 cycles and SM, slower than the gathers they replace.)
// Round 2, after the column / record carry below (6.25 -> 5.48 ms): the first use of the gathered rows holds 37 %
// of the stall samples, fixed-latency dependencies 24 %, fp64 pipe 44 %.  Two more decompositions measured at
// K = 12, 1.02e7 atoms and removed: one complex number per thread again (168 registers, 12 warps per SM) 5.71 ms;
// one lane per REAL number (K7q: 2 R lanes per atom, nine accumulators each, 128 registers, 16 warps per SM; the
// pair's geometry worked out once by one lane of the atom per chunk of 2 R neighbours and handed to the others
// through shared memory, so the fp64 work per pair stays 75 + 4 x 64) 6.96 ms: bit-compatible with the tests, but
// l1tex__data_pipe_lsu_wavefronts goes to 91 % -- the gathers cost the same ~9 wavefronts per pair in any
// decomposition (a neighbour's 288 bytes lie in lines that no other lane of the instruction shares) and the
// records add 6 per pair.  So the L1 data pipe, ~3.6 ms of the 5.48, is this pass's floor (staging the gathered
// rows in shared memory like window.cu does not fit: a 64-atom tile's window at K = 12 is 69 KB); prefetch.global.L1
// of the next neighbour's rows: 5.66 ms.  At 10^8 atoms the pass reads 1.4 x its algorithmic bytes from DRAM: a
// neighbour's rows are used again one lattice row (20 000 atoms, two grid strides) later, at the edge of what L2
// keeps; an L2 evict-first policy on the streamed prev / y rows changes neither bytes nor time, a tile-major
// numbering of the INPUT atoms (16 x 16 cells) brings 1.07 x and 54.4 instead of 56.6 ms.
// geometry + closed-form action of one pair on the neighbour's nine orbital elements x into acc
struct BondCtx {
  double Lx, Ly, Lz, iLx, iLy, iLz, r0, beta;
  const double* s_coef;
  int ns;
  template <int VW>
  __device__ __forceinline__ void apply(const Vec<4>& pi, int si, const Vec<4>& pj, const Vec<VW> (&x)[9],
                                        Vec<VW> (&acc)[9]) const {
        double dx = __dsub_rn(pj.v[0], pi.v[0]), dy = __dsub_rn(pj.v[1], pi.v[1]), dz = __dsub_rn(pj.v[2], pi.v[2]);
        dx = fma(-Lx, rint(dx * iLx), dx);
        dy = fma(-Ly, rint(dy * iLy), dy);
        dz = fma(-Lz, rint(dz * iLz), dz);
        const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
        const double inv = rsqrt(r2);
        Geometry g;
        g.l = dx * inv;
        g.m = dy * inv;
        g.n = dz * inv;
        g.f = beta == 0.0 ? 1.0 : exp(-beta * (r2 * inv / r0 - 1.0));
        const double* c0 = s_coef + (si * ns + (int)pj.v[3]) * kNc;
        double c[kNc];
#pragma unroll
        for (int q = 0; q < kNc; ++q) c[q] = c0[q] * g.f;
        double D[5];
        angular_d(g, D);
        const double hl = 0.5 * kS3 * g.l, hm = 0.5 * kS3 * g.m, hn = 0.5 * kS3 * g.n;
        const double l2 = 0.5 * g.l, m2 = 0.5 * g.m;
#pragma unroll
        for (int q = 0; q < VW; ++q) {
          const double xs = x[0].v[q], px = x[1].v[q], py = x[2].v[q], pz = x[3].v[q];
          const double d0 = x[4].v[q], d1 = x[5].v[q], d2 = x[6].v[q], d3 = x[7].v[q], d4 = x[8].v[q];
          const double up = fma(g.l, px, fma(g.m, py, g.n * pz));                             // u . x_p
          const double qd = fma(D[0], d0, fma(D[1], d1, fma(D[2], d2, fma(D[3], d3, D[4] * d4))));  // D . x_d
          const double wx = fma(hm, d0, fma(hn, d2, fma(hl, d3, -l2 * d4)));                  // sum_b G_b x_d[b]
          const double wy = fma(hl, d0, fma(hn, d1, fma(-hm, d3, -m2 * d4)));
          const double wz = fma(hm, d1, fma(hl, d2, g.n * d4));
          acc[0].v[q] = fma(c[0], xs, fma(c[1], up, fma(c[2], qd, acc[0].v[q])));
          const double P = fma(c[3], xs, fma(c[5], up, c[6] * qd));
          acc[1].v[q] = fma(c[4], px, fma(c[7], wx, fma(g.l, P, acc[1].v[q])));
          acc[2].v[q] = fma(c[4], py, fma(c[7], wy, fma(g.m, P, acc[2].v[q])));
          acc[3].v[q] = fma(c[4], pz, fma(c[7], wz, fma(g.n, P, acc[3].v[q])));
          const double Q = fma(c[8], xs, fma(c[9], up, c[12] * qd));
          const double vx = fma(c[10], px, c[13] * wx), vy = fma(c[10], py, c[13] * wy),
                       vz = fma(c[10], pz, c[13] * wz);
          acc[4].v[q] = fma(c[11], d0, fma(D[0], Q, fma(hm, vx, fma(hl, vy, acc[4].v[q]))));
          acc[5].v[q] = fma(c[11], d1, fma(D[1], Q, fma(hn, vy, fma(hm, vz, acc[5].v[q]))));
          acc[6].v[q] = fma(c[11], d2, fma(D[2], Q, fma(hn, vx, fma(hl, vz, acc[6].v[q]))));
          acc[7].v[q] = fma(c[11], d3, fma(D[3], Q, fma(hl, vx, fma(-hm, vy, acc[7].v[q]))));
          acc[8].v[q] = fma(c[11], d4, fma(D[4], Q, fma(-l2, vx, fma(-m2, vy, fma(g.n, vz, acc[8].v[q])))));
        }
  }
};

template <int VW, int LOG2T, bool kFirst, bool kDotL>
__global__ void __launch_bounds__(kBond9Threads, 2) cheb_bond9_kernel(const StepArgs a) {
  constexpr int T = 1 << LOG2T;
  __shared__ double s_coef[GTB_MAX_SPECIES * GTB_MAX_SPECIES * kNc];
  __shared__ double s_onsite[3][GTB_MAX_SPECIES];
  const BondHeader& h = *reinterpret_cast<const BondHeader*>(a.vals);
  const int ns = h.n_species;
  for (int q = threadIdx.x; q < ns * ns * kNc; q += kBond9Threads) s_coef[q] = (&h.coef[0][0])[q];
  for (int q = threadIdx.x; q < 3 * GTB_MAX_SPECIES; q += kBond9Threads) (&s_onsite[0][0])[q] = (&h.onsite[0][0])[q];
  // periodic axes: d -= L rint(d / L), as a multiplication by 1/L (a neighbour's d / L is within
  // cutoff / L < 1/2 of an integer, far from the ties where the two roundings could differ)
  BondCtx bond;
  bond.Lx = h.box[0]; bond.Ly = h.box[1]; bond.Lz = h.box[2];
  bond.iLx = h.pbc[0] ? 1.0 / bond.Lx : 0.0;
  bond.iLy = h.pbc[1] ? 1.0 / bond.Ly : 0.0;
  bond.iLz = h.pbc[2] ? 1.0 / bond.Lz : 0.0;
  bond.r0 = h.r0; bond.beta = h.beta;
  bond.s_coef = s_coef; bond.ns = ns;
  __syncthreads();
  const int64_t n = a.n / 9;   // atoms
  const int K = a.width;
  const int64_t total = n * T;
  const double* posw = a.vals + kBondHeaderBytes / 8;
  const double* shift = posw + 4 * n;
  double s1 = 0.0, s2 = 0.0;
  for (int64_t e = (int64_t)blockIdx.x * kBond9Threads + threadIdx.x; e < total;
       e += (int64_t)gridDim.x * kBond9Threads) {
    const int64_t i = e >> LOG2T;
    const int64_t t = e - i * T;
    const double* xt = a.phi_cur + t * VW;
    const Vec<4> pi = ld_rec(posw + 4 * i);
    const int si = (int)pi.v[3];
    Vec<VW> acc[9];
#pragma unroll
    for (int mu = 0; mu < 9; ++mu)
#pragma unroll
      for (int q = 0; q < VW; ++q) acc[mu].v[q] = 0.0;
    // Columns run two neighbours ahead and the neighbour's record one ahead, all carried as loaded (32-bit
    // index, raw record): ncu's source page showed 26 % of the pass's stall samples on the sign extension of
    // the "prefetched" column, which the compiler had placed right behind its load, and 10 % on the record.
    const int32_t self = (int32_t)i;
    int32_t j0 = K > 0 ? ld_stream_i32(a.cols + i) : self;
    int32_t j1 = K > 1 ? ld_stream_i32(a.cols + (size_t)n + i) : self;
    Vec<4> p0 = ld_rec(posw + 4 * (int64_t)j0);
    for (int k = 0; k < K; ++k) {
      const int32_t j2 = k + 2 < K ? ld_stream_i32(a.cols + (size_t)(k + 2) * n + i) : self;
      const Vec<4> p1 = ld_rec(posw + 4 * (int64_t)j1);
      if (j0 != self) {   // padding slots carry the atom's own index
        const int64_t j = j0;
        Vec<VW> x[9];
#pragma unroll
        for (int nu = 0; nu < 9; ++nu) x[nu] = load_gather<VW>(xt + vec_off<LOG2T>(j, nu) * VW);
        bond.apply(pi, si, p0, x, acc);
      }
      j0 = j1;
      j1 = j2;
      p0 = p1;
    }
    const double sh = ld_stream_f64(shift + i);
    double eps[9];
    eps[0] = s_onsite[0][si] + sh;
#pragma unroll
    for (int mu = 1; mu < 4; ++mu) eps[mu] = s_onsite[1][si] + sh;
#pragma unroll
    for (int mu = 4; mu < 9; ++mu) eps[mu] = s_onsite[2][si] + sh;
    epilogue9<VW, LOG2T, kFirst, kDotL>(a, i, t, acc, eps, s1, s2);
  }
  block_store_sums<kBond9Threads>(s1, s2, a.partial + blockIdx.x);
}

template <int LOG2T>
void pick_rep9(int rep, StepPlan* p) {
  p->vw = 4;
  p->T = 1 << LOG2T;
  if (rep == 1) {
    p->first = cheb_block9_kernel<LOG2T, true, false>;
    p->next = cheb_block9_kernel<LOG2T, false, false>;
    p->block = kBlock9Threads;
    p->smem = 0;
  } else {
    p->first = cheb_bond9_kernel<4, LOG2T, true, false>;
    p->next = cheb_bond9_kernel<4, LOG2T, false, false>;
    p->block = kBond9Threads;
    p->smem = 0;
  }
}

int grid_of(int64_t total, int threads) {
  return (int)std::max<int64_t>(1, std::min<int64_t>((total + threads - 1) / threads, kMaxGrid));
}

int check_spd_model(const gtb_spd_model* m) {
  if (!m || !m->onsite_s || !m->onsite_p || !m->onsite_d || !m->sk || m->n_species < 1 ||
      m->n_species > GTB_MAX_SPECIES)
    return GTB_ERR_INVALID_ARG;
  // same-l integrals belong to both orderings of the pair: an asymmetric entry has no symmetric H
  for (int s = 0; s < m->n_species; ++s)
    for (int t = 0; t < s; ++t)
      for (int q : {0, 2, 3, 7, 8, 9})
        if (m->sk[((size_t)s * m->n_species + t) * 10 + q] != m->sk[((size_t)t * m->n_species + s) * 10 + q])
          return GTB_ERR_INVALID_ARG;
  return GTB_OK;
}

}  // namespace

bool make_plan_rep9(const gtb_ell* H, int R, int rep, StepPlan* p) {
  if ((rep != 1 && rep != 2) || (R != 2 && R != 4 && R != 8) || H->width < 0 || !H->vals ||
      (H->width > 0 && !H->cols) || (reinterpret_cast<uintptr_t>(H->vals) & 31u))
    return false;
  if (R == 2) pick_rep9<0>(rep, p);
  else if (R == 4) pick_rep9<1>(rep, p);
  else pick_rep9<2>(rep, p);
  p->stages = 0;
  int dev = 0, sms = kSmCount, per_sm = 0;
  if (p->smem > 0 &&
      (cudaFuncSetAttribute(p->first, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->smem) != cudaSuccess ||
       cudaFuncSetAttribute(p->next, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->smem) != cudaSuccess))
    return false;
  if (cudaGetDevice(&dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, p->next, p->block, p->smem) != cudaSuccess)
    return false;
  per_sm = std::max(1, per_sm);
  const int64_t total = H->n * p->T;
  p->grid = (int)std::max<int64_t>(1, std::min<int64_t>((total + p->block - 1) / p->block, (int64_t)sms * per_sm));
  p->grid = std::min(p->grid, kMaxGrid);
  return true;
}

}  // namespace gtb

using namespace gtb;

extern "C" size_t gtb_spd_bonds_bytes(int64_t n) {
  if (n <= 0) return 0;
  return align_up(kBondHeaderBytes + (size_t)n * 40);
}

extern "C" int gtb_spd_bonds(const gtb_ell* nbr, const double* pos, const int32_t* species,
                             const double box[3], const int32_t pbc[3], const gtb_spd_model* model,
                             gtb_ell* Hm, int32_t* status, void* stream) {
  int rc = check_ell(nbr);
  if (rc != GTB_OK) return rc;
  rc = check_spd_model(model);
  if (rc != GTB_OK) return rc;
  if (!pos || !species || !box || !pbc || !Hm || !status || Hm->n != nbr->n || Hm->width != nbr->width ||
      Hm->cols != nbr->cols || !Hm->vals || (reinterpret_cast<uintptr_t>(Hm->vals) & 255u))
    return GTB_ERR_INVALID_ARG;
  if (9 * nbr->n > (int64_t)INT32_MAX - 64) return GTB_ERR_INDEX_RANGE;
  for (int a = 0; a < 3; ++a)
    if (pbc[a] && !(box[a] > 0.0)) return GTB_ERR_INVALID_ARG;
  BondHeader h{};
  const int ns = model->n_species;
  for (int a = 0; a < 3; ++a) {
    h.box[a] = box[a];
    h.pbc[a] = pbc[a];
  }
  h.r0 = model->r0;
  h.beta = model->beta;
  h.n_species = ns;
  h.n = nbr->n;
  for (int s = 0; s < ns; ++s) {
    h.onsite[0][s] = model->onsite_s[s];
    h.onsite[1][s] = model->onsite_p[s];
    h.onsite[2][s] = model->onsite_d[s];
    for (int t = 0; t < ns; ++t)
      pair_coefficients(model->sk + ((size_t)s * ns + t) * 10, model->sk + ((size_t)t * ns + s) * 10,
                        h.coef[s * ns + t]);
  }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int64_t n = nbr->n;
  // the header goes up from pageable memory: the copy has left the host buffer when the call returns
  GTB_CUDA_TRY(cudaMemcpyAsync(Hm->vals, &h, sizeof(h), cudaMemcpyHostToDevice, st));
  GTB_CUDA_TRY(cudaStreamSynchronize(st));
  GTB_CUDA_TRY(cudaMemsetAsync(status, 0, sizeof(int32_t), st));
  double* posw = Hm->vals + kBondHeaderBytes / 8;
  bond_record_kernel<<<grid_of(n, kBlock), kBlock, 0, st>>>(n, pos, species, model->onsite_shift, ns, posw,
                                                            posw + 4 * n, status);
  GTB_LAUNCHED();
  return GTB_OK;
}

extern "C" int gtb_spd_blocks(const gtb_ell* Hm, gtb_ell* Hb, void* stream) {
  int rc = check_ell(Hm);
  if (rc != GTB_OK) return rc;
  if (!Hb || Hb->n != Hm->n || Hb->width != Hm->width || Hb->cols != Hm->cols ||
      (Hb->width > 0 && !Hb->vals) || (reinterpret_cast<uintptr_t>(Hb->vals) & 31u))
    return GTB_ERR_INVALID_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int64_t n = Hm->n;
  if (Hm->width > 0) {
    block9_assemble_kernel<<<grid_of(n * Hm->width, 128), 128, 0, st>>>(Hm->cols, n, Hm->width, Hm->vals,
                                                                        Hb->vals);
    GTB_LAUNCHED();
  }
  if (Hb->diag) {
    onsite9_kernel<<<grid_of(n, kBlock), kBlock, 0, st>>>(n, Hm->vals, Hb->diag);
    GTB_LAUNCHED();
  }
  return GTB_OK;
}

extern "C" size_t gtb_spd_bounds_workspace_bytes(void) { return align_up(sizeof(double) * 2 * kMaxGrid); }

extern "C" int gtb_spd_bounds(const gtb_ell* H, int32_t mode, double* lo_hi, void* ws, size_t ws_bytes,
                              void* stream) {
  int rc = check_ell(H);
  if (rc != GTB_OK) return rc;
  if ((mode != GTB_MODE_BLOCK9 && mode != GTB_MODE_BOND9) || !lo_hi || !H->vals) return GTB_ERR_INVALID_ARG;
  rc = check_ws(ws, ws_bytes, gtb_spd_bounds_workspace_bytes());
  if (rc != GTB_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  double* partial = static_cast<double*>(ws);
  const int grid = grid_of(H->n, 128);
  if (mode == GTB_MODE_BOND9)
    bounds9_kernel<true><<<grid, 128, 0, st>>>(H->cols, H->n, H->width, H->vals, nullptr, partial);
  else
    bounds9_kernel<false><<<grid, 128, 0, st>>>(H->cols, H->n, H->width, H->vals, H->diag, partial);
  GTB_LAUNCHED();
  bounds9_final_kernel<<<1, 32, 0, st>>>(partial, grid, lo_hi);
  GTB_LAUNCHED();
  return GTB_OK;
}
