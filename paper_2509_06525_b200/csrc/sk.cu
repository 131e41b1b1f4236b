// Multi-orbital Slater-Koster blocks: the paper's Hamiltonian is made of
// onsite blocks H_ii and hopping blocks H_ij^{lm,l'm'} built from Slater-Koster parameters and the bond
// direction, with H_ij^{l l'} = (-1)^{l+l'} H_ji^{l' l}.  This file
// assembles the s, p_x, p_y, p_z case (reading S1) from the neighbour lists of an
// existing ELL matrix into a scalar ELL matrix over the 4n orbitals, which the KPM / VAC kernels then
// take unchanged.  Two-centre table (Slater & Koster 1954), (l, m, n) = (x_j - x_i)/r:
//   E_ss = V_ss_sigma;  E_{s,pa} = a V_sp_sigma;  E_{pa,s} = -a V_sp_sigma;
//   E_{pa,pb} = a b V_pp_sigma + (delta_ab - a b) V_pp_pi;   every V times exp(-beta (r/r0 - 1)).
#include <cmath>

#include "cheb.cuh"

namespace gtb {
namespace {

struct SkParams {
  double onsite_s[GTB_MAX_SPECIES];
  double onsite_p[GTB_MAX_SPECIES];
  double sk[GTB_MAX_SPECIES * GTB_MAX_SPECIES * 4];
  double r0, beta;
  double box[3];
  int32_t pbc[3];
  int32_t n_species;
};

// one thread per (atom i, neighbour slot k): the 4x4 block of the pair, 16 scalar entries
__global__ void __launch_bounds__(kBlock) sk_block_kernel(const int32_t* __restrict__ nbr_cols,
                                                          int64_t n, int32_t K,
                                                          const double* __restrict__ pos,
                                                          const int32_t* __restrict__ species,
                                                          const SkParams p, int32_t* __restrict__ cols,
                                                          double* __restrict__ vals,
                                                          int32_t* __restrict__ status) {
  const int64_t total = n * K;
  const int64_t N = 4 * n;
  for (int64_t e = (int64_t)blockIdx.x * kBlock + threadIdx.x; e < total;
       e += (int64_t)gridDim.x * kBlock) {
    const int64_t k = e / n;
    const int64_t i = e - k * n;
    const int64_t j = nbr_cols[e];
    double E[4][4];
#pragma unroll
    for (int mu = 0; mu < 4; ++mu)
#pragma unroll
      for (int nu = 0; nu < 4; ++nu) E[mu][nu] = 0.0;
    if (j != i) {
      const int si = species[i], sj = species[j];
      if (si < 0 || si >= p.n_species || sj < 0 || sj >= p.n_species) {
        atomicOr(status, 1);
        continue;
      }
      double d[3];
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        d[a] = __dsub_rn(pos[j * 3 + a], pos[i * 3 + a]);
        if (p.pbc[a]) d[a] = __dsub_rn(d[a], __dmul_rn(p.box[a], rint(__ddiv_rn(d[a], p.box[a]))));
      }
      const double r = sqrt(__dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])),
                                      __dmul_rn(d[2], d[2])));
      const double c[3] = {d[0] / r, d[1] / r, d[2] / r};
      const double f = p.beta == 0.0 ? 1.0 : exp(-p.beta * (r / p.r0 - 1.0));
      const double* V = p.sk + ((size_t)si * p.n_species + sj) * 4;
      const double Vss = V[0] * f, Vsp = V[1] * f, Vpp_s = V[2] * f, Vpp_p = V[3] * f;
      // E_{pa,s} = (-1)^{1+0} H_ji^{s,pa}: the s orbital sits on j, so the integral is the
      // table entry of the pair (s_j, s_i) -- H stays symmetric for a species-asymmetric table
      const double Vsp_ji = p.sk[((size_t)sj * p.n_species + si) * 4 + 1] * f;
      E[0][0] = Vss;
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        E[0][1 + a] = c[a] * Vsp;
        E[1 + a][0] = -(c[a] * Vsp_ji);
#pragma unroll
        for (int b = 0; b < 3; ++b)
          E[1 + a][1 + b] = c[a] * c[b] * Vpp_s + ((a == b ? 1.0 : 0.0) - c[a] * c[b]) * Vpp_p;
      }
    }
#pragma unroll
    for (int nu = 0; nu < 4; ++nu) {
      const size_t at = (size_t)(4 * k + nu) * N + 4 * i;
#pragma unroll
      for (int mu = 0; mu < 4; ++mu) {
        cols[at + mu] = (int32_t)(j != i ? 4 * j + nu : 4 * i + mu);
        vals[at + mu] = E[mu][nu];
      }
    }
  }
}

__global__ void __launch_bounds__(kBlock) sk_onsite_kernel(int64_t n, const int32_t* __restrict__ species,
                                                           const SkParams p,
                                                           const double* __restrict__ shift,
                                                           double* __restrict__ diag) {
  for (int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x; i < n;
       i += (int64_t)gridDim.x * kBlock) {
    const int s = min(max(species[i], 0), p.n_species - 1);
    const double sh = shift ? shift[i] : 0.0;
    diag[4 * i] = p.onsite_s[s] + sh;
    diag[4 * i + 1] = diag[4 * i + 2] = diag[4 * i + 3] = p.onsite_p[s] + sh;
  }
}


// ---- s, p, d (9 orbitals: s, px, py, pz, dxy, dyz, dzx, dx2-y2, dz2) -------------------------------
// Two-centre integrals are diagonal in the bond frame (e1, e2, u).  Per lab orbital a the coefficients
// on the frame orbitals m = sigma, pi1, pi2, delta1, delta2 are: s -> (1); p_alpha -> (u, e1, e2)_alpha;
// d_a -> from the symmetric traceless form B_m of the frame orbital: (2/sqrt3) B_m[x][y] (cyclic),
// (B_m[x][x] - B_m[y][y])/sqrt3, B_m[z][z].  E_ab = sum_m c_am V_{l_a l_b |m|} c_bm, times
// (-1)^{l_a + l_b} when l_a > l_b.
struct SpdParams {
  double onsite[3][GTB_MAX_SPECIES];                       // s, p, d
  double sk[GTB_MAX_SPECIES * GTB_MAX_SPECIES * 10];
  double r0, beta;
  double box[3];
  int32_t pbc[3];
  int32_t n_species;
};

__device__ __forceinline__ double spd_integral(const double* V, int lo, int hi, int m) {
  const int am = m == 0 ? 0 : (m <= 2 ? 1 : 2);
  if (hi == 0) return am == 0 ? V[0] : 0.0;
  if (hi == 1) return lo == 0 ? (am == 0 ? V[1] : 0.0) : (am == 0 ? V[2] : (am == 1 ? V[3] : 0.0));
  if (lo == 0) return am == 0 ? V[4] : 0.0;
  if (lo == 1) return am == 0 ? V[5] : (am == 1 ? V[6] : 0.0);
  return am == 0 ? V[7] : (am == 1 ? V[8] : V[9]);
}

__global__ void __launch_bounds__(128) spd_block_kernel(const int32_t* __restrict__ nbr_cols, int64_t n,
                                                        int32_t K, const double* __restrict__ pos,
                                                        const int32_t* __restrict__ species,
                                                        const SpdParams* __restrict__ pp,
                                                        int32_t* __restrict__ cols,
                                                        double* __restrict__ vals,
                                                        int32_t* __restrict__ status) {
  const SpdParams& p = *pp;
  const int64_t total = n * K;
  const int64_t N = 9 * n;
  for (int64_t e = (int64_t)blockIdx.x * 128 + threadIdx.x; e < total; e += (int64_t)gridDim.x * 128) {
    const int64_t k = e / n;
    const int64_t i = e - k * n;
    const int64_t j = nbr_cols[e];
    if (j == i) {  // padding: the row's own index, value 0
      for (int nu = 0; nu < 9; ++nu)
        for (int mu = 0; mu < 9; ++mu) {
          const size_t at = (size_t)(9 * k + nu) * N + 9 * i + mu;
          cols[at] = (int32_t)(9 * i + mu);
          vals[at] = 0.0;
        }
      continue;
    }
    const int si = species[i], sj = species[j];
    if (si < 0 || si >= p.n_species || sj < 0 || sj >= p.n_species) {
      atomicOr(status, 1);
      continue;
    }
    double d[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      d[a] = __dsub_rn(pos[j * 3 + a], pos[i * 3 + a]);
      if (p.pbc[a]) d[a] = __dsub_rn(d[a], __dmul_rn(p.box[a], rint(__ddiv_rn(d[a], p.box[a]))));
    }
    const double r = sqrt(__dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])),
                                    __dmul_rn(d[2], d[2])));
    const double u[3] = {d[0] / r, d[1] / r, d[2] / r};
    // frame: e1 = u x t / |u x t| with t = z (or x when u is close to z), e2 = u x e1
    const bool near_z = fabs(u[2]) > 0.9;
    const double t[3] = {near_z ? 1.0 : 0.0, 0.0, near_z ? 0.0 : 1.0};
    double e1[3] = {u[1] * t[2] - u[2] * t[1], u[2] * t[0] - u[0] * t[2], u[0] * t[1] - u[1] * t[0]};
    const double inv = 1.0 / sqrt(e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2]);
    e1[0] *= inv; e1[1] *= inv; e1[2] *= inv;
    const double e2[3] = {u[1] * e1[2] - u[2] * e1[1], u[2] * e1[0] - u[0] * e1[2], u[0] * e1[1] - u[1] * e1[0]};
    double c[9][5];
#pragma unroll
    for (int a = 0; a < 9; ++a)
#pragma unroll
      for (int m = 0; m < 5; ++m) c[a][m] = 0.0;
    c[0][0] = 1.0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      c[1 + a][0] = u[a];
      c[1 + a][1] = e1[a];
      c[1 + a][2] = e2[a];
    }
    const double s3 = 1.7320508075688772;
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      // B_m = f (v w^T + w v^T) - g 1 with (v, w, f, g) per frame orbital
      const double* v = m == 0 ? u : (m == 1 || m == 2) ? u : e1;
      const double* wv = m == 0 ? u : m == 1 ? e1 : m == 2 ? e2 : m == 3 ? e2 : e1;
      const double f = m == 0 ? 0.75 : s3 / 2;
      double B01 = f * (v[0] * wv[1] + wv[0] * v[1]);
      double B12 = f * (v[1] * wv[2] + wv[1] * v[2]);
      double B20 = f * (v[2] * wv[0] + wv[2] * v[0]);
      double B00 = f * 2.0 * v[0] * wv[0], B11 = f * 2.0 * v[1] * wv[1], B22 = f * 2.0 * v[2] * wv[2];
      if (m == 0) {           // (3 u u^T - 1)/2
        B00 -= 0.5; B11 -= 0.5; B22 -= 0.5;
      } else if (m == 4) {    // (sqrt3/2)(e1 e1^T - e2 e2^T)
        B01 -= s3 / 2 * 2.0 * e2[0] * e2[1]; B12 -= s3 / 2 * 2.0 * e2[1] * e2[2]; B20 -= s3 / 2 * 2.0 * e2[2] * e2[0];
        B00 -= s3 / 2 * 2.0 * e2[0] * e2[0]; B11 -= s3 / 2 * 2.0 * e2[1] * e2[1]; B22 -= s3 / 2 * 2.0 * e2[2] * e2[2];
        B01 *= 0.5; B12 *= 0.5; B20 *= 0.5; B00 *= 0.5; B11 *= 0.5; B22 *= 0.5;
      }
      c[4][m] = 2.0 / s3 * B01;
      c[5][m] = 2.0 / s3 * B12;
      c[6][m] = 2.0 / s3 * B20;
      c[7][m] = (B00 - B11) / s3;
      c[8][m] = B22;
    }
    const double fr = p.beta == 0.0 ? 1.0 : exp(-p.beta * (r / p.r0 - 1.0));
    // V: pair (s_i, s_j) for l_a <= l_b; Vt: pair (s_j, s_i) for l_a > l_b (that element is
    // the transposed one of the (j, i) block, whose lower-l orbital sits on atom j)
    double V[10], Vt[10];
#pragma unroll
    for (int q = 0; q < 10; ++q) {
      V[q] = p.sk[((size_t)si * p.n_species + sj) * 10 + q] * fr;
      Vt[q] = p.sk[((size_t)sj * p.n_species + si) * 10 + q] * fr;
    }
    for (int nu = 0; nu < 9; ++nu) {
      const int lb = nu == 0 ? 0 : (nu < 4 ? 1 : 2);
      for (int mu = 0; mu < 9; ++mu) {
        const int la = mu == 0 ? 0 : (mu < 4 ? 1 : 2);
        const int lo = min(la, lb), hi = max(la, lb);
        double sum = 0.0;
#pragma unroll
        for (int m = 0; m < 5; ++m) sum += c[mu][m] * spd_integral(la > lb ? Vt : V, lo, hi, m) * c[nu][m];
        const size_t at = (size_t)(9 * k + nu) * N + 9 * i + mu;
        cols[at] = (int32_t)(9 * j + nu);
        vals[at] = (la > lb && ((la + lb) & 1)) ? -sum : sum;
      }
    }
  }
}

__global__ void __launch_bounds__(kBlock) spd_onsite_kernel(int64_t n, const int32_t* __restrict__ species,
                                                            const SpdParams* __restrict__ pp,
                                                            const double* __restrict__ shift,
                                                            double* __restrict__ diag) {
  const SpdParams& p = *pp;
  for (int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x; i < n; i += (int64_t)gridDim.x * kBlock) {
    const int s = min(max(species[i], 0), p.n_species - 1);
    const double sh = shift ? shift[i] : 0.0;
    diag[9 * i] = p.onsite[0][s] + sh;
    for (int a = 1; a < 4; ++a) diag[9 * i + a] = p.onsite[1][s] + sh;
    for (int a = 4; a < 9; ++a) diag[9 * i + a] = p.onsite[2][s] + sh;
  }
}

}  // namespace
}  // namespace gtb

using namespace gtb;

extern "C" int gtb_sk_hamiltonian(const gtb_ell* nbr, const double* pos, const int32_t* species,
                                  const double box[3], const int32_t pbc[3],
                                  const gtb_sk_model* model, gtb_ell* H, int32_t* status,
                                  void* stream) {
  int rc = check_ell(nbr);
  if (rc != GTB_OK) return rc;
  if (!pos || !species || !box || !pbc || !model || !H || !status || !model->onsite_s ||
      !model->onsite_p || !model->sk || model->n_species < 1 || model->n_species > GTB_MAX_SPECIES ||
      H->n != 4 * nbr->n || H->width != 4 * nbr->width || (H->width > 0 && (!H->cols || !H->vals)))
    return GTB_ERR_INVALID_ARG;
  if (H->n > (int64_t)INT32_MAX - 64) return GTB_ERR_INDEX_RANGE;
  for (int a = 0; a < 3; ++a)
    if (pbc[a] && !(box[a] > 0.0)) return GTB_ERR_INVALID_ARG;
  SkParams p{};
  p.n_species = model->n_species;
  for (int s = 0; s < p.n_species; ++s) {
    p.onsite_s[s] = model->onsite_s[s];
    p.onsite_p[s] = model->onsite_p[s];
  }
  for (int q = 0; q < p.n_species * p.n_species * 4; ++q) p.sk[q] = model->sk[q];
  p.r0 = model->r0;
  p.beta = model->beta;
  for (int a = 0; a < 3; ++a) {
    p.box[a] = box[a];
    p.pbc[a] = pbc[a];
  }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int64_t n = nbr->n;
  GTB_CUDA_TRY(cudaMemsetAsync(status, 0, sizeof(int32_t), st));
  if (nbr->width > 0) {
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((n * nbr->width + kBlock - 1) / kBlock, kMaxGrid));
    sk_block_kernel<<<grid, kBlock, 0, st>>>(nbr->cols, n, nbr->width, pos, species, p, H->cols,
                                             H->vals, status);
    GTB_LAUNCHED();
  }
  if (H->diag) {
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((n + kBlock - 1) / kBlock, kMaxGrid));
    sk_onsite_kernel<<<grid, kBlock, 0, st>>>(n, species, p, model->onsite_shift, H->diag);
    GTB_LAUNCHED();
  }
  return GTB_OK;
}

extern "C" size_t gtb_spd_workspace_bytes(void) { return align_up(sizeof(SpdParams)); }

extern "C" int gtb_spd_hamiltonian(const gtb_ell* nbr, const double* pos, const int32_t* species,
                                   const double box[3], const int32_t pbc[3],
                                   const gtb_spd_model* model, gtb_ell* H, int32_t* status, void* ws,
                                   size_t ws_bytes, void* stream) {
  int rc = check_ell(nbr);
  if (rc != GTB_OK) return rc;
  if (!pos || !species || !box || !pbc || !model || !H || !status || !model->onsite_s ||
      !model->onsite_p || !model->onsite_d || !model->sk || model->n_species < 1 ||
      model->n_species > GTB_MAX_SPECIES || H->n != 9 * nbr->n || H->width != 9 * nbr->width ||
      (H->width > 0 && (!H->cols || !H->vals)))
    return GTB_ERR_INVALID_ARG;
  if (H->n > (int64_t)INT32_MAX - 64) return GTB_ERR_INDEX_RANGE;
  rc = check_ws(ws, ws_bytes, gtb_spd_workspace_bytes());
  if (rc != GTB_OK) return rc;
  for (int a = 0; a < 3; ++a)
    if (pbc[a] && !(box[a] > 0.0)) return GTB_ERR_INVALID_ARG;
  SpdParams p{};
  p.n_species = model->n_species;
  for (int s = 0; s < p.n_species; ++s) {
    p.onsite[0][s] = model->onsite_s[s];
    p.onsite[1][s] = model->onsite_p[s];
    p.onsite[2][s] = model->onsite_d[s];
  }
  for (int q = 0; q < p.n_species * p.n_species * 10; ++q) p.sk[q] = model->sk[q];
  p.r0 = model->r0;
  p.beta = model->beta;
  for (int a = 0; a < 3; ++a) {
    p.box[a] = box[a];
    p.pbc[a] = pbc[a];
  }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  // the parameter block (5.4 KB) exceeds the kernel-argument limit: it goes through the workspace.
  // The copy is from pageable memory, so it has completed on the host side when the call returns.
  GTB_CUDA_TRY(cudaMemcpyAsync(ws, &p, sizeof(p), cudaMemcpyHostToDevice, st));
  GTB_CUDA_TRY(cudaStreamSynchronize(st));
  const SpdParams* dp = static_cast<const SpdParams*>(ws);
  const int64_t n = nbr->n;
  GTB_CUDA_TRY(cudaMemsetAsync(status, 0, sizeof(int32_t), st));
  if (nbr->width > 0) {
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((n * nbr->width + 127) / 128, kMaxGrid));
    spd_block_kernel<<<grid, 128, 0, st>>>(nbr->cols, n, nbr->width, pos, species, dp, H->cols, H->vals,
                                           status);
    GTB_LAUNCHED();
  }
  if (H->diag) {
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((n + kBlock - 1) / kBlock, kMaxGrid));
    spd_onsite_kernel<<<grid, kBlock, 0, st>>>(n, species, dp, model->onsite_shift, H->diag);
    GTB_LAUNCHED();
  }
  return GTB_OK;
}
