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
      E[0][0] = Vss;
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        E[0][1 + a] = c[a] * Vsp;
        E[1 + a][0] = -(c[a] * Vsp);
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
