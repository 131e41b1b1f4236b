// Environment-dependent Hamiltonian from the paper's descriptor and MLPs (Eq. 2 and the text around it,
// PAPER.md:81-86), one orbital per atom:
//   f_k(r) = 1/2 [T_k(2 (r/r_cut - 1)^2 - 1) + 1] f_c(r),  C_n(r_ij) = sum_k c_nk^{ij} f_k(r_ij),
//   v_i = sum_{j in N(i)} C_n(r_ij),  e_ij = C_n(r_ij) * MLP_e(v_i + v_j),
//   t_ij = MLP_lambda(e_ij),  eps_i = MLP_{alpha(i)}(v_i),  SiLU hidden layers.
// Readings E1-E4: f_c(r) = 1/2 [1 + cos(pi r/r_cut)]; k = 0..Nb-1, n = 0..F-1,
// "*" element-wise; every MLP is input -> hidden (SiLU) -> linear output; synthetic weights.
// Three kernels on the neighbour lists of an existing ELL matrix: node features (one thread per
// atom), hoppings (one thread per (slot, atom) entry), onsite energies.  The weight blob (12 KB at
// F = Nb = 8, Hd = 16) is staged in shared memory by every block.
#include <cmath>

#include "cheb.cuh"
#include "spd_pair.cuh"

namespace gtb {
namespace {

struct MlpGeom {
  double box[3];
  int32_t pbc[3];
  double r_cut;
  int32_t ns;
};

// PH / PO: outputs of MLP_lambda / of the onsite MLPs (1, 1: one orbital per atom; 4, 2: s,p blocks)
template <int F, int NB, int HD, int PH = 1, int PO = 1>
struct Blob {
  static constexpr int kC = F * NB;                     // per species pair
  static constexpr int kEnv = HD * F + HD + F * HD + F;
  static constexpr int kHop = HD * F + HD + PH * HD + PH;
  static constexpr int kOns = HD * F + HD + PO * HD + PO;
  __host__ __device__ static int size(int ns) { return ns * ns * kC + kEnv + kHop + ns * kOns; }
  __device__ static const double* c(const double* w, int ns, int si, int sj) { return w + (si * ns + sj) * kC; }
  __device__ static const double* env(const double* w, int ns) { return w + ns * ns * kC; }
  __device__ static const double* hop(const double* w, int ns) { return env(w, ns) + kEnv; }
  __device__ static const double* ons(const double* w, int ns, int s) { return hop(w, ns) + kHop + s * kOns; }
};

__device__ __forceinline__ double silu(double x) { return x / (1.0 + exp(-x)); }
// out-of-range species are reported through *status; clamped here so that no lookup leaves the blob
__device__ __forceinline__ int sp(const int32_t* __restrict__ species, int64_t i, int ns) {
  return min(max(species[i], 0), ns - 1);
}

__device__ __forceinline__ double pair_distance(const double* __restrict__ pos, int64_t i, int64_t j,
                                                const MlpGeom& g) {
  double d[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    d[a] = __dsub_rn(pos[j * 3 + a], pos[i * 3 + a]);
    if (g.pbc[a]) d[a] = __dsub_rn(d[a], __dmul_rn(g.box[a], rint(__ddiv_rn(d[a], g.box[a]))));
  }
  return sqrt(__dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2])));
}

// C[n] = sum_k c[n][k] f_k(r)
template <int F, int NB>
__device__ __forceinline__ void descriptor(const double* c, double r, double r_cut, double (&C)[F]) {
  const double fc = r < r_cut ? 0.5 * (1.0 + cos(3.14159265358979323846 * r / r_cut)) : 0.0;
  const double q = r / r_cut - 1.0;
  const double x = 2.0 * q * q - 1.0;
#pragma unroll
  for (int n = 0; n < F; ++n) C[n] = 0.0;
  double t_prev = 1.0, t_cur = x;
#pragma unroll
  for (int k = 0; k < NB; ++k) {
    double Tk;
    if (k == 0) {
      Tk = 1.0;
    } else if (k == 1) {
      Tk = x;
    } else {
      Tk = 2.0 * x * t_cur - t_prev;
      t_prev = t_cur;
      t_cur = Tk;
    }
    const double f = 0.5 * (Tk + 1.0) * fc;
#pragma unroll
    for (int n = 0; n < F; ++n) C[n] += c[n * NB + k] * f;
  }
}

// y[o] = b2[o] + sum_a W2[o][a] silu(b1[a] + sum_n W1[a][n] x[n])
template <int F, int HD, int OUT>
__device__ __forceinline__ void mlp(const double* p, const double (&x)[F], double (&y)[OUT]) {
  const double* W1 = p;
  const double* b1 = W1 + HD * F;
  const double* W2 = b1 + HD;
  const double* b2 = W2 + OUT * HD;
#pragma unroll
  for (int o = 0; o < OUT; ++o) y[o] = b2[o];
#pragma unroll 4
  for (int a = 0; a < HD; ++a) {
    double s = b1[a];
#pragma unroll
    for (int n = 0; n < F; ++n) s += W1[a * F + n] * x[n];
    const double h = silu(s);
#pragma unroll
    for (int o = 0; o < OUT; ++o) y[o] += W2[o * HD + a] * h;
  }
}

template <int F, int NB, int HD, int PH = 1, int PO = 1>
__device__ __forceinline__ const double* stage_weights(const double* __restrict__ w, int ns) {
  extern __shared__ double s_w[];
  const int total = Blob<F, NB, HD, PH, PO>::size(ns);
  for (int q = threadIdx.x; q < total; q += blockDim.x) s_w[q] = w[q];
  __syncthreads();
  return s_w;
}

template <int F, int NB, int HD>
__global__ void __launch_bounds__(kBlock) node_feature_kernel(const int32_t* __restrict__ cols, int64_t n,
                                                              int32_t width, const double* __restrict__ pos,
                                                              const int32_t* __restrict__ species,
                                                              const MlpGeom g, const double* __restrict__ w,
                                                              double* __restrict__ v) {
  const double* sw = stage_weights<F, NB, HD>(w, g.ns);
  for (int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x; i < n; i += (int64_t)gridDim.x * kBlock) {
    const int si = sp(species, i, g.ns);
    double acc[F], C[F];
#pragma unroll
    for (int q = 0; q < F; ++q) acc[q] = 0.0;
    for (int k = 0; k < width; ++k) {
      const int64_t j = cols[(size_t)k * n + i];
      if (j == i) continue;
      descriptor<F, NB>(Blob<F, NB, HD>::c(sw, g.ns, si, sp(species, j, g.ns)), pair_distance(pos, i, j, g), g.r_cut, C);
#pragma unroll
      for (int q = 0; q < F; ++q) acc[q] += C[q];
    }
#pragma unroll
    for (int q = 0; q < F; ++q) v[i * F + q] = acc[q];
  }
}

template <int F, int NB, int HD>
__global__ void __launch_bounds__(kBlock) mlp_hopping_kernel(const int32_t* __restrict__ cols, int64_t n,
                                                             int32_t width, const double* __restrict__ pos,
                                                             const int32_t* __restrict__ species,
                                                             const MlpGeom g, const double* __restrict__ w,
                                                             const double* __restrict__ v,
                                                             double* __restrict__ vals) {
  const double* sw = stage_weights<F, NB, HD>(w, g.ns);
  const int64_t total = n * width;
  for (int64_t e = (int64_t)blockIdx.x * kBlock + threadIdx.x; e < total; e += (int64_t)gridDim.x * kBlock) {
    const int64_t i = e % n;
    const int64_t j = cols[e];
    double t[1] = {0.0};
    if (j != i) {
      double C[F], u[F], env[F];
      descriptor<F, NB>(Blob<F, NB, HD>::c(sw, g.ns, sp(species, i, g.ns), sp(species, j, g.ns)), pair_distance(pos, i, j, g),
                        g.r_cut, C);
#pragma unroll
      for (int q = 0; q < F; ++q) u[q] = v[i * F + q] + v[j * F + q];
      mlp<F, HD, F>(Blob<F, NB, HD>::env(sw, g.ns), u, env);
#pragma unroll
      for (int q = 0; q < F; ++q) u[q] = C[q] * env[q];   // e_ij
      mlp<F, HD, 1>(Blob<F, NB, HD>::hop(sw, g.ns), u, t);
    }
    vals[e] = t[0];
  }
}

template <int F, int NB, int HD>
__global__ void __launch_bounds__(kBlock) mlp_onsite_kernel(int64_t n, const int32_t* __restrict__ species,
                                                            const MlpGeom g, const double* __restrict__ w,
                                                            const double* __restrict__ v,
                                                            double* __restrict__ diag) {
  const double* sw = stage_weights<F, NB, HD>(w, g.ns);
  for (int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x; i < n; i += (int64_t)gridDim.x * kBlock) {
    double x[F], y[1];
#pragma unroll
    for (int q = 0; q < F; ++q) x[q] = v[i * F + q];
    mlp<F, HD, 1>(Blob<F, NB, HD>::ons(sw, g.ns, sp(species, i, g.ns)), x, y);
    diag[i] = y[0];
  }
}

// Eq. 2 feeding the s,p Slater-Koster blocks: MLP_lambda has four outputs, the bond integrals
// of the pair; one thread per (slot, atom) writes the 16 entries of the block in gtb_sk_hamiltonian's layout.
template <int F, int NB, int HD>
__global__ void __launch_bounds__(kBlock) mlp_sk_block_kernel(const int32_t* __restrict__ nbr_cols, int64_t n,
                                                              int32_t K, const double* __restrict__ pos,
                                                              const int32_t* __restrict__ species,
                                                              const MlpGeom g, const double* __restrict__ w,
                                                              const double* __restrict__ v,
                                                              int32_t* __restrict__ cols,
                                                              double* __restrict__ vals) {
  using B4 = Blob<F, NB, HD, 4, 2>;
  const double* sw = stage_weights<F, NB, HD, 4, 2>(w, g.ns);
  const int64_t total = n * K;
  const int64_t N = 4 * n;
  for (int64_t e = (int64_t)blockIdx.x * kBlock + threadIdx.x; e < total; e += (int64_t)gridDim.x * kBlock) {
    const int64_t k = e / n;
    const int64_t i = e - k * n;
    const int64_t j = nbr_cols[e];
    double E[4][4];
#pragma unroll
    for (int mu = 0; mu < 4; ++mu)
#pragma unroll
      for (int nu = 0; nu < 4; ++nu) E[mu][nu] = 0.0;
    if (j != i) {
      double d[3];
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        d[a] = __dsub_rn(pos[j * 3 + a], pos[i * 3 + a]);
        if (g.pbc[a]) d[a] = __dsub_rn(d[a], __dmul_rn(g.box[a], rint(__ddiv_rn(d[a], g.box[a]))));
      }
      const double r = sqrt(__dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])),
                                      __dmul_rn(d[2], d[2])));
      const double c[3] = {d[0] / r, d[1] / r, d[2] / r};
      double C[F], u[F], env[F], V[4];
      descriptor<F, NB>(B4::c(sw, g.ns, sp(species, i, g.ns), sp(species, j, g.ns)), r, g.r_cut, C);
#pragma unroll
      for (int q = 0; q < F; ++q) u[q] = v[i * F + q] + v[j * F + q];
      mlp<F, HD, F>(B4::env(sw, g.ns), u, env);
#pragma unroll
      for (int q = 0; q < F; ++q) u[q] = C[q] * env[q];
      mlp<F, HD, 4>(B4::hop(sw, g.ns), u, V);
      E[0][0] = V[0];
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        E[0][1 + a] = c[a] * V[1];
        E[1 + a][0] = -(c[a] * V[1]);
#pragma unroll
        for (int b = 0; b < 3; ++b)
          E[1 + a][1 + b] = c[a] * c[b] * V[2] + ((a == b ? 1.0 : 0.0) - c[a] * c[b]) * V[3];
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

template <int F, int NB, int HD>
__global__ void __launch_bounds__(kBlock) mlp_sk_onsite_kernel(int64_t n, const int32_t* __restrict__ species,
                                                               const MlpGeom g, const double* __restrict__ w,
                                                               const double* __restrict__ v,
                                                               double* __restrict__ diag) {
  const double* sw = stage_weights<F, NB, HD, 4, 2>(w, g.ns);
  for (int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x; i < n; i += (int64_t)gridDim.x * kBlock) {
    double x[F], y[2];
#pragma unroll
    for (int q = 0; q < F; ++q) x[q] = v[i * F + q];
    mlp<F, HD, 2>(Blob<F, NB, HD, 4, 2>::ons(sw, g.ns, sp(species, i, g.ns)), x, y);
    diag[4 * i] = y[0];
    diag[4 * i + 1] = diag[4 * i + 2] = diag[4 * i + 3] = y[1];
  }
}

// ---- Eq. 2 feeding the s,p,d blocks (reading E7): MLP_lambda with ten outputs, onsite MLPs with three --------
// one thread per (atom, neighbour slot): the pair's ten integrals from the networks, then the closed form of
// spd_pair.cuh into the block layout of gtb_spd_blocks, blocks[k][9 nu + mu][i]
template <int F, int NB, int HD>
__global__ void __launch_bounds__(128) mlp_spd_block_kernel(const int32_t* __restrict__ nbr_cols, int64_t n,
                                                            int32_t K, const double* __restrict__ pos,
                                                            const int32_t* __restrict__ species,
                                                            const MlpGeom g, const double* __restrict__ w,
                                                            const double* __restrict__ v,
                                                            double* __restrict__ blocks) {
  using B10 = Blob<F, NB, HD, 10, 3>;
  const double* sw = stage_weights<F, NB, HD, 10, 3>(w, g.ns);
  const int64_t total = n * K;
  for (int64_t e = (int64_t)blockIdx.x * 128 + threadIdx.x; e < total; e += (int64_t)gridDim.x * 128) {
    const int64_t k = e / n;
    const int64_t i = e - k * n;
    const int64_t j = nbr_cols[e];
    double E[9][9];
    if (j == i) {
      for (int mu = 0; mu < 9; ++mu)
        for (int nu = 0; nu < 9; ++nu) E[mu][nu] = 0.0;
    } else {
      double d[3];
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        d[a] = __dsub_rn(pos[j * 3 + a], pos[i * 3 + a]);
        if (g.pbc[a]) d[a] = __dsub_rn(d[a], __dmul_rn(g.box[a], rint(__ddiv_rn(d[a], g.box[a]))));
      }
      const double r = sqrt(__dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])),
                                      __dmul_rn(d[2], d[2])));
      double C[F], u[F], env[F], V[10], c[kNc];
      descriptor<F, NB>(B10::c(sw, g.ns, sp(species, i, g.ns), sp(species, j, g.ns)), r, g.r_cut, C);
#pragma unroll
      for (int q = 0; q < F; ++q) u[q] = v[i * F + q] + v[j * F + q];
      mlp<F, HD, F>(B10::env(sw, g.ns), u, env);
#pragma unroll
      for (int q = 0; q < F; ++q) u[q] = C[q] * env[q];
      mlp<F, HD, 10>(B10::hop(sw, g.ns), u, V);
      pair_coefficients(V, V, c);   // e_ij = e_ji: the same integrals serve both orderings of the pair
      Geometry geo;
      geo.l = d[0] / r;
      geo.m = d[1] / r;
      geo.n = d[2] / r;
      geo.f = 1.0;
      pair_block(geo, c, E);
    }
    double* out = blocks + (size_t)k * 81 * n + i;
    for (int nu = 0; nu < 9; ++nu)
      for (int mu = 0; mu < 9; ++mu) out[(size_t)(9 * nu + mu) * n] = E[mu][nu];
  }
}

template <int F, int NB, int HD>
__global__ void __launch_bounds__(kBlock) mlp_spd_onsite_kernel(int64_t n, const int32_t* __restrict__ species,
                                                                const MlpGeom g, const double* __restrict__ w,
                                                                const double* __restrict__ v,
                                                                double* __restrict__ onsite) {
  const double* sw = stage_weights<F, NB, HD, 10, 3>(w, g.ns);
  for (int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x; i < n; i += (int64_t)gridDim.x * kBlock) {
    double x[F], y[3];
#pragma unroll
    for (int q = 0; q < F; ++q) x[q] = v[i * F + q];
    mlp<F, HD, 3>(Blob<F, NB, HD, 10, 3>::ons(sw, g.ns, sp(species, i, g.ns)), x, y);
    for (int mu = 0; mu < 9; ++mu) onsite[(size_t)mu * n + i] = y[mu == 0 ? 0 : (mu < 4 ? 1 : 2)];
  }
}

__global__ void species_check_kernel(const int32_t* __restrict__ species, int64_t n, int32_t ns,
                                     int32_t* status) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
    if (species[i] < 0 || species[i] >= ns) atomicOr(status, 1);
}

template <int F, int NB, int HD>
int run(const gtb_mlp_model* m, const double* pos, const int32_t* species, const MlpGeom& g, gtb_ell* H,
        double* v, cudaStream_t st) {
  const size_t smem = sizeof(double) * Blob<F, NB, HD>::size(g.ns);
  if (smem > 200 * 1024) return GTB_ERR_INVALID_ARG;
  GTB_CUDA_TRY(cudaFuncSetAttribute(node_feature_kernel<F, NB, HD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  GTB_CUDA_TRY(cudaFuncSetAttribute(mlp_hopping_kernel<F, NB, HD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  GTB_CUDA_TRY(cudaFuncSetAttribute(mlp_onsite_kernel<F, NB, HD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int64_t n = H->n;
  auto grid = [](int64_t total) {
    return (int)std::max<int64_t>(1, std::min<int64_t>((total + kBlock - 1) / kBlock, kSmCount * 4));
  };
  node_feature_kernel<F, NB, HD><<<grid(n), kBlock, smem, st>>>(H->cols, n, H->width, pos, species, g,
                                                                m->weights, v);
  GTB_LAUNCHED();
  if (H->width > 0) {
    mlp_hopping_kernel<F, NB, HD><<<grid(n * H->width), kBlock, smem, st>>>(H->cols, n, H->width, pos,
                                                                            species, g, m->weights, v, H->vals);
    GTB_LAUNCHED();
  }
  if (H->diag) {
    mlp_onsite_kernel<F, NB, HD><<<grid(n), kBlock, smem, st>>>(n, species, g, m->weights, v, H->diag);
    GTB_LAUNCHED();
  }
  return GTB_OK;
}

template <int F, int NB, int HD>
int run_sk(const gtb_mlp_model* m, const gtb_ell* nbr, const double* pos, const int32_t* species,
           const MlpGeom& g, gtb_ell* H, double* v, cudaStream_t st) {
  // node features with the (4, 2)-output blob: only the c table is read, which sits first in both layouts
  const size_t smem = sizeof(double) * Blob<F, NB, HD, 4, 2>::size(g.ns);
  if (smem > 200 * 1024) return GTB_ERR_INVALID_ARG;
  GTB_CUDA_TRY(cudaFuncSetAttribute(node_feature_kernel<F, NB, HD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  GTB_CUDA_TRY(cudaFuncSetAttribute(mlp_sk_block_kernel<F, NB, HD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  GTB_CUDA_TRY(cudaFuncSetAttribute(mlp_sk_onsite_kernel<F, NB, HD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int64_t n = nbr->n;
  auto grid = [](int64_t total) {
    return (int)std::max<int64_t>(1, std::min<int64_t>((total + kBlock - 1) / kBlock, kSmCount * 4));
  };
  node_feature_kernel<F, NB, HD><<<grid(n), kBlock, smem, st>>>(nbr->cols, n, nbr->width, pos, species, g,
                                                                m->weights, v);
  GTB_LAUNCHED();
  if (nbr->width > 0) {
    mlp_sk_block_kernel<F, NB, HD><<<grid(n * nbr->width), kBlock, smem, st>>>(
        nbr->cols, n, nbr->width, pos, species, g, m->weights, v, H->cols, H->vals);
    GTB_LAUNCHED();
  }
  if (H->diag) {
    mlp_sk_onsite_kernel<F, NB, HD><<<grid(n), kBlock, smem, st>>>(n, species, g, m->weights, v, H->diag);
    GTB_LAUNCHED();
  }
  return GTB_OK;
}

template <int F, int NB, int HD>
int run_spd(const gtb_mlp_model* m, const gtb_ell* nbr, const double* pos, const int32_t* species,
            const MlpGeom& g, gtb_ell* Hb, double* v, cudaStream_t st) {
  const size_t smem = sizeof(double) * Blob<F, NB, HD, 10, 3>::size(g.ns);
  if (smem > 200 * 1024) return GTB_ERR_INVALID_ARG;
  GTB_CUDA_TRY(cudaFuncSetAttribute(node_feature_kernel<F, NB, HD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  GTB_CUDA_TRY(cudaFuncSetAttribute(mlp_spd_block_kernel<F, NB, HD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  GTB_CUDA_TRY(cudaFuncSetAttribute(mlp_spd_onsite_kernel<F, NB, HD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int64_t n = nbr->n;
  auto grid = [](int64_t total, int threads) {
    return (int)std::max<int64_t>(1, std::min<int64_t>((total + threads - 1) / threads, kSmCount * 4));
  };
  node_feature_kernel<F, NB, HD><<<grid(n, kBlock), kBlock, smem, st>>>(nbr->cols, n, nbr->width, pos, species, g,
                                                                        m->weights, v);
  GTB_LAUNCHED();
  if (nbr->width > 0) {
    mlp_spd_block_kernel<F, NB, HD><<<grid(n * nbr->width, 128), 128, smem, st>>>(
        nbr->cols, n, nbr->width, pos, species, g, m->weights, v, Hb->vals);
    GTB_LAUNCHED();
  }
  if (Hb->diag) {
    mlp_spd_onsite_kernel<F, NB, HD><<<grid(n, kBlock), kBlock, smem, st>>>(n, species, g, m->weights, v, Hb->diag);
    GTB_LAUNCHED();
  }
  return GTB_OK;
}

}  // namespace
}  // namespace gtb

using namespace gtb;

extern "C" size_t gtb_mlp_weight_count(int32_t ns, int32_t F, int32_t Nb, int32_t Hd) {
  if (ns <= 0 || F <= 0 || Nb <= 0 || Hd <= 0) return 0;
  return (size_t)ns * ns * F * Nb + ((size_t)Hd * F + Hd + (size_t)F * Hd + F) +
         (size_t)(ns + 1) * ((size_t)Hd * F + Hd + Hd + 1);
}

extern "C" int gtb_mlp_hamiltonian(const gtb_mlp_model* m, const double* pos, const int32_t* species,
                                   const double box[3], const int32_t pbc[3], gtb_ell* H, double* v,
                                   int32_t* status, void* stream) {
  if (!m || !pos || !species || !box || !pbc || !H || !v || !status || !m->weights || H->n <= 0 ||
      H->width < 0 || (H->width > 0 && (!H->cols || !H->vals)) || m->n_species < 1 ||
      m->n_species > GTB_MAX_SPECIES || !(m->r_cut > 0.0))
    return GTB_ERR_INVALID_ARG;
  if (H->n > (int64_t)INT32_MAX - 64) return GTB_ERR_INDEX_RANGE;
  MlpGeom g{};
  for (int a = 0; a < 3; ++a) {
    if (pbc[a] && !(box[a] > 0.0)) return GTB_ERR_INVALID_ARG;
    g.box[a] = box[a];
    g.pbc[a] = pbc[a];
  }
  g.r_cut = m->r_cut;
  g.ns = m->n_species;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  GTB_CUDA_TRY(cudaMemsetAsync(status, 0, sizeof(int32_t), st));
  species_check_kernel<<<kSmCount, 256, 0, st>>>(species, H->n, g.ns, status);
  GTB_LAUNCHED();
  const int F = m->n_features, Nb = m->n_basis, Hd = m->n_hidden;
  if (F == 8 && Nb == 8 && Hd == 16) return run<8, 8, 16>(m, pos, species, g, H, v, st);
  if (F == 4 && Nb == 4 && Hd == 8) return run<4, 4, 8>(m, pos, species, g, H, v, st);
  if (F == 16 && Nb == 8 && Hd == 32) return run<16, 8, 32>(m, pos, species, g, H, v, st);
  return GTB_ERR_INVALID_ARG;  // sizes are compile-time in the kernels: these three are instantiated
}

extern "C" size_t gtb_mlp_sk_weight_count(int32_t ns, int32_t F, int32_t Nb, int32_t Hd) {
  if (ns <= 0 || F <= 0 || Nb <= 0 || Hd <= 0) return 0;
  return (size_t)ns * ns * F * Nb + ((size_t)Hd * F + Hd + (size_t)F * Hd + F) +
         ((size_t)Hd * F + Hd + 4 * (size_t)Hd + 4) + (size_t)ns * ((size_t)Hd * F + Hd + 2 * (size_t)Hd + 2);
}

extern "C" int gtb_mlp_sk_hamiltonian(const gtb_mlp_model* m, const gtb_ell* nbr, const double* pos,
                                      const int32_t* species, const double box[3], const int32_t pbc[3],
                                      gtb_ell* H, double* v, int32_t* status, void* stream) {
  int rc = check_ell(nbr);
  if (rc != GTB_OK) return rc;
  if (!m || !pos || !species || !box || !pbc || !H || !v || !status || !m->weights ||
      H->n != 4 * nbr->n || H->width != 4 * nbr->width || (H->width > 0 && (!H->cols || !H->vals)) ||
      m->n_species < 1 || m->n_species > GTB_MAX_SPECIES || !(m->r_cut > 0.0))
    return GTB_ERR_INVALID_ARG;
  if (H->n > (int64_t)INT32_MAX - 64) return GTB_ERR_INDEX_RANGE;
  MlpGeom g{};
  for (int a = 0; a < 3; ++a) {
    if (pbc[a] && !(box[a] > 0.0)) return GTB_ERR_INVALID_ARG;
    g.box[a] = box[a];
    g.pbc[a] = pbc[a];
  }
  g.r_cut = m->r_cut;
  g.ns = m->n_species;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  GTB_CUDA_TRY(cudaMemsetAsync(status, 0, sizeof(int32_t), st));
  species_check_kernel<<<kSmCount, 256, 0, st>>>(species, nbr->n, g.ns, status);
  GTB_LAUNCHED();
  if (m->n_features == 8 && m->n_basis == 8 && m->n_hidden == 16)
    return run_sk<8, 8, 16>(m, nbr, pos, species, g, H, v, st);
  return GTB_ERR_INVALID_ARG;  // (F, Nb, Hd) = (8, 8, 16) is the instantiated size
}

extern "C" size_t gtb_mlp_spd_weight_count(int32_t ns, int32_t F, int32_t Nb, int32_t Hd) {
  if (ns <= 0 || F <= 0 || Nb <= 0 || Hd <= 0) return 0;
  return (size_t)ns * ns * F * Nb + ((size_t)Hd * F + Hd + (size_t)F * Hd + F) +
         ((size_t)Hd * F + Hd + 10 * (size_t)Hd + 10) + (size_t)ns * ((size_t)Hd * F + Hd + 3 * (size_t)Hd + 3);
}

extern "C" int gtb_mlp_spd_blocks(const gtb_mlp_model* m, const gtb_ell* nbr, const double* pos,
                                  const int32_t* species, const double box[3], const int32_t pbc[3],
                                  gtb_ell* Hb, double* v, int32_t* status, void* stream) {
  int rc = check_ell(nbr);
  if (rc != GTB_OK) return rc;
  if (!m || !pos || !species || !box || !pbc || !Hb || !v || !status || !m->weights || Hb->n != nbr->n ||
      Hb->width != nbr->width || Hb->cols != nbr->cols || (Hb->width > 0 && !Hb->vals) ||
      (reinterpret_cast<uintptr_t>(Hb->vals) & 31u) || m->n_species < 1 || m->n_species > GTB_MAX_SPECIES ||
      !(m->r_cut > 0.0))
    return GTB_ERR_INVALID_ARG;
  if (9 * nbr->n > (int64_t)INT32_MAX - 64) return GTB_ERR_INDEX_RANGE;
  MlpGeom g{};
  for (int a = 0; a < 3; ++a) {
    if (pbc[a] && !(box[a] > 0.0)) return GTB_ERR_INVALID_ARG;
    g.box[a] = box[a];
    g.pbc[a] = pbc[a];
  }
  g.r_cut = m->r_cut;
  g.ns = m->n_species;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  GTB_CUDA_TRY(cudaMemsetAsync(status, 0, sizeof(int32_t), st));
  species_check_kernel<<<kSmCount, 256, 0, st>>>(species, nbr->n, g.ns, status);
  GTB_LAUNCHED();
  if (m->n_features == 8 && m->n_basis == 8 && m->n_hidden == 16)
    return run_spd<8, 8, 16>(m, nbr, pos, species, g, Hb, v, st);
  return GTB_ERR_INVALID_ARG;  // (F, Nb, Hd) = (8, 8, 16) is the instantiated size
}
