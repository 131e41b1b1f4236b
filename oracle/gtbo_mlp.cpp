// CPU ORACLE (test infrastructure only; see gtbo.h) -- environment-dependent hopping and onsite
// energies from the paper's descriptor and MLPs, one orbital per atom.
//
// What the paper fixes (Eq. 2 and the text around it):
//   f_k(r)   = 1/2 [ T_k( 2 (r/r_cut - 1)^2 - 1 ) + 1 ] f_c(r)          (Chebyshev radial functions)
//   C_n(r_ij) = sum_k c_nk^{ij} f_k(r_ij),  c depends on the types of atoms i and j
//   v_i      = sum_{j in N(i)} C_n(r_ij)                                  (node feature)
//   e_ij     = C_n(r_ij) * MLP_e( sum_{k in N(i)} C_n(r_ik) + sum_{l in N(j)} C_n(r_jl) )   (edge feature)
//   hopping  = MLP_lambda(e_ij)  (one SK parameter here: the p_z - p_z integral, so t_ij itself)
//   onsite   = MLP_{l,alpha}(v_i), alpha = type of atom i;  MLPs use the SiLU activation.
// Readings: E1 f_c(r) = 1/2 [1 + cos(pi r / r_cut)] ("smooth cutoff function",
// not printed); E2 k = 0..N_b-1, n = 0..F-1, "*" in e_ij is the element-wise product; E3 every MLP is
// input -> hidden (SiLU) -> output (linear), one set of weights for MLP_e and MLP_lambda, one per
// species for the onsite MLP; E4 weights are synthetic inputs (the trained ones are not available).
// Weight blob layout (doubles): c [ns][ns][F][Nb] | MLP_e: W1 [Hd][F], b1 [Hd], W2 [F][Hd], b2 [F] |
// MLP_lambda: W1 [Hd][F], b1 [Hd], W2 [Hd], b2 [1] | per species: W1 [Hd][F], b1 [Hd], W2 [Hd], b2 [1].
#include "gtbo.h"

#include <cmath>
#include <vector>

namespace {

double silu(double x) { return x / (1.0 + std::exp(-x)); }

struct Layout {
  int ns, F, Nb, Hd;
  const double* w;
  const double* c(int si, int sj) const { return w + ((size_t)si * ns + sj) * F * Nb; }
  const double* env() const { return w + (size_t)ns * ns * F * Nb; }
  const double* hop() const { return env() + (size_t)Hd * F + Hd + (size_t)F * Hd + F; }
  const double* ons(int s) const { return hop() + (size_t)Hd * F + Hd + Hd + 1 + (size_t)s * ((size_t)Hd * F + Hd + Hd + 1); }
};

// y = W2 silu(W1 x + b1) + b2, out_dim outputs
void mlp(const double* p, int F, int Hd, int out_dim, const double* x, double* y) {
  const double* W1 = p;
  const double* b1 = W1 + (size_t)Hd * F;
  const double* W2 = b1 + Hd;
  const double* b2 = W2 + (size_t)out_dim * Hd;
  std::vector<double> h(Hd);
  for (int a = 0; a < Hd; ++a) {
    double s = b1[a];
    for (int n = 0; n < F; ++n) s += W1[(size_t)a * F + n] * x[n];
    h[a] = silu(s);
  }
  for (int o = 0; o < out_dim; ++o) {
    double s = b2[o];
    for (int a = 0; a < Hd; ++a) s += W2[(size_t)o * Hd + a] * h[a];
    y[o] = s;
  }
}

double distance(const double* pos, int64_t i, int64_t j, const double box[3], const int32_t pbc[3]) {
  double d[3];
  for (int a = 0; a < 3; ++a) {
    d[a] = pos[3 * j + a] - pos[3 * i + a];
    if (pbc[a]) d[a] = d[a] - box[a] * std::rint(d[a] / box[a]);
  }
  return std::sqrt((d[0] * d[0] + d[1] * d[1]) + d[2] * d[2]);
}

// C_n(r), n = 0..F-1, for the species pair whose coefficients are c [F][Nb]
void descriptor(const double* c, int F, int Nb, double r, double r_cut, double* C) {
  const double pi = 3.14159265358979323846;
  const double fc = r < r_cut ? 0.5 * (1.0 + std::cos(pi * r / r_cut)) : 0.0;
  const double q = r / r_cut - 1.0;
  const double x = 2.0 * q * q - 1.0;
  for (int n = 0; n < F; ++n) C[n] = 0.0;
  double t_prev = 1.0, t_cur = x;  // T_0, T_1
  for (int k = 0; k < Nb; ++k) {
    double Tk;
    if (k == 0) {
      Tk = 1.0;
    } else if (k == 1) {
      Tk = x;
    } else {
      Tk = 2.0 * x * t_cur - t_prev;  // T_k = 2 x T_{k-1} - T_{k-2}
      t_prev = t_cur;
      t_cur = Tk;
    }
    const double f = 0.5 * (Tk + 1.0) * fc;
    for (int n = 0; n < F; ++n) C[n] += c[(size_t)n * Nb + k] * f;
  }
}

}  // namespace

extern "C" int gtbo_mlp_descriptor(const gtbo_mlp_model* m, int32_t si, int32_t sj, double r, double* C) {
  if (!m || !C || si < 0 || sj < 0 || si >= m->n_species || sj >= m->n_species) return GTBO_ERR_INVALID_ARG;
  const Layout L{m->n_species, m->n_features, m->n_basis, m->n_hidden, m->weights};
  descriptor(L.c(si, sj), L.F, L.Nb, r, m->r_cut, C);
  return GTBO_OK;
}

// v [n][F] (optional output), H->vals / H->diag filled on the pattern H->cols (neighbour lists)
extern "C" int gtbo_mlp_hamiltonian(const gtbo_mlp_model* m, const double* pos, const int32_t* species,
                                    const double box[3], const int32_t pbc[3], gtbo_ell* H, double* v_out) {
  if (!m || !pos || !species || !box || !pbc || !H || !H->cols || !H->vals || !m->weights ||
      m->n_species <= 0 || m->n_features <= 0 || m->n_basis <= 0 || m->n_hidden <= 0 || !(m->r_cut > 0.0))
    return GTBO_ERR_INVALID_ARG;
  const Layout L{m->n_species, m->n_features, m->n_basis, m->n_hidden, m->weights};
  const int64_t n = H->n;
  const int F = L.F;
  std::vector<double> v((size_t)n * F, 0.0), C(F), u(F), env(F), e(F);
  for (int64_t i = 0; i < n; ++i)  // node features
    for (int32_t k = 0; k < H->width; ++k) {
      const int64_t j = H->cols[(size_t)k * n + i];
      if (j == i) continue;
      descriptor(L.c(species[i], species[j]), F, L.Nb, distance(pos, i, j, box, pbc), m->r_cut, C.data());
      for (int q = 0; q < F; ++q) v[(size_t)i * F + q] += C[q];
    }
  for (int64_t i = 0; i < n; ++i) {
    for (int32_t k = 0; k < H->width; ++k) {
      const int64_t j = H->cols[(size_t)k * n + i];
      double t = 0.0;
      if (j != i) {
        descriptor(L.c(species[i], species[j]), F, L.Nb, distance(pos, i, j, box, pbc), m->r_cut, C.data());
        for (int q = 0; q < F; ++q) u[q] = v[(size_t)i * F + q] + v[(size_t)j * F + q];
        mlp(L.env(), F, L.Hd, F, u.data(), env.data());
        for (int q = 0; q < F; ++q) e[q] = C[q] * env[q];
        mlp(L.hop(), F, L.Hd, 1, e.data(), &t);
      }
      H->vals[(size_t)k * n + i] = t;
    }
    if (H->diag) mlp(L.ons(species[i]), F, L.Hd, 1, &v[(size_t)i * F], &H->diag[i]);
  }
  if (v_out) for (size_t q = 0; q < v.size(); ++q) v_out[q] = v[q];
  return GTBO_OK;
}

// ---- Eq. 2 feeding the Slater-Koster blocks: the paper's full hopping formula ----------------------
//   H_ij^{lm,l'm'} = sum_lambda MLP_lambda(e_ij) P_lambda^{lm,l'm'}(r^_ij),   H_ii^{lm,lm} = MLP_{l,alpha}(v_i)
// for the s,p basis: MLP_lambda has four outputs, the bond integrals ss_sigma, sp_sigma,
// pp_sigma, pp_pi of the pair, which enter the two-centre table of gtbo_sk.cpp; the onsite MLP has two
// outputs (eps_s, eps_p).  Reading E6: one MLP_lambda with a 4-vector output
// instead of four networks.  Blob layout as above with MLP_lambda: W1 [Hd][F], b1 [Hd], W2 [4][Hd],
// b2 [4] and per species: W1 [Hd][F], b1 [Hd], W2 [2][Hd], b2 [2].
extern "C" int gtbo_mlp_sk_hamiltonian(const gtbo_mlp_model* m, const gtbo_ell* nbr, const double* pos,
                                       const int32_t* species, const double box[3],
                                       const int32_t pbc[3], gtbo_ell* H) {
  if (!m || !nbr || !pos || !species || !box || !pbc || !H || !H->cols || !H->vals || !m->weights ||
      H->n != 4 * nbr->n || H->width != 4 * nbr->width || !(m->r_cut > 0.0))
    return GTBO_ERR_INVALID_ARG;
  const int ns = m->n_species, F = m->n_features, Nb = m->n_basis, Hd = m->n_hidden;
  const double* w = m->weights;
  const double* w_env = w + (size_t)ns * ns * F * Nb;
  const double* w_hop = w_env + (size_t)Hd * F + Hd + (size_t)F * Hd + F;
  const size_t hop_size = (size_t)Hd * F + Hd + 4 * (size_t)Hd + 4;
  const size_t ons_size = (size_t)Hd * F + Hd + 2 * (size_t)Hd + 2;
  const int64_t n = nbr->n, N = 4 * n;
  std::vector<double> v((size_t)n * F, 0.0), C(F), u(F), env(F), e(F);
  for (int64_t i = 0; i < n; ++i)
    for (int32_t k = 0; k < nbr->width; ++k) {
      const int64_t j = nbr->cols[(size_t)k * n + i];
      if (j == i) continue;
      descriptor(w + ((size_t)species[i] * ns + species[j]) * F * Nb, F, Nb, distance(pos, i, j, box, pbc),
                 m->r_cut, C.data());
      for (int q = 0; q < F; ++q) v[(size_t)i * F + q] += C[q];
    }
  for (int64_t i = 0; i < n; ++i) {
    for (int32_t k = 0; k < nbr->width; ++k) {
      const int64_t j = nbr->cols[(size_t)k * n + i];
      double E[4][4] = {{0.0}};
      if (j != i) {
        double d[3];
        for (int a = 0; a < 3; ++a) {
          d[a] = pos[3 * j + a] - pos[3 * i + a];
          if (pbc[a]) d[a] = d[a] - box[a] * std::rint(d[a] / box[a]);
        }
        const double r = std::sqrt((d[0] * d[0] + d[1] * d[1]) + d[2] * d[2]);
        const double c[3] = {d[0] / r, d[1] / r, d[2] / r};
        descriptor(w + ((size_t)species[i] * ns + species[j]) * F * Nb, F, Nb, r, m->r_cut, C.data());
        for (int q = 0; q < F; ++q) u[q] = v[(size_t)i * F + q] + v[(size_t)j * F + q];
        mlp(w_env, F, Hd, F, u.data(), env.data());
        for (int q = 0; q < F; ++q) e[q] = C[q] * env[q];
        double V[4];
        mlp(w_hop, F, Hd, 4, e.data(), V);
        E[0][0] = V[0];
        for (int a = 0; a < 3; ++a) {
          E[0][1 + a] = c[a] * V[1];
          E[1 + a][0] = -(c[a] * V[1]);
          for (int b = 0; b < 3; ++b)
            E[1 + a][1 + b] = c[a] * c[b] * V[2] + ((a == b ? 1.0 : 0.0) - c[a] * c[b]) * V[3];
        }
      }
      for (int mu = 0; mu < 4; ++mu)
        for (int nu = 0; nu < 4; ++nu) {
          const size_t at = (size_t)(4 * k + nu) * N + (4 * i + mu);
          H->cols[at] = (int32_t)(j != i ? 4 * j + nu : 4 * i + mu);
          H->vals[at] = j != i ? E[mu][nu] : 0.0;
        }
    }
    if (H->diag) {
      double eps[2];
      mlp(w_hop + hop_size + (size_t)species[i] * ons_size, F, Hd, 2, &v[(size_t)i * F], eps);
      H->diag[4 * i] = eps[0];
      for (int a = 1; a < 4; ++a) H->diag[4 * i + a] = eps[1];
    }
  }
  return GTBO_OK;
}

// Eq. 2 feeding the s,p,d Slater-Koster blocks (reading E7 of DESIGN.md sec. 14): the
// paper's model.  MLP_lambda has TEN outputs, the two-centre integrals ss_sigma, sp_sigma, pp_sigma, pp_pi,
// sd_sigma, pd_sigma, pd_pi, dd_sigma, dd_pi, dd_delta of the pair, which enter the block construction of
// gtbo_spd.cpp; the onsite MLPs have three (eps_s, eps_p, eps_d).  e_ij = e_ji (c is symmetric in the species
// pair), so the same integrals serve both orderings of the pair.  Weight blob as gtbo_mlp_sk_hamiltonian's
// with 10 / 3 in place of 4 / 2.  Output: scalar ELL over the 9n orbitals as gtbo_spd_hamiltonian's.
extern "C" int gtbo_mlp_spd_hamiltonian(const gtbo_mlp_model* m, const gtbo_ell* nbr, const double* pos,
                                        const int32_t* species, const double box[3],
                                        const int32_t pbc[3], gtbo_ell* H) {
  if (!m || !nbr || !pos || !species || !box || !pbc || !H || !H->cols || !H->vals || !m->weights ||
      H->n != 9 * nbr->n || H->width != 9 * nbr->width || !(m->r_cut > 0.0))
    return GTBO_ERR_INVALID_ARG;
  const int ns = m->n_species, F = m->n_features, Nb = m->n_basis, Hd = m->n_hidden;
  const double* w = m->weights;
  const double* w_env = w + (size_t)ns * ns * F * Nb;
  const double* w_hop = w_env + (size_t)Hd * F + Hd + (size_t)F * Hd + F;
  const size_t hop_size = (size_t)Hd * F + Hd + 10 * (size_t)Hd + 10;
  const size_t ons_size = (size_t)Hd * F + Hd + 3 * (size_t)Hd + 3;
  const int64_t n = nbr->n, N = 9 * n;
  std::vector<double> v((size_t)n * F, 0.0), C(F), u(F), env(F), e(F);
  for (int64_t i = 0; i < n; ++i)
    for (int32_t k = 0; k < nbr->width; ++k) {
      const int64_t j = nbr->cols[(size_t)k * n + i];
      if (j == i) continue;
      descriptor(w + ((size_t)species[i] * ns + species[j]) * F * Nb, F, Nb, distance(pos, i, j, box, pbc),
                 m->r_cut, C.data());
      for (int q = 0; q < F; ++q) v[(size_t)i * F + q] += C[q];
    }
  for (int64_t i = 0; i < n; ++i) {
    for (int32_t k = 0; k < nbr->width; ++k) {
      const int64_t j = nbr->cols[(size_t)k * n + i];
      double E[81] = {0.0};
      if (j != i) {
        double d[3];
        for (int a = 0; a < 3; ++a) {
          d[a] = pos[3 * j + a] - pos[3 * i + a];
          if (pbc[a]) d[a] = d[a] - box[a] * std::rint(d[a] / box[a]);
        }
        const double r = std::sqrt((d[0] * d[0] + d[1] * d[1]) + d[2] * d[2]);
        const double dir[3] = {d[0] / r, d[1] / r, d[2] / r};
        descriptor(w + ((size_t)species[i] * ns + species[j]) * F * Nb, F, Nb, r, m->r_cut, C.data());
        for (int q = 0; q < F; ++q) u[q] = v[(size_t)i * F + q] + v[(size_t)j * F + q];
        mlp(w_env, F, Hd, F, u.data(), env.data());
        for (int q = 0; q < F; ++q) e[q] = C[q] * env[q];
        double V[10];
        mlp(w_hop, F, Hd, 10, e.data(), V);
        gtbo_spd_block_from_integrals(dir, V, V, E);
      }
      for (int mu = 0; mu < 9; ++mu)
        for (int nu = 0; nu < 9; ++nu) {
          const size_t at = (size_t)(9 * k + nu) * N + (9 * i + mu);
          H->cols[at] = (int32_t)(j != i ? 9 * j + nu : 9 * i + mu);
          H->vals[at] = j != i ? E[9 * mu + nu] : 0.0;
        }
    }
    if (H->diag) {
      double eps[3];
      mlp(w_hop + hop_size + (size_t)species[i] * ons_size, F, Hd, 3, &v[(size_t)i * F], eps);
      H->diag[9 * i] = eps[0];
      for (int a = 1; a < 4; ++a) H->diag[9 * i + a] = eps[1];
      for (int a = 4; a < 9; ++a) H->diag[9 * i + a] = eps[2];
    }
  }
  return GTBO_OK;
}
