// CPU ORACLE (test infrastructure only; see gtbo.h) -- Slater-Koster blocks for the s, p, d basis of the
// paper's runs (9 orbitals per atom: PAPER.md:96 "s, p, d orbital basis", :106 "approximately 1 billion
// orbitals" for 10^8 atoms); completes SURVEY.md sec. 8(f) NEXT-2.
//
// What the paper fixes: hopping blocks H_ij^{lm,l'm'} = sum_lambda MLP_lambda(e_ij) P_lambda^{lm,l'm'}(r^_ij)
// with P the Slater-Koster conversion coefficients of the bond direction and the symmetry
// H_ij^{l l'} = (-1)^{l+l'} H_ji^{l' l}.  It prints no table.  Reading S4:
// the two-centre integrals are diagonal in the bond frame, so every block follows from rotating the real
// orbitals into the frame (e1, e2, u), u = (x_j - x_i)/r:
//   s:  1;          p_alpha:  sigma -> u_alpha,  pi -> e1_alpha, e2_alpha;
//   d_a (a = xy, yz, zx, x2-y2, z2) is the quadratic form r^T A_a r with
//       A_xy = (sqrt3/2)(x y^T + y x^T) (cyclic), A_x2-y2 = (sqrt3/2)(x x^T - y y^T), A_z2 = (3 z z^T - 1)/2,
//       and <d_a|d_b> = (2/3) tr(A_a A_b); the bond-frame forms are A_sigma = (3 u u^T - 1)/2,
//       A_pi_k = (sqrt3/2)(u e_k^T + e_k u^T), A_delta1 = (sqrt3/2)(e1 e2^T + e2 e1^T),
//       A_delta2 = (sqrt3/2)(e1 e1^T - e2 e2^T);  c_{a,m} = (2/3) tr(A_a A_m).
//   E_{ab} = sum_m c_{a,m} V_{l_a l_b |m|} c_{b,m}  for l_a <= l_b, and (-1)^{l_a + l_b} times that for l_a > l_b.
// The ten integrals per species pair: ss_sigma, sp_sigma, pp_sigma, pp_pi, sd_sigma, pd_sigma, pd_pi,
// dd_sigma, dd_pi, dd_delta, each scaled by exp(-beta (r/r0 - 1)); onsite eps_s, eps_p, eps_d.
// Orbital order: s, px, py, pz, dxy, dyz, dzx, dx2-y2, dz2.  Output: scalar ELL over the 9n orbitals in
// the layout of gtbo_sk.cpp with 9 in place of 4.
#include "gtbo.h"

#include <cmath>

namespace {

constexpr int kOrb = 9;
const int kL[kOrb] = {0, 1, 1, 1, 2, 2, 2, 2, 2};

// c[a][m]: coefficient of bond-frame orbital m (0: sigma, 1-2: pi, 3-4: delta) in lab orbital a
void frame_coefficients(const double u[3], double c[kOrb][5]) {
  // any orthonormal e1, e2 perpendicular to u: the pi and delta sums do not depend on the choice
  double t[3] = {0.0, 0.0, 1.0};
  if (std::fabs(u[2]) > 0.9) { t[0] = 1.0; t[2] = 0.0; }
  double e1[3] = {u[1] * t[2] - u[2] * t[1], u[2] * t[0] - u[0] * t[2], u[0] * t[1] - u[1] * t[0]};
  const double n1 = std::sqrt(e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2]);
  for (int a = 0; a < 3; ++a) e1[a] /= n1;
  const double e2[3] = {u[1] * e1[2] - u[2] * e1[1], u[2] * e1[0] - u[0] * e1[2], u[0] * e1[1] - u[1] * e1[0]};
  for (int a = 0; a < kOrb; ++a)
    for (int m = 0; m < 5; ++m) c[a][m] = 0.0;
  c[0][0] = 1.0;
  for (int a = 0; a < 3; ++a) {
    c[1 + a][0] = u[a];
    c[1 + a][1] = e1[a];
    c[1 + a][2] = e2[a];
  }
  const double s3 = std::sqrt(3.0);
  double A[5][3][3] = {};   // lab d orbitals
  A[0][0][1] = A[0][1][0] = s3 / 2;            // xy
  A[1][1][2] = A[1][2][1] = s3 / 2;            // yz
  A[2][2][0] = A[2][0][2] = s3 / 2;            // zx
  A[3][0][0] = s3 / 2; A[3][1][1] = -s3 / 2;   // x2 - y2
  A[4][0][0] = A[4][1][1] = -0.5; A[4][2][2] = 1.0;  // 3z2 - r2
  double Bm[5][3][3];       // bond-frame d orbitals
  for (int p = 0; p < 3; ++p)
    for (int q = 0; q < 3; ++q) {
      Bm[0][p][q] = 1.5 * u[p] * u[q] - (p == q ? 0.5 : 0.0);
      Bm[1][p][q] = s3 / 2 * (u[p] * e1[q] + e1[p] * u[q]);
      Bm[2][p][q] = s3 / 2 * (u[p] * e2[q] + e2[p] * u[q]);
      Bm[3][p][q] = s3 / 2 * (e1[p] * e2[q] + e2[p] * e1[q]);
      Bm[4][p][q] = s3 / 2 * (e1[p] * e1[q] - e2[p] * e2[q]);
    }
  for (int a = 0; a < 5; ++a)
    for (int m = 0; m < 5; ++m) {
      double tr = 0.0;
      for (int p = 0; p < 3; ++p)
        for (int q = 0; q < 3; ++q) tr += A[a][p][q] * Bm[m][q][p];
      c[4 + a][m] = 2.0 / 3.0 * tr;
    }
}

// V_{l l' |m|}, l <= l', from the ten integrals (already scaled)
double integral(const double* V, int l, int lp, int m) {
  const int am = m == 0 ? 0 : (m <= 2 ? 1 : 2);
  if (l == 0 && lp == 0) return am == 0 ? V[0] : 0.0;
  if (l == 0 && lp == 1) return am == 0 ? V[1] : 0.0;
  if (l == 1 && lp == 1) return am == 0 ? V[2] : (am == 1 ? V[3] : 0.0);
  if (l == 0 && lp == 2) return am == 0 ? V[4] : 0.0;
  if (l == 1 && lp == 2) return am == 0 ? V[5] : (am == 1 ? V[6] : 0.0);
  return am == 0 ? V[7] : (am == 1 ? V[8] : V[9]);   // d-d
}

// E[a][b] from the bond direction u and the (already scaled) integrals V of (s_i, s_j), Vt of (s_j, s_i)
void block_from_integrals(const double u[3], const double* V, const double* Vt, double E[kOrb][kOrb]) {
  double c[kOrb][5];
  frame_coefficients(u, c);
  for (int a = 0; a < kOrb; ++a)
    for (int b = 0; b < kOrb; ++b) {
      const int la = kL[a], lb = kL[b];
      const int lo = la < lb ? la : lb, hi = la < lb ? lb : la;
      double s = 0.0;
      for (int m = 0; m < 5; ++m) s += c[a][m] * integral(la > lb ? Vt : V, lo, hi, m) * c[b][m];
      E[a][b] = (la > lb && ((la + lb) & 1)) ? -s : s;
    }
}

// the 9x9 hopping block E[a][b] of the pair (i, j), j != i: the construction of the file header
void pair_block(const double* pos, const double box[3], const int32_t pbc[3], const gtbo_spd_model* model,
                int64_t i, int64_t j, int si, int sj, double E[kOrb][kOrb]) {
  const int ns = model->n_species;
  double d[3];
  for (int a = 0; a < 3; ++a) {
    d[a] = pos[3 * j + a] - pos[3 * i + a];
    if (pbc[a]) d[a] = d[a] - box[a] * std::rint(d[a] / box[a]);
  }
  const double r = std::sqrt((d[0] * d[0] + d[1] * d[1]) + d[2] * d[2]);
  const double u[3] = {d[0] / r, d[1] / r, d[2] / r};
  const double f = model->beta == 0.0 ? 1.0 : std::exp(-model->beta * (r / model->r0 - 1.0));
  // V: integrals of the pair (s_i, s_j), used for l_a <= l_b; Vt: those of (s_j, s_i), used for
  // l_a > l_b -- PAPER.md:88, H_ij^{l l'} = (-1)^{l+l'} H_ji^{l' l}: the (l_a > l_b) element of the
  // (i, j) block is the (l_b, l_a) element of the (j, i) block, whose lower-l orbital sits on j.
  double V[10], Vt[10];
  for (int q = 0; q < 10; ++q) {
    V[q] = model->sk[((size_t)si * ns + sj) * 10 + q] * f;
    Vt[q] = model->sk[((size_t)sj * ns + si) * 10 + q] * f;
  }
  block_from_integrals(u, V, Vt, E);
}

}  // namespace

extern "C" int gtbo_spd_hamiltonian(const gtbo_ell* nbr, const double* pos, const int32_t* species,
                                    const double box[3], const int32_t pbc[3],
                                    const gtbo_spd_model* model, gtbo_ell* H) {
  if (!nbr || !pos || !species || !box || !pbc || !model || !H || !H->cols || !H->vals ||
      H->n != kOrb * nbr->n || H->width != kOrb * nbr->width || model->n_species <= 0)
    return GTBO_ERR_INVALID_ARG;
  const int64_t n = nbr->n, N = kOrb * n;
  const int ns = model->n_species;
  for (int64_t i = 0; i < n; ++i) {
    const int si = species[i];
    if (si < 0 || si >= ns) return GTBO_ERR_INVALID_ARG;
    for (int32_t k = 0; k < nbr->width; ++k) {
      const int64_t j = nbr->cols[(size_t)k * n + i];
      double E[kOrb][kOrb] = {{0.0}};
      if (j != i) {
        const int sj = species[j];
        if (sj < 0 || sj >= ns) return GTBO_ERR_INVALID_ARG;
        pair_block(pos, box, pbc, model, i, j, si, sj, E);
      }
      for (int mu = 0; mu < kOrb; ++mu)
        for (int nu = 0; nu < kOrb; ++nu) {
          const size_t at = (size_t)(kOrb * k + nu) * N + (kOrb * i + mu);
          H->cols[at] = (int32_t)(j != i ? kOrb * j + nu : kOrb * i + mu);
          H->vals[at] = j != i ? E[mu][nu] : 0.0;
        }
    }
    if (H->diag) {
      const double shift = model->onsite_shift ? model->onsite_shift[i] : 0.0;
      for (int a = 0; a < kOrb; ++a)
        H->diag[kOrb * i + a] = (kL[a] == 0 ? model->onsite_s[si] : kL[a] == 1 ? model->onsite_p[si]
                                                                               : model->onsite_d[si]) + shift;
    }
  }
  return GTBO_OK;
}

// One Chebyshev step of the orbital matrix on SAMPLED atoms, without materialising H (at 10^8 atoms the
// scalar ELL of gtbo_spd_hamiltonian would need 10^12 bytes): for every listed atom i the blocks of its
// pairs are built exactly as above and applied to the neighbours' orbital rows,
//   out[q][mu] = ((H x)_{9 i + mu} - b x_{9 i + mu}) * (first ? 1/a : 2/a)  [- prev_{9 i + mu} unless first],
// row sum in slot order 9 k + nu, then the onsite term: the order of gtbo_kpm_step_rows on the scalar ELL.
// The vectors are given SPARSELY: x_own [n_rows][9][R][2] (rows of the listed atoms), x_nbr
// [n_rows][K][9][R][2] (rows of their neighbours, slot by slot; padding slots ignored), prev like x_own.
extern "C" int gtbo_spd_step_atoms(const gtbo_ell* nbr, const double* pos, const int32_t* species,
                                   const double box[3], const int32_t pbc[3], const gtbo_spd_model* model,
                                   double a, double b, int32_t first, int32_t R, const int64_t* atoms,
                                   int64_t n_rows, const double* x_own, const double* x_nbr,
                                   const double* prev, double* out) {
  if (!nbr || !pos || !species || !box || !pbc || !model || !atoms || !x_own || !x_nbr || !out ||
      (!first && !prev) || R <= 0 || model->n_species <= 0)
    return GTBO_ERR_INVALID_ARG;
  const int64_t n = nbr->n;
  const int32_t K = nbr->width;
  const int ns = model->n_species;
  for (int64_t q = 0; q < n_rows; ++q) {
    const int64_t i = atoms[q];
    if (i < 0 || i >= n) return GTBO_ERR_INVALID_ARG;
    const int si = species[i];
    if (si < 0 || si >= ns) return GTBO_ERR_INVALID_ARG;
    const double shift = model->onsite_shift ? model->onsite_shift[i] : 0.0;
    for (int mu = 0; mu < kOrb; ++mu)
      for (int32_t r = 0; r < R; ++r)
        for (int c = 0; c < 2; ++c) {
          double acc = 0.0;
          for (int32_t k = 0; k < K; ++k) {
            const int64_t j = nbr->cols[(size_t)k * n + i];
            if (j == i) continue;
            const int sj = species[j];
            if (sj < 0 || sj >= ns) return GTBO_ERR_INVALID_ARG;
            double E[kOrb][kOrb];
            pair_block(pos, box, pbc, model, i, j, si, sj, E);
            for (int nu = 0; nu < kOrb; ++nu)
              acc = acc + E[mu][nu] * x_nbr[((((size_t)q * K + k) * kOrb + nu) * R + r) * 2 + c];
          }
          const double own = x_own[(((size_t)q * kOrb + mu) * R + r) * 2 + c];
          const double eps = (kL[mu] == 0 ? model->onsite_s[si] : kL[mu] == 1 ? model->onsite_p[si]
                                                                              : model->onsite_d[si]) + shift;
          acc = acc + eps * own;
          double v = (acc - b * own) * ((first ? 1.0 : 2.0) / a);
          if (!first) v = v - prev[(((size_t)q * kOrb + mu) * R + r) * 2 + c];
          out[(((size_t)q * kOrb + mu) * R + r) * 2 + c] = v;
        }
  }
  return GTBO_OK;
}

// The step of the construction that turns a bond direction and ten two-centre integrals into the 9x9 block
// (exported for gtbo_mlp.cpp, where the integrals come from MLP_lambda instead of a species table, and for the
// tests): E [9][9] row-major; V for l_a <= l_b, Vt for l_a > l_b.
extern "C" int gtbo_spd_block_from_integrals(const double u[3], const double* V, const double* Vt, double* E) {
  if (!u || !V || !Vt || !E) return GTBO_ERR_INVALID_ARG;
  double B[kOrb][kOrb];
  block_from_integrals(u, V, Vt, B);
  for (int a = 0; a < kOrb; ++a)
    for (int b = 0; b < kOrb; ++b) E[a * kOrb + b] = B[a][b];
  return GTBO_OK;
}
