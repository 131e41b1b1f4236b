// CPU ORACLE (test infrastructure only; see gtbo.h) -- multi-orbital Slater-Koster blocks
// (SURVEY.md sec. 8(f) NEXT-2).
//
// What the paper fixes: the Hamiltonian is a sum of onsite blocks H_ii and hopping blocks
// H_ij^{lm,l'm'} between the orbitals (l, m) of atom i and (l', m') of atom j, obtained from
// Slater-Koster parameters and the bond direction, and
// H_ij^{l l'} = (-1)^{l+l'} H_ji^{l' l}.  It prints no Slater-Koster table; the
// two-centre s,p table is the textbook one (Slater & Koster 1954, Table I), written out here for the
// basis (s, p_x, p_y, p_z) -- reading S1 of DESIGN.md sec. 13; d orbitals are not built:
//   (l, m, n) = (x_j - x_i)/r  (minimum image), each V scaled by exp(-beta (r/r0 - 1)),
//   E_{s,s}   = V_ss_sigma
//   E_{s,pa}  =  a V_sp_sigma            (s on atom i, p_a on atom j;  a = l, m, n)
//   E_{pa,s}  = -a V_sp_sigma            (p_a on atom i, s on atom j)
//   E_{pa,pb} = a b V_pp_sigma + (delta_ab - a b) V_pp_pi
//   onsite: eps_s, eps_p (+ onsite_shift[i] on all four).
// Output: a scalar ELL matrix over the 4n orbitals, orbital index 4 i + mu, in the canonical
// layout: row (i, mu) has the 4 K entries (slot 4 k + nu, column 4 j + nu), j = the k-th neighbour
// of i in ascending order; padding slots (j = i) carry column = the row's own index and value 0.
#include "gtbo.h"

#include <cmath>

extern "C" int gtbo_sk_hamiltonian(const gtbo_ell* nbr, const double* pos, const int32_t* species,
                                   const double box[3], const int32_t pbc[3],
                                   const gtbo_sk_model* model, gtbo_ell* H) {
  if (!nbr || !pos || !species || !box || !pbc || !model || !H || !H->cols || !H->vals ||
      H->n != 4 * nbr->n || H->width != 4 * nbr->width || model->n_species <= 0)
    return GTBO_ERR_INVALID_ARG;
  const int64_t n = nbr->n, N = 4 * n;
  const int ns = model->n_species;
  for (int64_t i = 0; i < n; ++i) {
    const int si = species[i];
    if (si < 0 || si >= ns) return GTBO_ERR_INVALID_ARG;
    for (int32_t k = 0; k < nbr->width; ++k) {
      const int64_t j = nbr->cols[(size_t)k * n + i];
      double E[4][4] = {{0.0}};
      if (j != i) {
        const int sj = species[j];
        if (sj < 0 || sj >= ns) return GTBO_ERR_INVALID_ARG;
        double d[3];
        for (int a = 0; a < 3; ++a) {
          d[a] = pos[3 * j + a] - pos[3 * i + a];
          if (pbc[a]) d[a] = d[a] - box[a] * std::rint(d[a] / box[a]);
        }
        const double r = std::sqrt((d[0] * d[0] + d[1] * d[1]) + d[2] * d[2]);
        const double c[3] = {d[0] / r, d[1] / r, d[2] / r};
        const double f = model->beta == 0.0 ? 1.0 : std::exp(-model->beta * (r / model->r0 - 1.0));
        const double* V = model->sk + ((size_t)si * ns + sj) * 4;  // ss_sigma, sp_sigma, pp_sigma, pp_pi
        const double Vss = V[0] * f, Vsp = V[1] * f, Vpp_s = V[2] * f, Vpp_p = V[3] * f;
        // H_ij^{p,s} = (-1)^{1+0} H_ji^{s,p}, and H_ji^{s,p} is made of the (s on j, p on i)
        // integral, i.e. the table entry of the pair (s_j, s_i): with a species-asymmetric table
        // (V_sp(A s, B p) != V_sp(B s, A p)) this is what keeps H symmetric.  The bond direction seen
        // from j is -c, so H_ji^{s,p_a} = -c_a V_sp(ji) and E_{p_a,s} = H_ji^{s,p_a} = -c_a V_sp(ji).
        const double Vsp_ji = model->sk[((size_t)sj * ns + si) * 4 + 1] * f;
        E[0][0] = Vss;
        for (int a = 0; a < 3; ++a) {
          E[0][1 + a] = c[a] * Vsp;
          E[1 + a][0] = -(c[a] * Vsp_ji);
          for (int b = 0; b < 3; ++b)
            E[1 + a][1 + b] = c[a] * c[b] * Vpp_s + ((a == b ? 1.0 : 0.0) - c[a] * c[b]) * Vpp_p;
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
      const double shift = model->onsite_shift ? model->onsite_shift[i] : 0.0;
      H->diag[4 * i] = model->onsite_s[si] + shift;
      for (int a = 1; a < 4; ++a) H->diag[4 * i + a] = model->onsite_p[si] + shift;
    }
  }
  return GTBO_OK;
}
