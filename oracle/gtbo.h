/*
 * gtbo.h -- CPU ORACLE for the KPM / LSQT density-of-states path of GPUTB
 * (arxiv/paper_2509_06525).  TEST INFRASTRUCTURE ONLY.
 *
 * This is a plain, slow, obviously-correct restatement of what the hot path
 * computes, written from the paper and from BASELINE.json:north_star
 * (the paper names the ingredients of the method at PAPER.md:55 (sec. 2.4) but
 * prints no recursion; the textbook KPM identities used are written out in
 * SURVEY.md sec. 8(c) C1-C7 and restated beside each function below).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this library.  The product (the CUDA path
 * under paper_2509_06525_b200/) never does, and shares no code, header,
 * table or helper with it: this header is private to oracle/.
 *
 * All pointers are HOST pointers.  All arrays are caller-owned.
 * Layouts (the interface contract of the boundary):
 *   pos      double [n][3]            Cartesian coordinates, Angstrom, unwrapped
 *   species  int32  [n]
 *   ELL      cols int32 [width][n], vals double [width][n]  (slot-major);
 *            row i's entries sorted by ascending column; padding slots have
 *            col = i and val = +0.0;  diag double [n] or NULL (= all zero)
 *   phi      double [n][R][2]         complex128, vectors interleaved per atom
 *   mu       double [M]
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"): every function below is
 * pinned by something other than itself -- closed-form honeycomb eigenvalues,
 * closed-walk counts, numpy eigvalsh on tiny lattices, brute force O(N^2)
 * neighbour lists, the published splitmix64 first output, Jackson-kernel
 * positivity / normalisation.  No function here is "parity unpinned".
 */
#ifndef GTBO_H
#define GTBO_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
  GTBO_OK = 0,
  GTBO_ERR_INVALID_ARG = -1,
  GTBO_ERR_BOX_TOO_SMALL = -2, /* a periodic length < 2*cutoff            */
  GTBO_ERR_ELL_OVERFLOW = -3   /* a row needs more slots than `width`     */
};

/* Hopping model of Eq. 1 reduced to one orbital per atom:
 *   t_ij = t0[s_i][s_j]                       if beta == 0
 *   t_ij = t0[s_i][s_j]*exp(-beta*(r/r0 - 1)) otherwise
 *   eps_i = onsite[s_i] (+ onsite_shift[i] if onsite_shift != NULL)        */
typedef struct gtbo_model {
  int32_t n_species;
  const double* onsite;       /* [n_species]              eV */
  const double* t0;           /* [n_species][n_species]   eV */
  double r0;
  double beta;
  const double* onsite_shift; /* [n] or NULL              eV */
} gtbo_model;

typedef struct gtbo_ell {
  int64_t n;
  int32_t width;
  int32_t* cols; /* [width][n] */
  double* vals;  /* [width][n] */
  double* diag;  /* [n] or NULL */
} gtbo_ell;

/* --- C2: neighbour sets N(i) = { j != i : r_ij^2 < cutoff^2 } (Eq. 1) ----- */
/* counts[i] = |N(i)|; returns max_i counts[i] in *width_out.
 * method 0 = brute force O(n^2); 1 = cell buckets.                          */
int gtbo_neighbor_counts(const double* pos, int64_t n, const double box[3],
                         const int32_t pbc[3], double cutoff, int32_t method,
                         int32_t* counts /* [n] or NULL */, int32_t* width_out);

/* Fill H (caller-allocated, H->width given).  method as above.             */
int gtbo_build_hamiltonian(const double* pos, const int32_t* species, int64_t n,
                           const double box[3], const int32_t pbc[3],
                           double cutoff, const gtbo_model* model,
                           int32_t method, gtbo_ell* H);

/* --- C7: Gershgorin bounds; lo_hi[0] = E_lo, lo_hi[1] = E_hi --------------- */
int gtbo_spectral_bounds(const gtbo_ell* H, double lo_hi[2]);

/* --- C3: counter-based random phases ------------------------------------- */
uint64_t gtbo_mix64(uint64_t z);                         /* splitmix64 output */
uint64_t gtbo_hash(uint64_t seed, uint32_t r, uint64_t i); /* h(seed, r, i)   */
double gtbo_uniform(uint64_t seed, uint32_t r, uint64_t i); /* (h>>11)*2^-53  */
/* phi[i][k] = exp(i*theta), theta = fl(2*pi*u(seed, r0+k, i)), k = 0..R-1    */
/* rows[q] of the vectors gtbo_random_phase_fill would write: phi [n_rows][R][2]. */
int gtbo_random_phase_rows(uint64_t seed, int32_t r0, int32_t R, const int64_t* rows, int64_t n_rows,
                           double* phi);
int gtbo_random_phase_fill(uint64_t seed, int32_t r0, int32_t R, int64_t n,
                           double* phi);

/* --- C4/C5: Chebyshev moments --------------------------------------------- */
/* mode 0: R random-phase vectors r = 0..R-1 (seed).
 * mode 1: exact trace over all n basis vectors (R, seed ignored).
 * algo 0: direct definition m_n = Re<phi_0|phi_n>, M SpMVs        (C4)
 * algo 1: doubling identities, ceil(M/2) SpMVs                     (C5)
 * mu[n] = sum_r m_n^(r) / (n_atoms * R)  (mode 1: / n_atoms).
 * im_max (optional): max_n |Im sum_r <phi_0|phi_n>| / (n_atoms*R), algo 0.  */
int gtbo_kpm_moments(const gtbo_ell* H, double a, double b, int32_t M,
                     int32_t R, uint64_t seed, int32_t mode, int32_t algo,
                     double* mu, double* im_max);

/* One recursion step on selected rows only (sampled full-size parity):
 *   first != 0 : out[i] = (H phi_cur - b phi_cur)[i] / a
 *   first == 0 : out[i] = (H phi_cur - b phi_cur)[i] * (2/a) - phi_prev[i]
 * phi_* are [n][R][2]; out is [n_rows][R][2].                               */
int gtbo_kpm_step_rows(const gtbo_ell* H, double a, double b, int32_t first,
                       int32_t R, const double* phi_prev, const double* phi_cur,
                       const int64_t* rows, int64_t n_rows, double* out);

/* --- C6: Jackson-damped DOS (Eq. 4) -------------------------- */
/* kernel 0 = none (g_n = 1), 1 = Jackson.  rho = 0 where |(E-b)/a| >= 1 - 8 eps (reading A13b). */
int gtbo_dos(const double* mu, int32_t M, double a, double b, int32_t kernel,
             const double* energies, int32_t G, double scale, double* rho);
/* g[n], n = 0..M-1 (exported so the kernel itself can be pinned).           */
int gtbo_jackson(int32_t M, double* g);

/* --- VAC conductivity (Eq. 3) -- */
/* Units hbar = 1: times in hbar/eV, velocities in eV*Angstrom.  Readings V1-V6
 * are listed at the top of gtbo_vac.cpp and in DESIGN.md sec. 11.
 * V1: vvals[k][i] = vals[k][i]*(x_j - x_i)_axis (minimum image), V = i*vvals. */
int gtbo_velocity_ell(const gtbo_ell* H, const double* pos, const double box[3],
                      const int32_t pbc[3], int32_t axis, double* vvals /*[width][n]*/);
/* y = V x on R interleaved vectors ([n][R][2]). */
int gtbo_velocity_apply(const gtbo_ell* H, const double* vvals, int32_t R,
                        const double* x, double* y);
/* V4: y = exp(-i H dt) x by the Chebyshev-Bessel expansion; *terms = its length. */
int gtbo_evolve(const gtbo_ell* H, double a, double b, double dt, int32_t R,
                const double* x, double* y, int32_t* terms);
/* V2/V3: C[j][n] = (1/(N R)) sum_r Re<U^j phi_r| T_n(H~) V |U^j V phi_r>,
 * j = 0..n_steps-1, n = 0..M-1.  mode 0 random-phase vectors, 1 all basis vectors. */
int gtbo_vac_moments(const gtbo_ell* H, const double* vvals, double a, double b,
                     int32_t M, int32_t n_steps, double dt, int32_t R, uint64_t seed,
                     int32_t mode, double* C /*[n_steps][M]*/);
/* V5/V6: rho_vv[j][g] (optional) = reconstruction of C[j][:] as gtbo_dos;
 * sigma[j][g] = scale * trapezoid integral of rho_vv over tau in [0, j dt]. */
int gtbo_vac_conductivity(const double* C, int32_t M, int32_t n_steps, double a,
                          double b, int32_t kernel, const double* energies, int32_t G,
                          double dt, double scale, double* rho_vv, double* sigma);

/* --- multi-orbital Slater-Koster blocks (NEXT-2) ----- */
/* s,p_x,p_y,p_z on every atom; the table is written out at the top of gtbo_sk.cpp. */
typedef struct gtbo_sk_model {
  int32_t n_species;
  const double* onsite_s;     /* [n_species] eV */
  const double* onsite_p;     /* [n_species] eV */
  const double* sk;           /* [n_species][n_species][4]: ss_sigma, sp_sigma, pp_sigma, pp_pi (eV) */
  double r0;
  double beta;                /* every V scaled by exp(-beta (r/r0 - 1)); 0 -> no scaling */
  const double* onsite_shift; /* [n] or NULL */
} gtbo_sk_model;
/* nbr: any ELL over the n atoms whose cols are the neighbour lists (vals unused).
 * H: caller-allocated scalar ELL over 4n orbitals, width 4*nbr->width, diag [4n] or NULL. */
int gtbo_sk_hamiltonian(const gtbo_ell* nbr, const double* pos, const int32_t* species,
                        const double box[3], const int32_t pbc[3],
                        const gtbo_sk_model* model, gtbo_ell* H);

/* --- environment-dependent hopping from the paper's descriptor + MLPs (Eq. 2; NEXT-3) */
/* One orbital per atom.  Formulas, readings E1-E4 and the weight blob layout: top of gtbo_mlp.cpp. */
typedef struct gtbo_mlp_model {
  int32_t n_species, n_features /*F*/, n_basis /*Nb*/, n_hidden /*Hd*/;
  double r_cut;
  const double* weights;
} gtbo_mlp_model;
/* C[n] = C_n(r) for the species pair (si, sj), n = 0..F-1. */
int gtbo_mlp_descriptor(const gtbo_mlp_model* m, int32_t si, int32_t sj, double r, double* C);
/* H->cols given (neighbour lists); fills H->vals (t_ij; padding 0) and H->diag (eps_i) if non-NULL;
 * v_out ([n][F], optional) receives the node features v_i. */
int gtbo_mlp_hamiltonian(const gtbo_mlp_model* m, const double* pos, const int32_t* species,
                         const double box[3], const int32_t pbc[3], gtbo_ell* H, double* v_out);

/* --- Slater-Koster blocks for the s,p,d basis (9 orbitals; NEXT-2) */
/* Orbital order s, px, py, pz, dxy, dyz, dzx, dx2-y2, dz2; construction: top of gtbo_spd.cpp. */
typedef struct gtbo_spd_model {
  int32_t n_species;
  const double* onsite_s;     /* [n_species] eV */
  const double* onsite_p;
  const double* onsite_d;
  const double* sk;           /* [n_species][n_species][10]: ss_s, sp_s, pp_s, pp_p, sd_s, pd_s, pd_p, dd_s, dd_p, dd_d */
  double r0;
  double beta;
  const double* onsite_shift; /* [n] or NULL */
} gtbo_spd_model;
/* H: caller-allocated scalar ELL over 9n orbitals, width 9*nbr->width, diag [9n] or NULL. */
/* One Chebyshev step of the s,p,d orbital matrix on sampled atoms without materialising H (for sizes
 * whose scalar ELL does not fit the host); vectors given sparsely, see gtbo_spd.cpp. */
int gtbo_spd_step_atoms(const gtbo_ell* nbr, const double* pos, const int32_t* species,
                        const double box[3], const int32_t pbc[3], const gtbo_spd_model* model,
                        double a, double b, int32_t first, int32_t R, const int64_t* atoms,
                        int64_t n_rows, const double* x_own, const double* x_nbr, const double* prev,
                        double* out);
/* bond direction + ten integrals (V for l_a <= l_b, Vt for l_a > l_b) -> E [9][9] row-major */
int gtbo_spd_block_from_integrals(const double u[3], const double* V, const double* Vt, double* E);
/* Eq. 2 feeding the s,p,d blocks: MLP_lambda with ten outputs, onsite MLPs with three (gtbo_mlp.cpp). */
int gtbo_mlp_spd_hamiltonian(const gtbo_mlp_model* m, const gtbo_ell* nbr, const double* pos,
                             const int32_t* species, const double box[3], const int32_t pbc[3],
                             gtbo_ell* H);
int gtbo_spd_hamiltonian(const gtbo_ell* nbr, const double* pos, const int32_t* species,
                         const double box[3], const int32_t pbc[3],
                         const gtbo_spd_model* model, gtbo_ell* H);

/* Eq. 2 feeding the s,p Slater-Koster blocks: MLP_lambda with four outputs (ss_sigma,
 * sp_sigma, pp_sigma, pp_pi of the pair), onsite MLP with two (eps_s, eps_p); blob layout in gtbo_mlp.cpp.
 * H: scalar ELL over 4n orbitals as gtbo_sk_hamiltonian's. */
int gtbo_mlp_sk_hamiltonian(const gtbo_mlp_model* m, const gtbo_ell* nbr, const double* pos,
                            const int32_t* species, const double box[3], const int32_t pbc[3],
                            gtbo_ell* H);

/* Fig. 4b post-processing (readings V7, V8 in gtbo_vac.cpp): n(E_j) = int_{e_ref}^{E_j} rho dE (trapezoid,
 * rho interpolated at e_ref; energies strictly ascending, e_ref inside the grid);
 * mu_j = scale * sigma_j / |n_j| where |n_j| > n_min, else 0. */
int gtbo_carrier_density(const double* rho, const double* energies, int32_t G, double e_ref, double* n_out);
int gtbo_mobility(const double* sigma, const double* n, int32_t G, double scale, double n_min, double* mu);

#ifdef __cplusplus
}
#endif
#endif /* GTBO_H */
