/*
 * gtb.h -- C ABI of libgtb_kpm.so: the B200 (sm_100a) hot path of GPUTB's
 * large-scale stage (arxiv/paper_2509_06525): linear-scaling quantum transport
 * density of states by the Kernel Polynomial Method.
 *
 *   build_hamiltonian(positions, species, box, cutoff, hopping model) -> ELL H
 *   kpm_moments(H, a, b, M, R, seed)                                  -> mu_0..mu_{M-1}
 *   dos(mu, Jackson kernel, energy grid)                              -> rho(E)
 *
 * What each call computes is fixed by PAPER.md:78-81 (Eq. 1, the orthogonal
 * tight-binding Hamiltonian with neighbours inside a cutoff)
 * (sec. 2.4: Chebyshev expansion, KPM, sparse matrix-vector multiplication,
 * random phase approximation), PAPER.md:66 (Eq. 4, rho(E) = (2/Omega) Tr
 * delta(E - H)) and, for everything the paper leaves out, by
 * BASELINE.json:north_star and the readings C1-C7 / A1-A23 listed in DESIGN.md.
 *
 * Conventions
 *  - extern "C", plain pointers and sizes.  Every function returns an int
 *    status (GTB_OK = 0, negatives are errors) unless stated otherwise.
 *  - "device" = pointer into CUDA device memory of the current device, owned by
 *    the caller; "host" = ordinary host memory.  The library allocates nothing
 *    persistent: scratch comes from a caller-provided device workspace whose
 *    minimum size is returned by the matching *_workspace_bytes query.
 *  - `stream` is a cudaStream_t passed as void* (NULL = the legacy default
 *    stream).  Calls marked ASYNC only enqueue work on that stream and return;
 *    calls marked SYNC synchronise that stream before returning.
 *  - Indices are int32 (n <= 2^31-1-64); all byte/element offsets are 64-bit.
 *  - Layouts:
 *      pos      double [n][3]     Cartesian, Angstrom, unwrapped
 *      species  int32  [n]        0 <= s < n_species
 *      ELL      cols int32 [width][n], vals double [width][n]   (slot-major);
 *               row i's entries sorted by ascending column; padding slots have
 *               col = i and val = +0.0; diag double [n] or NULL (= all zero)
 *      phi      double [n][R][2]  complex128, the R vectors interleaved per atom
 *      mu       double [M];  rho, energies  double [G]
 *  - No CPU fallback exists: without a CUDA device every compute call returns
 *    GTB_ERR_CUDA.
 */
#ifndef GTB_H
#define GTB_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
  GTB_OK = 0,
  GTB_ERR_INVALID_ARG = -1,
  GTB_ERR_BOX_TOO_SMALL = -2, /* a periodic box length < 2*cutoff                  */
  GTB_ERR_ELL_OVERFLOW = -3,  /* a row needs more slots than H->width              */
  GTB_ERR_WORKSPACE = -4,     /* workspace NULL, misaligned (256 B) or too small   */
  GTB_ERR_DIVERGED = -5,      /* non-finite moments: spectrum outside [b-a, b+a]   */
  GTB_ERR_CUDA = -6,          /* CUDA runtime error; see gtb_last_cuda_error()     */
  GTB_ERR_INDEX_RANGE = -7,   /* n too large for int32 indices                     */
  GTB_ERR_NOT_PACKABLE = -8,  /* gtb_pack_ell: width > 4, a column offset beyond +-32767 rows or more than
                                 65535 distinct values: stay on the plain ELL path       */
  GTB_ERR_STATIC_LIMIT = -9   /* gtb_kpm_moments_static: the run needs more than GTB_STATIC_WS_BYTES of
                                 scratch; use gtb_kpm_moments with a caller-owned workspace           */
};

#define GTB_MODE_ORB4 16 /* flag for gtb_kpm_moments' mode: H comes from gtb_sk_hamiltonian  (4 orbitals) */
#define GTB_MODE_ORB9 32 /* ... from gtb_spd_hamiltonian (9 orbitals per atom)                           */
#define GTB_MODE_BLOCK9 64  /* ... H holds the 9x9 blocks written by gtb_spd_blocks (H->n = atoms)          */
#define GTB_MODE_PACKED 256 /* ... H holds the packed rows and value dictionary written by gtb_pack_ell     */
#define GTB_MODE_WINDOW 512 /* ... H holds the windowed tiles written by gtb_window_ell (wide rows, K7w)          */
#define GTB_MODE_BOND9 128  /* ... H holds the bond description written by gtb_spd_bonds (matrix-free)      */
#define GTB_MAX_SPECIES 8
#define GTB_MAX_WIDTH 64 /* largest ELL width build_hamiltonian can assemble */

/* Hopping model: Eq. 1 with one p_z orbital per atom
 * (north_star).  t_ij = t0[s_i][s_j] if beta == 0, else
 * t0[s_i][s_j] * exp(-beta * (r_ij/r0 - 1));  eps_i = onsite[s_i] (+ onsite_shift[i]). */
typedef struct gtb_hopping_model {
  int32_t n_species;          /* 1..GTB_MAX_SPECIES                                */
  const double* onsite;       /* HOST   [n_species]             eV                 */
  const double* t0;           /* HOST   [n_species][n_species]  eV, symmetric      */
  double r0;                  /* Angstrom (used only when beta != 0)               */
  double beta;
  const double* onsite_shift; /* DEVICE [n] or NULL             eV                 */
} gtb_hopping_model;

/* ELL matrix, all arrays DEVICE, caller-owned.  cols/vals are 16-byte aligned. */
typedef struct gtb_ell {
  int64_t n;
  int32_t width;  /* K: off-diagonal slots per row */
  int32_t* cols;  /* [width][n] */
  double* vals;   /* [width][n] */
  double* diag;   /* [n] or NULL */
} gtb_ell;

/* Kernel selection and timing hooks of the fused Chebyshev pass, for callers that need to pin a
 * kernel (the parity tests compare every variant with the oracle; bench.py times them).  Passing
 * NULL wherever a `const gtb_kpm_options*` is taken means "all zero": the library picks the kernel
 * from the matrix shape.  The library never reads the environment. */
enum {
  GTB_KERNEL_AUTO = 0,
  GTB_KERNEL_ROW = 1,    /* K7: one 256-bit element per thread per iteration (any width)              */
  GTB_KERNEL_ROW_X2 = 2, /* K7x2: two elements in flight per thread; width <= 4, R in {2,4,8}          */
  GTB_KERNEL_TILE = 3    /* K7t: ELL slots staged by TMA; R in {2,4,8}, n % 4 == 0, 16-byte aligned H  */
};
#define GTB_OPT_PER_PASS_LAUNCH 1 /* never fold a small system's passes into one launch (K7p, K7c)        */
#define GTB_OPT_SCALAR_BLOCKS 2   /* ignore GTB_MODE_ORB4 / ORB9: run the scalar kernels on the expanded H */
#define GTB_OPT_BLOCK_DIRECT 4    /* K7b9: strided block loads instead of the shared-memory hand-off      */
#define GTB_OPT_GRID_SYNC 16      /* tiny systems: K7p (cooperative launch, grid barrier) instead of K7c (one cluster)   */
#define GTB_OPT_SEPARATE_AXPY 8   /* gtb_vac_moments: one accumulation launch per Chebyshev-Bessel term
                                     instead of the accumulation fused into the propagation pass (same bits) */
typedef struct gtb_kpm_options {
  int32_t kernel;       /* GTB_KERNEL_*; a kernel that cannot take (H, R_batch) -> GTB_ERR_INVALID_ARG  */
  int32_t tile_stages;  /* K7t ring depth, 1..8; 0 = default (2)                                       */
  int32_t flags;        /* GTB_OPT_*                                                                   */
  /* Timing hooks: caller-owned cudaEvent_t (as void*) or NULL.  If both are given they are recorded
   * on `stream` around the recursion loop of the LAST batch (first pass excluded; gtb_vac_moments:
   * around the M-1 moment passes of the last time step), and *loop_passes (HOST, may be NULL)
   * receives the number of fused passes between them.  The library keeps no timing state. */
  void* loop_begin;
  void* loop_end;
  int32_t* loop_passes;
  /* gtb_vac_moments only: a compressed form of the SAME matrix (from gtb_pack_ell or gtb_window_ell built for
   * R_batch) on which the moment passes (packed rows: and the propagation passes) run; the velocity operator
   * keeps reading H.  NULL: none.
   * alt_mode = GTB_MODE_PACKED or GTB_MODE_WINDOW. */
  const struct gtb_ell* alt;
  int32_t alt_mode;
} gtb_kpm_options;

/* ---- status -------------------------------------------------------------- */
const char* gtb_status_string(int status);
const char* gtb_last_cuda_error(void); /* text of the last CUDA error seen by this thread */
int gtb_version(void);                 /* 10000*major + 100*minor + patch */
/* number of kernel launches this library has enqueued since load (monotonic). */
int64_t gtb_launch_count(void);

/* ---- Hamiltonian assembly (Eq. 1; north_star (1); readings C2, A14, A15) -- */
/* Neighbour set: N(i) = { j != i : r2 < cutoff*cutoff }, with
 *   d_a = x_j[a]-x_i[a];  periodic a: d_a -= L_a*rint(d_a/L_a);
 *   r2 = (d_x*d_x + d_y*d_y) + d_z*d_z     (fp64, no FMA contraction, strict <).
 * Requires L_a >= 2*cutoff on every periodic axis (GTB_ERR_BOX_TOO_SMALL). */
size_t gtb_build_workspace_bytes(int64_t n);

/* SYNC.  *width_out (HOST) = max_i |N(i)|;  counts (DEVICE [n] or NULL) = |N(i)|. */
int gtb_neighbor_width(const double* pos /*device*/, int64_t n, const double box[3] /*host*/,
                       const int32_t pbc[3] /*host*/, double cutoff, int32_t* counts,
                       void* ws, size_t ws_bytes, void* stream, int32_t* width_out);

/* SYNC.  Fills H->cols, H->vals (and H->diag if non-NULL) in the layout above;
 * H->n must equal n and H->width is the caller's allocation.  If some row needs
 * more than H->width slots, returns GTB_ERR_ELL_OVERFLOW, stores the required
 * width in *width_needed (HOST, may be NULL) and leaves H unspecified. */
int gtb_build_hamiltonian(const double* pos /*device*/, const int32_t* species /*device*/,
                          int64_t n, const double box[3], const int32_t pbc[3], double cutoff,
                          const gtb_hopping_model* model, gtb_ell* H, void* ws, size_t ws_bytes,
                          void* stream, int32_t* width_needed);

/* ASYNC.  Gershgorin bounds (reading C7): lo_hi[0] = min_i(diag_i - sum_k|vals[k][i]|),
 * lo_hi[1] = max_i(diag_i + sum_k|vals[k][i]|).  lo_hi is DEVICE [2].
 * Workspace: gtb_bounds_workspace_bytes(n). */
size_t gtb_bounds_workspace_bytes(int64_t n);
int gtb_spectral_bounds(const gtb_ell* H, double* lo_hi, void* ws, size_t ws_bytes, void* stream);

/* ---- random-phase vectors (north_star (2); reading C3) --- */
/* ASYNC.  phi[i][k] = exp(i*theta), theta = fl(6.283185307179586 * u),
 * u = (h >> 11) * 2^-53,  h = mix(mix(seed + (r0+k+1)*g) + (i+1)*g),
 * g = 0x9E3779B97F4A7C15, mix = the splitmix64 output function; k = 0..R-1. */
int gtb_random_phase_fill(uint64_t seed, int32_t r0, int32_t R, int64_t n, double* phi /*device*/,
                          void* stream);

/* ---- Chebyshev moments (north_star (3); readings C4, C5, A17) - */
/* Recursion |phi_{n+1}> = 2 H~ |phi_n> - |phi_{n-1}>, H~ = (H - b)/a, run for
 * ceil(M/2) fused passes; moments by the doubling identities
 *   m_{2n} = 2<phi_n|phi_n> - m_0,  m_{2n+1} = 2 Re<phi_{n+1}|phi_n> - m_1,
 * mu_n = sum_r m_n^(r) / (n * R_total)           (mode 1: / n).
 * mode 0: R_total random-phase vectors r = 0..R_total-1 of `seed`, processed
 *         R_batch at a time (each pass of H serves R_batch vectors).
 * mode 1: exact trace over all n basis vectors e_i (R_total and seed ignored),
 *         R_batch of them per pass.
 * mode | GTB_MODE_BLOCK9 / GTB_MODE_BOND9: H is the block / bond form of an s,p,d Hamiltonian (see
 *         gtb_spd_bonds below); H->n counts atoms, the vectors have 9 H->n rows.
 * mode | GTB_MODE_ORB4 (or GTB_MODE_ORB9): the caller promises that H is the orbital-blocked matrix
 *         written by gtb_sk_hamiltonian (4 orbitals per atom; gtb_spd_hamiltonian: 9); the fused pass
 *         then works on whole 4x4 (9x9) blocks (one gather of the neighbour's orbitals per block).  Same results; ignored
 *         when R_batch is not 2, 4 or 8.  A matrix without that structure gives wrong results.
 * R_batch: 1..64.  R_batch in {2,4,8} takes the 256-bit vector path.
 * ASYNC.  mu is DEVICE [M].  Workspace: gtb_kpm_workspace_bytes(n, M, R_batch). */
size_t gtb_kpm_workspace_bytes(int64_t n, int32_t M, int32_t R_batch);
int gtb_kpm_moments(const gtb_ell* H, double a, double b, int32_t M, int32_t R_total,
                    int32_t R_batch, uint64_t seed, int32_t mode, double* mu, void* ws,
                    size_t ws_bytes, void* stream, const gtb_kpm_options* opt);

/* SYNC.  GTB_ERR_DIVERGED if the last gtb_kpm_moments run on this workspace
 * produced a non-finite moment, else GTB_OK. */
int gtb_kpm_status(const void* ws, void* stream);

/* ---- the same moments with NO allocation and no caller workspace ------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid it).  gtb_kpm_moments_static is gtb_kpm_moments (north_star (3); same arguments,
 * same kernels, same results bit for bit) with the workspace taken from a static device array inside the
 * library instead of from the caller: GTB_STATIC_WS_BYTES (4 MiB) on every GPU that loads the library, held
 * until the process exits.  The caller still owns and passes H and mu (DEVICE [M]).
 * Limit: gtb_kpm_workspace_bytes(rows, M, R_batch) <= GTB_STATIC_WS_BYTES, rows = H->n (9 H->n in the
 * BLOCK9 / BOND9 modes); e.g. config 1 (2304 atoms, M = 256, R = 4) needs 2.7 MiB.  Anything larger returns
 * GTB_ERR_STATIC_LIMIT before a kernel is launched.
 * The call uses no cudaMalloc / cudaFree or other allocating routine (once per device it asks the runtime for
 * the array's device address).  ASYNC on the caller's stream.
 * Sharing: every call on a device uses the SAME array, which keeps the previous call's contents.  What must
 * start at zero is cleared on the stream at the start of each call; calls that may overlap on the GPU (two
 * streams, two host threads) race on it -- order them.  There is no status word to read afterwards: a
 * diverged run (spectrum outside [b - a, b + a]) shows as non-finite mu. */
#define GTB_STATIC_WS_BYTES (4 << 20)
int gtb_kpm_moments_static(const gtb_ell* H, double a, double b, int32_t M, int32_t R_total,
                           int32_t R_batch, uint64_t seed, int32_t mode, double* mu, void* stream,
                           const gtb_kpm_options* opt);

/* ASYNC.  One fused recursion pass, exported for the full-size sampled parity test:
 *   first != 0:  out = (H phi_cur - b phi_cur) / a                 (phi_io is written only)
 *   first == 0:  out = (H phi_cur - b phi_cur)*(2/a) - phi_io      (phi_io read, then overwritten)
 * sums (DEVICE [2]) = { sum_{i,r} |phi_cur|^2 ,  sum_{i,r} Re(conj(out) phi_cur) }.
 * phi_cur, phi_io: DEVICE [n][R][2], 32-byte aligned, must not overlap.
 * mode: 0, or one of GTB_MODE_ORB4 / ORB9 / BLOCK9 / BOND9 with the meaning they have in gtb_kpm_moments
 * (BLOCK9 / BOND9: n = 9 H->n vector rows).
 * Workspace: gtb_kpm_workspace_bytes(n, 2, R). */
int gtb_kpm_step(const gtb_ell* H, double a, double b, int32_t first, int32_t R,
                 const double* phi_cur, double* phi_io, double* sums, int32_t mode, void* ws,
                 size_t ws_bytes, void* stream, const gtb_kpm_options* opt);

/* ---- density of states (Eq. 4; north_star (4); reading C6) ---- */
/* ASYNC.  rho(E_j) = scale*[g_0 mu_0 + 2 sum_{n=1}^{M-1} g_n mu_n T_n(x_j)] / (pi a sqrt(1-x_j^2)),
 * x_j = (E_j - b)/a, and rho = 0 where |x_j| >= 1 - 8 eps, eps = 2^-52 (the end points b +- a of a grid, up
 * to the rounding of x_j: reading A13b).
 * kernel 0: g_n = 1;  kernel 1 (Jackson):
 *   g_n = [(M-n+1) cos(pi n/(M+1)) + sin(pi n/(M+1)) cot(pi/(M+1))]/(M+1).
 * mu, energies, rho: DEVICE. */
int gtb_dos(const double* mu, int32_t M, double a, double b, int32_t kernel,
            const double* energies, int32_t G, double scale, double* rho, void* stream);
/* ASYNC.  g (DEVICE [M]) = Jackson coefficients as above. */
int gtb_jackson(int32_t M, double* g, void* stream);

/* ---- VAC conductivity (Eq. 3; time step and step count :60, :68) ----
 * sigma(E, t) = (2 e^2/Omega) int_0^t Tr[delta(E - H) Re(V V(tau))] dtau,  V(tau) = e^{iH tau} V e^{-iH tau}.
 * The paper prints no formula for V, the propagator or the estimator; readings V1-V6 of
 * DESIGN.md sec. 11.  Units hbar = 1: times in hbar/eV (0.1 fs = 0.1/0.6582119569), velocities
 * in eV*Angstrom; the prefactor 2 e^2/(Omega hbar^2) N is the caller's `scale`. */

/* ASYNC.  V1: V = i [H, X_axis]  =>  V_ij = i * vvals_ij,
 *   vvals[k][i] = vals[k][i] * d,  d = x_j - x_i (axis component), j = cols[k][i];
 *   periodic axis: d -= L*rint(d/L)   (fp64, no FMA contraction).
 * pos DEVICE [n][3]; box, pbc HOST; vvals DEVICE [width][n] (same layout as H->vals). */
int gtb_velocity_ell(const gtb_ell* H, const double* pos, const double box[3],
                     const int32_t pbc[3], int32_t axis, double* vvals, void* stream);

/* ASYNC.  y = V x = i * (vvals x) on R interleaved vectors; x, y DEVICE [n][R][2], x != y. */
int gtb_velocity_apply(const gtb_ell* H, const double* vvals, int32_t R, const double* x,
                       double* y, void* stream);

/* ASYNC.  V4: phi <- exp(-i H dt) phi by the Chebyshev-Bessel expansion
 *   e^{-i b dt} sum_m (2 - delta_m0) (-i)^m J_m(a dt) T_m(H~),  H~ = (H - b)/a,
 * truncated after the first m > a*dt with |J_m(a dt)| < 1e-18 (*terms, HOST, may be NULL,
 * receives the number of terms).  phi DEVICE [n][R][2], 32-byte aligned, updated in place.
 * Workspace: gtb_evolve_workspace_bytes(n, R). */
size_t gtb_evolve_workspace_bytes(int64_t n, int32_t R);
int gtb_evolve(const gtb_ell* H, double a, double b, double dt, int32_t R, double* phi,
               int32_t* terms, void* ws, size_t ws_bytes, void* stream);

/* ASYNC.  V2/V3: VAC Chebyshev moments on the time grid tau_j = j*dt, j = 0..n_steps-1:
 *   C[j][n] = (1/(N R_total)) sum_r Re < psiL_r(tau_j) | T_n(H~) V | psiR_r(tau_j) >,  n = 0..M-1,
 *   psiL_r(tau) = U(tau) phi_r,  psiR_r(tau) = U(tau) V phi_r,  U(tau_j) = U(dt)^j,
 * by chi_0 = V psiR, chi_1 = H~ chi_0, chi_{n+1} = 2 H~ chi_n - chi_{n-1}, C_n = Re<psiL|chi_n>:
 * M-1 fused passes per time step (the DOS kernel with the dot products taken against psiL).
 * mode (incl. the GTB_MODE_ORB4 flag), R_total, R_batch, seed: as gtb_kpm_moments (mode 1: / N).
 * C is DEVICE [n_steps][M].
 * Workspace: gtb_vac_workspace_bytes(n, M, n_steps, R_batch); gtb_kpm_status(ws) reports
 * non-finite results as GTB_ERR_DIVERGED. */
size_t gtb_vac_workspace_bytes(int64_t n, int32_t M, int32_t n_steps, int32_t R_batch);
int gtb_vac_moments(const gtb_ell* H, const double* vvals, double a, double b, int32_t M,
                    int32_t n_steps, double dt, int32_t R_total, int32_t R_batch, uint64_t seed,
                    int32_t mode, double* C, void* ws, size_t ws_bytes, void* stream,
                    const gtb_kpm_options* opt);

/* ASYNC.  V5/V6: rho_vv[j][g] = kernel-damped reconstruction of C[j][:] at E_g exactly as
 * gtb_dos (scale 1); sigma[0][g] = 0, sigma[j][g] = sigma[j-1][g] + scale*dt*(rho_vv[j-1][g] +
 * rho_vv[j][g])/2 (trapezoid rule).  C, energies, rho_vv, sigma: DEVICE; rho_vv and sigma
 * are [n_steps][G], both written. */
int gtb_vac_conductivity(const double* C, int32_t M, int32_t n_steps, double a, double b,
                         int32_t kernel, const double* energies, int32_t G, double dt,
                         double scale, double* rho_vv, double* sigma, void* stream);

/* ---- multi-orbital Slater-Koster blocks (reading S1) ----
 * The paper's H consists of onsite blocks H_ii and hopping blocks H_ij^{lm,l'm'} from Slater-Koster
 * parameters and the bond direction.  This call assembles the s, p_x, p_y, p_z case: with
 * (l, m, n) = (x_j - x_i)/r (minimum image) and every V scaled by exp(-beta (r/r0 - 1)),
 *   E_ss = V_ss_sigma;  E_{s,pa} = a V_sp_sigma;  E_{pa,s} = -a V_sp_sigma;
 *   E_{pa,pb} = a b V_pp_sigma + (delta_ab - a b) V_pp_pi;   onsite eps_s, eps_p (+ onsite_shift[i]).
 * The result is a scalar ELL matrix over the 4n orbitals (orbital index 4 i + mu, mu = s, x, y, z) in
 * the layout of this header: row (i, mu), slot 4 k + nu holds column 4 j + nu and E_{mu nu}, j = the
 * k-th neighbour of atom i; padding slots (j = i) hold the row's own index and +0.  It is accepted
 * by gtb_kpm_moments, gtb_velocity_ell (with positions repeated per orbital) and the rest unchanged. */
typedef struct gtb_sk_model {
  int32_t n_species;          /* 1..GTB_MAX_SPECIES                                          */
  const double* onsite_s;     /* HOST [n_species] eV                                         */
  const double* onsite_p;     /* HOST [n_species] eV                                         */
  const double* sk;           /* HOST [n_species][n_species][4]: ss_sigma, sp_sigma, pp_sigma, pp_pi */
  double r0;
  double beta;
  const double* onsite_shift; /* DEVICE [n] or NULL                                          */
} gtb_sk_model;

/* ASYNC.  nbr: any ELL matrix over the n atoms whose cols are the neighbour lists (vals unused),
 * e.g. the output of gtb_build_hamiltonian.  H: caller-allocated, H->n = 4 n, H->width =
 * 4 nbr->width, H->diag [4 n] or NULL.  pos, species: DEVICE.  *status (DEVICE int32) is set
 * non-zero if a species index is out of range. */
int gtb_sk_hamiltonian(const gtb_ell* nbr, const double* pos, const int32_t* species,
                       const double box[3], const int32_t pbc[3], const gtb_sk_model* model,
                       gtb_ell* H, int32_t* status, void* stream);

/* ---- environment-dependent Hamiltonian from the descriptor + MLPs of Eq. 2 ----
 * One orbital per atom.  With f_c(r) = 1/2 [1 + cos(pi r/r_cut)] (reading E1; the paper's "smooth
 * cutoff function" is not printed), x = 2 (r/r_cut - 1)^2 - 1:
 *   f_k(r) = 1/2 [T_k(x) + 1] f_c(r), k = 0..Nb-1;   C_n(r_ij) = sum_k c[s_i][s_j][n][k] f_k(r_ij), n = 0..F-1;
 *   v_i = sum_{j in N(i)} C(r_ij);   e_ij = C(r_ij) * MLP_e(v_i + v_j)  (element-wise);
 *   t_ij = MLP_lambda(e_ij);   eps_i = MLP_{s_i}(v_i);   MLP(x) = W2 silu(W1 x + b1) + b2.
 * weights: DEVICE blob of gtb_mlp_weight_count() doubles, laid out as
 *   c [ns][ns][F][Nb] | MLP_e: W1 [Hd][F], b1 [Hd], W2 [F][Hd], b2 [F] |
 *   MLP_lambda: W1 [Hd][F], b1 [Hd], W2 [Hd], b2 [1] | per species s: W1 [Hd][F], b1 [Hd], W2 [Hd], b2 [1].
 * Instantiated sizes (F, Nb, Hd): (8, 8, 16), (4, 4, 8), (16, 8, 32); others -> GTB_ERR_INVALID_ARG. */
typedef struct gtb_mlp_model {
  int32_t n_species, n_features, n_basis, n_hidden;
  double r_cut;
  const double* weights; /* DEVICE */
} gtb_mlp_model;
size_t gtb_mlp_weight_count(int32_t n_species, int32_t n_features, int32_t n_basis, int32_t n_hidden);
/* ASYNC.  H->cols must hold the neighbour lists (e.g. from gtb_build_hamiltonian with the same
 * cutoff <= r_cut); H->vals and, if non-NULL, H->diag are overwritten (padding slots: 0).
 * v: DEVICE [n][F], receives the node features.  *status (DEVICE) non-zero: species out of range. */
int gtb_mlp_hamiltonian(const gtb_mlp_model* m, const double* pos, const int32_t* species,
                        const double box[3], const int32_t pbc[3], gtb_ell* H, double* v,
                        int32_t* status, void* stream);

/* ---- Slater-Koster blocks for the s, p, d basis of the paper's runs (reading S4) ----
 * 9 orbitals per atom in the order s, px, py, pz, dxy, dyz, dzx, dx2-y2, dz2.  Two-centre integrals are
 * diagonal in the bond frame (e1, e2, u), u = (x_j - x_i)/r; with c_{a,m} the coefficient of lab orbital a on
 * the frame orbital m (sigma, pi1, pi2, delta1, delta2):
 *   E_ab = sum_m c_{a,m} V_{l_a l_b |m|} c_{b,m},  times (-1)^{l_a + l_b} when l_a > l_b,
 * V = { ss_sigma, sp_sigma, pp_sigma, pp_pi, sd_sigma, pd_sigma, pd_pi, dd_sigma, dd_pi, dd_delta } per
 * species pair, each times exp(-beta (r/r0 - 1)); onsite eps_s, eps_p, eps_d (+ onsite_shift[i]).
 * Output: scalar ELL over the 9n orbitals, laid out as gtb_sk_hamiltonian's with 9 in place of 4. */
typedef struct gtb_spd_model {
  int32_t n_species;
  const double* onsite_s;     /* HOST [n_species] eV */
  const double* onsite_p;
  const double* onsite_d;
  const double* sk;           /* HOST [n_species][n_species][10] eV */
  double r0;
  double beta;
  const double* onsite_shift; /* DEVICE [n] or NULL */
} gtb_spd_model;
size_t gtb_spd_workspace_bytes(void);
/* SYNC on the parameter upload, then ASYNC.  H->n = 9 n, H->width = 9 nbr->width, H->diag [9 n] or NULL.
 * Workspace: gtb_spd_workspace_bytes() (holds the parameter block while the kernels run). */
int gtb_spd_hamiltonian(const gtb_ell* nbr, const double* pos, const int32_t* species,
                        const double box[3], const int32_t pbc[3], const gtb_spd_model* model,
                        gtb_ell* H, int32_t* status, void* ws, size_t ws_bytes, void* stream);

/* ---- s,p,d at the paper's scale: block and bond representations (Fig. 4a :192) ----
 * The scalar ELL of gtb_spd_hamiltonian costs 972 K bytes per atom (81 K column copies + 81 K values) and
 * stops near 10^7 atoms.  Two other representations of the SAME operator, each with its own fused pass:
 *
 * bonds (GTB_MODE_BOND9, matrix-free): the pass rebuilds every pair's 9x9 action from the bond vector and
 *   the species pair's ten integrals in registers (closed form of reading S4 summed over the bond frame:
 *   csrc/spd9.cu).  H costs 4 K + 40 bytes per atom: 10^8 atoms x 9 orbitals with a
 *   third-neighbour cutoff fit one 180 GB B200.
 *     Hm->n = atoms, Hm->width = K and Hm->cols = the neighbour lists of `nbr` (shared, not copied),
 *     Hm->vals = a caller-allocated DEVICE block of gtb_spd_bonds_bytes(n) bytes (256-byte aligned) that
 *     receives the parameter tables and one record (x, y, z, species) + onsite shift per atom;
 *     Hm->diag is ignored (the onsite energies of the model are always applied).
 *   The model's same-l integrals (ss, pp, dd) must be symmetric in the species pair (GTB_ERR_INVALID_ARG
 *   otherwise: no symmetric H exists); the mixed-l ones (sp, sd, pd) may differ between (A, B) and (B, A).
 *   SYNC on the parameter upload, then ASYNC.  *status (DEVICE int32) non-zero: species out of range.
 *
 * blocks (GTB_MODE_BLOCK9): the pairs' blocks stored once, every load coalesced:
 *     Hb->n = atoms, Hb->width = K, Hb->cols = Hm->cols (shared), Hb->vals = double [K][81][n]
 *     (entry 9 nu + mu of block k of atom i at ((k*81 + 9 nu + mu) * n + i); padding slots: zeros),
 *     Hb->diag = double [9][n] (onsite energy of orbital mu of atom i at mu*n + i) or NULL.
 *   gtb_spd_blocks fills them from the bond form.  ASYNC.  652 K + 72 bytes per atom.
 *
 * Both go to gtb_kpm_moments(H, ..., mode | GTB_MODE_BLOCK9 / GTB_MODE_BOND9, ...) with R_batch in
 * {2, 4, 8}; the vectors have 9 n rows (orbital 9 i + mu, as in the scalar form), so the workspace is
 * gtb_kpm_workspace_bytes(9 n, M, R_batch) and the moments are normalised by 9 n R.  Same moments as the
 * scalar form up to rounding (another summation order inside a block).
 * gtb_spd_bounds: ASYNC, the Gershgorin interval of the orbital matrix from either form (lo_hi DEVICE [2];
 * mode = GTB_MODE_BLOCK9 or GTB_MODE_BOND9; workspace gtb_spd_bounds_workspace_bytes()). */
size_t gtb_spd_bonds_bytes(int64_t n_atoms);
int gtb_spd_bonds(const gtb_ell* nbr, const double* pos, const int32_t* species, const double box[3],
                  const int32_t pbc[3], const gtb_spd_model* model, gtb_ell* Hm, int32_t* status,
                  void* stream);
int gtb_spd_blocks(const gtb_ell* Hm, gtb_ell* Hb, void* stream);
size_t gtb_spd_bounds_workspace_bytes(void);
int gtb_spd_bounds(const gtb_ell* H, int32_t mode, double* lo_hi, void* ws, size_t ws_bytes, void* stream);

/* ---- compressed Hamiltonian stream for narrow rows ----
 * For K <= 4 a row is packed into one 16-byte word: per slot a 16-bit column offset relative to the row
 * (ring distance) and a 16-bit index into a dictionary of the distinct fp64 hopping values (lossless);
 * with K <= 3 the fourth slot carries the dictionary index of the onsite energy.  H then costs 16 bytes per
 * atom and pass instead of 12 K + 8 [diag]: config 5 132 -> 112, config 4 428 -> 400 bytes per atom.
 * SHORT rows: with K <= 3 and at most 16 distinct values (hoppings and onsite energies together) a row is ONE
 * 8-byte word, three 16-bit offsets and four 4-bit dictionary indices: config 5 132 -> 104 bytes per atom.
 * gtb_pack_ell picks the format; on return P->width = K | 0x100 for short rows (the pass reads the flag).
 *   P->n = H->n, P->width = H->width, P->cols = caller-allocated DEVICE block of gtb_packed_rows_bytes(n)
 *   bytes (16-byte aligned) receiving the packed rows, P->vals = caller-allocated DEVICE block of
 *   gtb_packed_dict_bytes() bytes receiving a 256-byte header and the dictionary; on return P->diag = NULL,
 *   or H->diag when K = 4 (the diagonal array is then still read).
 * SYNC.  GTB_ERR_NOT_PACKABLE when the matrix does not fit the format (any beta != 0 model: every hopping
 * distinct); *n_values (HOST, may be NULL) receives the dictionary size.
 * gtb_kpm_moments / gtb_kpm_step(P, ..., mode | GTB_MODE_PACKED) run K7x2p, the two-elements-in-flight
 * pass reading this word: R_batch in {2, 4, 8}; same values in the same order, so bit-identical vectors. */
size_t gtb_pack_workspace_bytes(void);
size_t gtb_packed_rows_bytes(int64_t n);
size_t gtb_packed_dict_bytes(void);
int gtb_pack_ell(const gtb_ell* H, gtb_ell* P, void* ws, size_t ws_bytes, void* stream, int32_t* n_values);

/* ---- windowed tiles for wide rows (K7w; sliced ELL + 16-bit relative columns) ----
 * A re-arrangement of an ELL matrix for R_batch = R vectors, tile by tile (256 / (R/2) rows; R = 8: 32 rows): the distinct
 * 1 KB blocks of phi rows the tile's columns touch (its window, at most 40), every column as a 16-bit index
 * into that window, the tile's own slot count (longest row of the tile), and its hoppings / diagonal /
 * columns contiguous.  The pass (gtb_kpm_moments / gtb_kpm_step with mode | GTB_MODE_WINDOW, R_batch = R,
 * R_total a multiple of R) copies window and tile into shared memory with bulk copies and gathers from there.
 * At R = 4 the slots of row pairs are stored in another order than the ELL's (so that the two rows' window indices
 * differ in parity position by position: no shared-memory bank conflicts between them); the sums over a row then run
 * in that order and the vectors equal the plain pass's to rounding, not bit for bit.  R = 2 and R = 8 keep the order.
 *   Wd->n = H->n, Wd->width = H->width, Wd->vals = caller-allocated DEVICE block of
 *   gtb_window_bytes(n, width, R, H->diag != NULL) bytes (128-byte aligned); on return Wd->cols = H->cols
 *   (unused), Wd->diag = H->diag (only its presence matters: the values are in the tiles) and Wd->width =
 *   K | (blocks of the largest window) << 16 | R << 24: the window sizes the shared-memory stage of the pass,
 *   and a pass asked for another R_batch than the tiles were built for is GTB_ERR_INVALID_ARG.
 * SYNC.  scratch: DEVICE int32.  GTB_ERR_NOT_PACKABLE when some tile's neighbours need more than 40 blocks
 * (*blocks_needed, HOST, may be NULL, receives the largest count): the numbering has no locality to use. */
size_t gtb_window_bytes(int64_t n, int32_t width, int32_t R, int32_t with_diag);
int gtb_window_ell(const gtb_ell* H, int32_t R, gtb_ell* Wd, int32_t* scratch, void* stream,
                   int32_t* blocks_needed);

/* ---- the same matrix with its slots in an order the gathers like (north_star (1): the ELL layout leaves the
 * order of a row's slots free) ----
 * ASYNC.  Hp (caller-allocated cols / vals of H's shape, distinct from H's; Hp->diag is set to H->diag) receives
 * the same rows with their entries in another slot order: at R = 4 vectors per pass (a gathered neighbour is half
 * an L1 line) the slots of rows 2q and 2q + 1 are arranged so that, position by position, one column is even and
 * the other odd, and the two gathers share one L1 wavefront; at R = 2 (a quarter of a line) the slots
 * of rows 4q .. 4q + 3 are permuted so that the four columns differ in their two low bits (width <= 4: every
 * permutation tried; up to 48: position by position).  Padding slots stay
 * (column = the row, value 0).  Any other R, or a wider matrix (48 at R = 4): a plain copy.  Hp is an ordinary gtb_ell for every call of this header; sums over
 * a row run in the new order, so results equal those on H to rounding, not bit for bit. */
int gtb_pair_slots(const gtb_ell* H, int32_t R, gtb_ell* Hp, void* stream);

/* ---- Eq. 2 feeding the s,p Slater-Koster blocks: the paper's hopping formula ----
 *   H_ij^{lm,l'm'} = sum_lambda MLP_lambda(e_ij) P_lambda^{lm,l'm'}(r^_ij),   H_ii^{lm,lm} = MLP_{l,alpha}(v_i):
 * MLP_lambda has four outputs, the bond integrals ss_sigma, sp_sigma, pp_sigma, pp_pi of the pair (reading E6),
 * which enter the two-centre table of gtb_sk_hamiltonian; the onsite MLPs have two (eps_s, eps_p).
 * Weight blob as gtb_mlp_hamiltonian's with MLP_lambda: ..., W2 [4][Hd], b2 [4] and per species
 * ..., W2 [2][Hd], b2 [2]: gtb_mlp_sk_weight_count() doubles.  (F, Nb, Hd) = (8, 8, 16) only.
 * ASYNC.  nbr: neighbour lists over the n atoms; H: scalar ELL over 4n orbitals (H->n = 4 n,
 * H->width = 4 nbr->width, diag [4 n] or NULL), usable with GTB_MODE_ORB4; v: DEVICE [n][F]. */
size_t gtb_mlp_sk_weight_count(int32_t n_species, int32_t n_features, int32_t n_basis, int32_t n_hidden);
int gtb_mlp_sk_hamiltonian(const gtb_mlp_model* m, const gtb_ell* nbr, const double* pos,
                           const int32_t* species, const double box[3], const int32_t pbc[3],
                           gtb_ell* H, double* v, int32_t* status, void* stream);

/* ---- Eq. 2 feeding the s,p,d blocks: the paper's model (reading E7) ----
 * MLP_lambda has TEN outputs, the two-centre integrals ss_sigma .. dd_delta of the pair, which enter the block
 * construction of gtb_spd_blocks; the onsite MLPs have three (eps_s, eps_p, eps_d).  e_ij = e_ji, so the same
 * integrals serve both orderings of a pair.  Weight blob as gtb_mlp_sk_hamiltonian's with 10 / 3 in place of
 * 4 / 2: gtb_mlp_spd_weight_count() doubles.  (F, Nb, Hd) = (8, 8, 16) only.
 * ASYNC.  Output in the BLOCK form (GTB_MODE_BLOCK9): Hb->n = atoms, Hb->width = K, Hb->cols = nbr->cols (shared),
 * Hb->vals = double [K][81][n], Hb->diag = double [9][n] or NULL; v: DEVICE [n][F]. */
size_t gtb_mlp_spd_weight_count(int32_t n_species, int32_t n_features, int32_t n_basis, int32_t n_hidden);
int gtb_mlp_spd_blocks(const gtb_mlp_model* m, const gtb_ell* nbr, const double* pos, const int32_t* species,
                       const double box[3], const int32_t pbc[3], gtb_ell* Hb, double* v, int32_t* status,
                       void* stream);

/* ---- 1-D strip decomposition with one halo exchange per pass, on one device ----
 * The rows are cut into n_strips contiguous strips (multiples of 4 rows, the last takes the rest); a strip owns
 * its rows of the vectors plus a lo and a hi halo of `halo` rows each -- the rows of its ring neighbours that its
 * columns reach -- and runs the fused pass on its own column-localised copy of H.  Per pass: one contiguous
 * copy per strip and side from the neighbour's owned rows (the exchange step; a peer copy on several GPUs),
 * then the pass on every strip; block sums are reduced strip after strip in a fixed order.  Same vectors bit
 * for bit as gtb_kpm_moments, moments equal up to the order of the block sums.  Unmeasured on more than one GPU.
 * gtb_strip_plan: HOST only; out = { row0, rows, lo_first, hi_first, lo_owner, hi_owner } of strip p (lo_first /
 * hi_first: global index of the first halo row on the ring); GTB_ERR_INVALID_ARG when a strip is narrower than
 * the halo.  gtb_ring_halo: SYNC, *halo = largest ring distance min(|col - row|, n - |col - row|) in H.
 * gtb_kpm_moments_strips: ASYNC; mode 0 / 1 as gtb_kpm_moments; phi_out (DEVICE [n][R_batch][2] or NULL)
 * receives the last Chebyshev vector of the last batch gathered from the strips. */
int gtb_strip_plan(int64_t n, int32_t n_strips, int64_t halo, int32_t p, int64_t out[6]);
int gtb_ring_halo(const gtb_ell* H, int32_t* scratch, void* stream, int64_t* halo);
size_t gtb_strips_workspace_bytes(int64_t n, int32_t width, int32_t with_diag, int32_t n_strips, int64_t halo,
                                  int32_t M, int32_t R_batch);
int gtb_kpm_moments_strips(const gtb_ell* H, int32_t n_strips, int64_t halo, double a, double b, int32_t M,
                           int32_t R_total, int32_t R_batch, uint64_t seed, int32_t mode, double* mu,
                           double* phi_out, void* ws, size_t ws_bytes, void* stream, const gtb_kpm_options* opt);

/* ---- Fig. 4b post-processing: carrier density and mobility (readings V7, V8) ----
 * ASYNC.  n_out[j] = int_{e_ref}^{E_j} rho(E) dE by the trapezoid rule on the grid (rho interpolated
 * linearly at e_ref; negative below it).  energies strictly ascending, e_ref inside the grid, G >= 2;
 * otherwise *status (DEVICE int32) is set non-zero.  rho, energies, n_out: DEVICE [G]. */
int gtb_carrier_density(const double* rho, const double* energies, int32_t G, double e_ref,
                        double* n_out, int32_t* status, void* stream);
/* ASYNC.  mu[j] = scale * sigma[j] / |n[j]| where |n[j]| > n_min, else 0 (e and units in `scale`). */
int gtb_mobility(const double* sigma, const double* n, int32_t G, double scale, double n_min,
                 double* mu, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* GTB_H */
