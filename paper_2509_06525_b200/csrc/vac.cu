// Velocity-autocorrelation (VAC) conductivity on the device: Eq. 3 of the paper,
//     sigma(E, t) = (2 e^2 / Omega) int_0^t Tr[ delta(E - H) Re( V V(tau) ) ] dtau,
// time step 0.1 fs and > 200 propagation steps.  The paper prints no formula for
// V, the propagator or the estimator; the readings V1-V6 of DESIGN.md sec. 11 are used (hbar = 1):
//   V = i [H, X];   C_n(tau) = (1/(N R)) sum_r Re < U phi_r | T_n(H~) V | U V phi_r >,  U = e^{-i H tau};
//   U(dt) by the Chebyshev-Bessel expansion; kernel-damped reconstruction as for the DOS; trapezoid
//   rule in time.
// The hot loop is the same fused Chebyshev pass as the DOS path (K7/K7t in kpm.cu) with the two dot
// products taken against the evolved bra U phi instead of the vector itself: M - 1 passes per time
// step, one HBM pass each.  Everything else here runs once per time step or once per batch.
#include <cmath>
#include <math.h>

#include <algorithm>
#include <vector>

#include "cheb.cuh"

namespace gtb {
namespace {

// V1: vvals[k][i] = vals[k][i] * (x_j - x_i), minimum image on a periodic axis (no FMA contraction)
__global__ void __launch_bounds__(kBlock) velocity_ell_kernel(const int32_t* __restrict__ cols,
                                                              const double* __restrict__ vals,
                                                              const double* __restrict__ pos, int64_t n,
                                                              int32_t width, int32_t axis, double L,
                                                              int32_t periodic, double* __restrict__ out) {
  const int64_t total = n * width;
  for (int64_t e = (int64_t)blockIdx.x * kBlock + threadIdx.x; e < total;
       e += (int64_t)gridDim.x * kBlock) {
    const int64_t i = e % n;
    const int64_t j = cols[e];
    double d = __dsub_rn(pos[j * 3 + axis], pos[i * 3 + axis]);
    if (periodic) d = __dsub_rn(d, __dmul_rn(L, rint(__ddiv_rn(d, L))));
    out[e] = __dmul_rn(vals[e], d);
  }
}

// y = V x = i (A x), A = vvals on the pattern of H; one thread per complex element of [n][R].
// partial[block] = (0, sum Re conj(L) y) when L != NULL.
__global__ void __launch_bounds__(kBlock) velocity_apply_kernel(const int32_t* __restrict__ cols,
                                                                const double* __restrict__ vvals,
                                                                int64_t n, int32_t width, int32_t R,
                                                                const double2* __restrict__ x,
                                                                double2* __restrict__ y,
                                                                const double2* __restrict__ L,
                                                                double2* __restrict__ partial) {
  const int64_t total = n * R;
  double s = 0.0;
  for (int64_t e = (int64_t)blockIdx.x * kBlock + threadIdx.x; e < total;
       e += (int64_t)gridDim.x * kBlock) {
    const int64_t i = e / R;
    const int64_t r = e - i * R;
    double re = 0.0, im = 0.0;
    for (int k = 0; k < width; ++k) {
      const int64_t c = cols[(size_t)k * n + i];
      const double v = vvals[(size_t)k * n + i];
      const double2 xv = x[c * R + r];
      re = fma(v, xv.x, re);
      im = fma(v, xv.y, im);
    }
    const double2 out = make_double2(-im, re);  // multiply by i
    y[e] = out;
    if (L) {
      const double2 l = L[e];
      s = fma(l.x, out.x, s);
      s = fma(l.y, out.y, s);
    }
  }
  __shared__ double red[kBlock / 32];
  s = warp_sum(s);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0 && partial) {
    for (int w = 1; w < kBlock / 32; ++w) s += red[w];
    partial[blockIdx.x] = make_double2(0.0, s);
  }
}

// acc = (init ? 0 : acc) + c * t   (complex), one thread per complex element
__global__ void __launch_bounds__(kBlock) caxpy_kernel(int64_t total, double cr, double ci,
                                                       const double2* __restrict__ t,
                                                       double2* __restrict__ acc, int32_t init) {
  for (int64_t e = (int64_t)blockIdx.x * kBlock + threadIdx.x; e < total;
       e += (int64_t)gridDim.x * kBlock) {
    const double2 v = t[e];
    double2 a = init ? make_double2(0.0, 0.0) : acc[e];
    a.x = fma(cr, v.x, fma(-ci, v.y, a.x));
    a.y = fma(cr, v.y, fma(ci, v.x, a.y));
    acc[e] = a;
  }
}

// C[j][n] = sums[j][n].y / norm;  flags non-finite values
__global__ void __launch_bounds__(kBlock) finish_vac_kernel(const double2* __restrict__ sums,
                                                            int64_t total, double norm,
                                                            double* __restrict__ C, int32_t* status) {
  const int64_t e = (int64_t)blockIdx.x * kBlock + threadIdx.x;
  if (e >= total) return;
  const double v = sums[e].y / norm;
  C[e] = v;
  if (!isfinite(v)) atomicOr(status, 1);
}

// sigma[0][g] = 0; sigma[j][g] = sigma[j-1][g] + scale*dt*(rho[j-1][g] + rho[j][g])/2   (V6)
__global__ void __launch_bounds__(kBlock) cumtrapz_kernel(const double* __restrict__ rho, int32_t n_steps,
                                                          int32_t G, double dt, double scale,
                                                          double* __restrict__ sigma) {
  const int g = blockIdx.x * kBlock + threadIdx.x;
  if (g >= G) return;
  double s = 0.0;
  sigma[g] = 0.0;
  for (int j = 1; j < n_steps; ++j) {
    s = s + scale * dt * (rho[(size_t)(j - 1) * G + g] + rho[(size_t)j * G + g]) / 2.0;
    sigma[(size_t)j * G + g] = s;
  }
}

int grid_for(int64_t total) {
  return (int)std::max<int64_t>(1, std::min<int64_t>((total + kBlock - 1) / kBlock, kMaxGrid));
}

// V4: c_m = e^{-i b dt} (2 - delta_m0) (-i)^m J_m(a dt), m = 0..P-1; P = first m > a dt with
// |J_m| < 1e-18.  J_m from the C library's jn().
std::vector<double2> bessel_coefficients(double a, double b, double dt) {
  const double z = a * dt;
  const double pr = std::cos(b * dt), pi = -std::sin(b * dt);
  std::vector<double2> c;
  for (int m = 0; m < 100000; ++m) {
    const double j = ::jn(m, z);
    if ((double)m > z && std::fabs(j) < 1e-18) break;
    const double w = (m == 0 ? 1.0 : 2.0) * j;
    double re, im;  // w * (-i)^m
    switch (m & 3) {
      case 0: re = w; im = 0.0; break;
      case 1: re = 0.0; im = -w; break;
      case 2: re = -w; im = 0.0; break;
      default: re = 0.0; im = w; break;
    }
    c.push_back(make_double2(re * pr - im * pi, re * pi + im * pr));
  }
  return c;
}

// state <- U(dt) state.  Buffers: *state (in), *s1, *s2 scratch; on return *state points at the
// result and *s1, *s2 at the two free buffers.  fused: `plan` is a mode-2 plan (make_plan(..., 2, ...)):
// the accumulation acc += c_m t_m runs inside the pass that produces t_m; else one caxpy launch per term.
int evolve_in_place(const gtb_ell* H, int32_t aux, const StepPlan& plan, bool fused, double a, double b,
                    const std::vector<double2>& c, int R, double** state, double** s1, double** s2,
                    double2* scratch_partial, cudaStream_t st) {
  const int64_t total = H->n * R;
  const int g = grid_for(total);
  double* x = *state;   // t_0
  double* t = *s1;      // t_1, then alternating with x
  double* acc = *s2;
  caxpy_kernel<<<g, kBlock, 0, st>>>(total, c[0].x, c[0].y, reinterpret_cast<const double2*>(x),
                                     reinterpret_cast<double2*>(acc), 1);
  GTB_LAUNCHED();
  // H: the matrix of the passes (plain, or the packed / windowed form of it: aux = blocks of the largest window)
  StepArgs sa{H->cols, H->vals, H->diag, H->n, H->width & 0xffff, plan.T, x, t, 1.0 / a, b, scratch_partial,
              nullptr};
  sa.aux = aux;
  double* cur = x;
  double* io = t;
  for (size_t m = 1; m < c.size(); ++m) {
    sa.phi_cur = cur;
    sa.phi_io = io;
    sa.scale = (m == 1 ? 1.0 : 2.0) / a;
    sa.axpy_acc = acc;
    sa.axpy_cr = c[m].x;
    sa.axpy_ci = c[m].y;
    launch_step(plan, m == 1, sa, st);  // io <- t_m  (fused: and acc += c_m t_m)
    GTB_LAUNCHED();
    if (!fused) {
      caxpy_kernel<<<g, kBlock, 0, st>>>(total, c[m].x, c[m].y, reinterpret_cast<const double2*>(io),
                                         reinterpret_cast<double2*>(acc), 0);
      GTB_LAUNCHED();
    }
    std::swap(cur, io);  // cur = t_m, io = t_{m-1} (overwritten by t_{m+1} next)
  }
  *state = acc;
  *s1 = cur;
  *s2 = io;
  return GTB_OK;
}

struct VacWs {
  int32_t* status;
  double* buf[4];
  double2* partial;  // [M][kMaxGrid]
  double2* sums;     // [n_steps][M]
  size_t bytes;
};

VacWs carve_vac(void* ws, int64_t n, int32_t M, int32_t n_steps, int32_t R) {
  Carver c(ws);
  VacWs w;
  w.status = c.take<int32_t>(64);
  for (int k = 0; k < 4; ++k) w.buf[k] = c.take<double>((size_t)n * R * 2);
  w.partial = c.take<double2>((size_t)std::max(M, 2) * kMaxGrid);
  w.sums = c.take<double2>((size_t)n_steps * M);
  w.bytes = c.off;
  return w;
}

}  // namespace
}  // namespace gtb

using namespace gtb;

extern "C" int gtb_velocity_ell(const gtb_ell* H, const double* pos, const double box[3],
                                const int32_t pbc[3], int32_t axis, double* vvals, void* stream) {
  int rc = check_ell(H);
  if (rc != GTB_OK) return rc;
  if (!pos || !box || !pbc || !vvals || axis < 0 || axis > 2) return GTB_ERR_INVALID_ARG;
  if (pbc[axis] && !(box[axis] > 0.0)) return GTB_ERR_INVALID_ARG;
  if (H->width == 0) return GTB_OK;
  velocity_ell_kernel<<<grid_for(H->n * H->width), kBlock, 0, static_cast<cudaStream_t>(stream)>>>(
      H->cols, H->vals, pos, H->n, H->width, axis, box[axis], pbc[axis] != 0, vvals);
  GTB_LAUNCHED();
  return GTB_OK;
}

extern "C" int gtb_velocity_apply(const gtb_ell* H, const double* vvals, int32_t R, const double* x,
                                  double* y, void* stream) {
  int rc = check_ell(H);
  if (rc != GTB_OK) return rc;
  if (!vvals || !x || !y || x == y || R <= 0 || R > 64) return GTB_ERR_INVALID_ARG;
  velocity_apply_kernel<<<grid_for(H->n * R), kBlock, 0, static_cast<cudaStream_t>(stream)>>>(
      H->cols, vvals, H->n, H->width, R, reinterpret_cast<const double2*>(x),
      reinterpret_cast<double2*>(y), nullptr, nullptr);
  GTB_LAUNCHED();
  return GTB_OK;
}

extern "C" size_t gtb_evolve_workspace_bytes(int64_t n, int32_t R) {
  if (n <= 0 || R <= 0) return 0;
  return carve_vac(nullptr, n, 2, 1, R).bytes;
}

extern "C" int gtb_evolve(const gtb_ell* H, double a, double b, double dt, int32_t R, double* phi,
                          int32_t* terms, void* ws, size_t ws_bytes, void* stream) {
  int rc = check_ell(H);
  if (rc != GTB_OK) return rc;
  if (!phi || !(a > 0.0) || !std::isfinite(b) || !std::isfinite(dt) || R <= 0 || R > 64 ||
      (reinterpret_cast<uintptr_t>(phi) & 31u))
    return GTB_ERR_INVALID_ARG;
  rc = check_ws(ws, ws_bytes, gtb_evolve_workspace_bytes(H->n, R));
  if (rc != GTB_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const VacWs w = carve_vac(ws, H->n, 2, 1, R);
  StepPlan plan;
  rc = make_plan(H, R, 2, nullptr, &plan);
  if (rc != GTB_OK) return rc;
  const std::vector<double2> c = bessel_coefficients(a, b, dt);
  if (terms) *terms = (int32_t)c.size();
  const size_t bytes = sizeof(double) * (size_t)H->n * R * 2;
  double *state = w.buf[0], *s1 = w.buf[1], *s2 = w.buf[2];
  GTB_CUDA_TRY(cudaMemcpyAsync(state, phi, bytes, cudaMemcpyDeviceToDevice, st));
  rc = evolve_in_place(H, 0, plan, true, a, b, c, R, &state, &s1, &s2, w.partial, st);
  if (rc != GTB_OK) return rc;
  GTB_CUDA_TRY(cudaMemcpyAsync(phi, state, bytes, cudaMemcpyDeviceToDevice, st));
  return GTB_OK;
}

extern "C" size_t gtb_vac_workspace_bytes(int64_t n, int32_t M, int32_t n_steps, int32_t R_batch) {
  if (n <= 0 || M <= 0 || n_steps <= 0 || R_batch <= 0) return 0;
  return carve_vac(nullptr, n, M, n_steps, R_batch).bytes;
}

extern "C" int gtb_vac_moments(const gtb_ell* H, const double* vvals, double a, double b, int32_t M,
                               int32_t n_steps, double dt, int32_t R_total, int32_t R_batch,
                               uint64_t seed, int32_t mode_flags, double* C, void* ws, size_t ws_bytes,
                               void* stream, const gtb_kpm_options* opt) {
  int rc = check_ell(H);
  if (rc != GTB_OK) return rc;
  rc = check_options(opt);
  if (rc != GTB_OK) return rc;
  const int opt_flags = opt ? opt->flags : 0;
  cudaEvent_t ev_beg = opt ? static_cast<cudaEvent_t>(opt->loop_begin) : nullptr;
  cudaEvent_t ev_end = opt ? static_cast<cudaEvent_t>(opt->loop_end) : nullptr;
  if ((mode_flags & ~(1 | GTB_MODE_ORB4 | GTB_MODE_ORB9)) ||
      ((mode_flags & GTB_MODE_ORB4) && (mode_flags & GTB_MODE_ORB9)))
    return GTB_ERR_INVALID_ARG;
  const int32_t mode = mode_flags & 1;
  const int orb = (mode_flags & GTB_MODE_ORB4) ? 4 : (mode_flags & GTB_MODE_ORB9) ? 9 : 0;
  if (!vvals || !C || M <= 0 || n_steps <= 0 || !(a > 0.0) || !std::isfinite(b) ||
      !std::isfinite(dt) || R_batch <= 0 || R_batch > 64 || (mode != 0 && mode != 1) ||
      (mode == 0 && R_total <= 0))
    return GTB_ERR_INVALID_ARG;
  rc = check_ws(ws, ws_bytes, gtb_vac_workspace_bytes(H->n, M, n_steps, R_batch));
  if (rc != GTB_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int64_t n = H->n;
  const VacWs w = carve_vac(ws, n, M, n_steps, R_batch);
  const int64_t n_vec = mode == 0 ? (int64_t)R_total : n;
  GTB_CUDA_TRY(cudaMemsetAsync(w.sums, 0, sizeof(double2) * (size_t)n_steps * M, st));
  GTB_CUDA_TRY(cudaMemsetAsync(w.status, 0, sizeof(int32_t) * 64, st));
  const std::vector<double2> coef = bessel_coefficients(a, b, dt);
  for (int64_t r0 = 0; r0 < n_vec; r0 += R_batch) {
    const int R = (int)std::min<int64_t>(R_batch, n_vec - r0);
    const bool last_batch = r0 + R_batch >= n_vec;
    StepPlan plan, dplan;  // evolution passes (no bra) and moment passes (dot with psiL)
    const bool direct = (opt_flags & GTB_OPT_BLOCK_DIRECT) != 0;
    bool fused = false;   // the blocked passes (K7b, K7b9) keep the separate accumulation kernel
    // the fused passes may run on a compressed form of the same matrix (gtb_kpm_options.alt): packed rows or
    // windowed tiles; the velocity operator always reads the plain ELL
    const gtb_ell *Hprop = H, *Hmom = H;   // matrices of the propagation / moment passes
    int32_t aux = 0;
    if (opt && opt->alt) {
      const gtb_ell* A = opt->alt;
      bool ok = A->n == n && !orb && R == R_batch;
      if (ok && opt->alt_mode == GTB_MODE_PACKED) {
        ok = make_plan_packed(A, R, 2, &plan) && make_plan_packed(A, R, 1, &dplan);
        Hprop = Hmom = A;
      } else if (ok && opt->alt_mode == GTB_MODE_WINDOW) {
        // windowed tiles serve the moment passes; the propagation passes (a fourth streamed vector beside a
        // 50 KB stage) measured slower on them than on K7t and stay on the plain matrix
        ok = make_plan_window(A, R, 1, opt->tile_stages, &dplan) && make_plan(H, R, 2, nullptr, &plan) == GTB_OK;
        Hmom = A;
        aux = (A->width >> 16) & 0xff;
      } else {
        ok = false;
      }
      if (!ok) return GTB_ERR_INVALID_ARG;
      fused = true;
    } else
    if (!(orb && !(opt_flags & GTB_OPT_SCALAR_BLOCKS) && make_plan_orb(H, R, orb, false, direct, &plan) &&
          make_plan_orb(H, R, orb, true, direct, &dplan))) {
      fused = !(opt_flags & GTB_OPT_SEPARATE_AXPY);
      rc = make_plan(H, R, fused ? 2 : 0, opt, &plan);
      if (rc != GTB_OK) return rc;
      rc = make_plan(H, R, 1, opt, &dplan);
      if (rc != GTB_OK) return rc;
    }
    double *psiL = w.buf[0], *psiR = w.buf[1], *sa_ = w.buf[2], *sb_ = w.buf[3];
    launch_fill(mode, seed, r0, R, n, psiL, st);
    GTB_LAUNCHED();
    velocity_apply_kernel<<<dplan.grid, kBlock, 0, st>>>(  // psiR = V phi
        H->cols, vvals, n, H->width, R, reinterpret_cast<const double2*>(psiL),
        reinterpret_cast<double2*>(psiR), nullptr, nullptr);
    GTB_LAUNCHED();
    for (int j = 0; j < n_steps; ++j) {
      if (j > 0) {
        rc = evolve_in_place(Hprop, 0, plan, fused, a, b, coef, R, &psiL, &sa_, &sb_, w.partial, st);
        if (rc != GTB_OK) return rc;
        rc = evolve_in_place(Hprop, 0, plan, fused, a, b, coef, R, &psiR, &sa_, &sb_, w.partial, st);
        if (rc != GTB_OK) return rc;
      }
      double* cur = sa_;  // chi_0 = V psiR, partial slot 0 = Re<psiL|chi_0>
      double* io = sb_;
      velocity_apply_kernel<<<dplan.grid, kBlock, 0, st>>>(
          H->cols, vvals, n, H->width, R, reinterpret_cast<const double2*>(psiR),
          reinterpret_cast<double2*>(cur), reinterpret_cast<const double2*>(psiL), w.partial);
      GTB_LAUNCHED();
      const bool timed = last_batch && j == n_steps - 1;
      if (timed && ev_beg) GTB_CUDA_TRY(cudaEventRecord(ev_beg, st));
      StepArgs sa{Hmom->cols, Hmom->vals, Hmom->diag, n, Hmom->width & 0xffff, dplan.T, cur, io, 1.0 / a, b,
                  w.partial + kMaxGrid, psiL};
      sa.aux = aux;
      for (int k = 1; k < M; ++k) {  // io <- chi_k, slot k = (Re<psiL|chi_{k-1}>, Re<psiL|chi_k>)
        sa.phi_cur = cur;
        sa.phi_io = io;
        sa.scale = (k == 1 ? 1.0 : 2.0) / a;
        sa.partial = w.partial + (size_t)k * kMaxGrid;
        launch_step(dplan, k == 1, sa, st);
        GTB_LAUNCHED();
        std::swap(cur, io);
      }
      if (timed && ev_end) {
        GTB_CUDA_TRY(cudaEventRecord(ev_end, st));
        if (opt->loop_passes) *opt->loop_passes = M - 1;
      }
      launch_reduce_partials(w.partial, kMaxGrid, dplan.grid, w.sums + (size_t)j * M, M, st);
      GTB_LAUNCHED();
    }
  }
  const double norm = mode == 0 ? (double)n * (double)R_total : (double)n;
  const int64_t total = (int64_t)n_steps * M;
  finish_vac_kernel<<<(int)((total + kBlock - 1) / kBlock), kBlock, 0, st>>>(w.sums, total, norm, C,
                                                                             w.status);
  GTB_LAUNCHED();
  return GTB_OK;
}

extern "C" int gtb_vac_conductivity(const double* C, int32_t M, int32_t n_steps, double a, double b,
                                    int32_t kernel, const double* energies, int32_t G, double dt,
                                    double scale, double* rho_vv, double* sigma, void* stream) {
  if (!C || !energies || !rho_vv || !sigma || M <= 0 || n_steps <= 0 || G < 0 || !(a > 0.0))
    return GTB_ERR_INVALID_ARG;
  if (G == 0) return GTB_OK;
  for (int j = 0; j < n_steps; ++j) {
    const int rc = gtb_dos(C + (size_t)j * M, M, a, b, kernel, energies, G, 1.0,
                           rho_vv + (size_t)j * G, stream);
    if (rc != GTB_OK) return rc;
  }
  cumtrapz_kernel<<<(G + kBlock - 1) / kBlock, kBlock, 0, static_cast<cudaStream_t>(stream)>>>(
      rho_vv, n_steps, G, dt, scale, sigma);
  GTB_LAUNCHED();
  return GTB_OK;
}

// ---- Fig. 4b post-processing (readings V7, V8 of DESIGN.md sec. 11) -------------
namespace gtb {
namespace {
// n_j = int_{e_ref}^{E_j} rho dE by the trapezoid rule; one block, a serial scan per 1024-point segment is
// not worth it at G ~ 4001: thread 0 accumulates, the others wait (G is tiny next to everything else).
__global__ void carrier_density_kernel(const double* __restrict__ rho, const double* __restrict__ E,
                                       int32_t G, double e_ref, double* __restrict__ n_out,
                                       int32_t* __restrict__ status) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  if (!(e_ref >= E[0] && e_ref <= E[G - 1])) {
    atomicOr(status, 1);
    return;
  }
  double cum = 0.0;
  n_out[0] = 0.0;
  for (int j = 1; j < G; ++j) {
    if (!(E[j] > E[j - 1])) atomicOr(status, 1);
    cum = cum + (E[j] - E[j - 1]) * (rho[j - 1] + rho[j]) / 2.0;
    n_out[j] = cum;
  }
  int k = 0;
  while (k + 2 < G && E[k + 1] < e_ref) ++k;
  const double h = E[k + 1] - E[k];
  const double t = (e_ref - E[k]) / h;
  const double rho_ref = rho[k] + t * (rho[k + 1] - rho[k]);
  const double cum_ref = n_out[k] + (e_ref - E[k]) * (rho[k] + rho_ref) / 2.0;
  for (int j = 0; j < G; ++j) n_out[j] = n_out[j] - cum_ref;
}

__global__ void __launch_bounds__(kBlock) mobility_kernel(const double* __restrict__ sigma,
                                                          const double* __restrict__ n, int32_t G,
                                                          double scale, double n_min,
                                                          double* __restrict__ mu) {
  const int j = blockIdx.x * kBlock + threadIdx.x;
  if (j >= G) return;
  const double a = fabs(n[j]);
  mu[j] = a > n_min ? scale * sigma[j] / a : 0.0;
}
}  // namespace
}  // namespace gtb

extern "C" int gtb_carrier_density(const double* rho, const double* energies, int32_t G, double e_ref,
                                   double* n_out, int32_t* status, void* stream) {
  if (!rho || !energies || !n_out || !status || G < 2 || !std::isfinite(e_ref)) return GTB_ERR_INVALID_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  GTB_CUDA_TRY(cudaMemsetAsync(status, 0, sizeof(int32_t), st));
  carrier_density_kernel<<<1, 32, 0, st>>>(rho, energies, G, e_ref, n_out, status);
  GTB_LAUNCHED();
  return GTB_OK;
}

extern "C" int gtb_mobility(const double* sigma, const double* n, int32_t G, double scale, double n_min,
                            double* mu, void* stream) {
  if (!sigma || !n || !mu || G < 0 || !(n_min >= 0.0)) return GTB_ERR_INVALID_ARG;
  if (G == 0) return GTB_OK;
  mobility_kernel<<<(G + kBlock - 1) / kBlock, kBlock, 0, static_cast<cudaStream_t>(stream)>>>(
      sigma, n, G, scale, n_min, mu);
  GTB_LAUNCHED();
  return GTB_OK;
}
