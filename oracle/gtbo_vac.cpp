// CPU ORACLE (test infrastructure only; see gtbo.h) -- velocity autocorrelation (VAC) conductivity,
// the second quantity of the paper's LSQT stage.
//
// What the paper fixes (sec. 2.4, Eq. 3):
//     sigma(E, t) = (2 e^2 / Omega) int_0^t Tr[ delta(E - H) Re( V V(tau) ) ] dtau,
//     V(tau) = e^{i H tau} V e^{-i H tau},   V the velocity operator,
// a time step of 0.1 fs and "random states ... propagated for over 200 steps"
// (PAPER.md:68).  It prints no formula for V, for the propagator or for the trace estimator; the
// readings taken (V1-V6) are the textbook ones, in units hbar = 1 (time in
// hbar/eV, velocity in eV*Angstrom):
//   V1  V = i [H, X]  =>  V_ij = i H_ij (x_j - x_i), minimum image on periodic axes.
//   V2  Re(A) = (A + A^dagger)/2, so Tr[delta Re(V V(tau))] = Re Tr[delta U^dagger V U V],
//       U = e^{-i H tau}; with a start vector |phi>:
//           Re < U phi | delta(E - H) V | U V phi >.
//   V3  Chebyshev moments of that:  C_n(tau) = (1/(N R)) sum_r Re < psiL_r(tau) | T_n(H~) V | psiR_r(tau) >,
//       psiL(tau) = U(tau) phi, psiR(tau) = U(tau) V phi, by the recursion chi_0 = V psiR,
//       chi_1 = H~ chi_0, chi_{n+1} = 2 H~ chi_n - chi_{n-1}, C_n = Re <psiL|chi_n>  (M - 1 SpMVs per time).
//   V4  U(dt) = e^{-i b dt} sum_m (2 - delta_m0) (-i)^m J_m(a dt) T_m(H~)  (Chebyshev-Bessel expansion),
//       truncated after the first m > a dt with |J_m(a dt)| < 1e-18; states advance step by step.
//   V5  rho_vv(E, tau) = the kernel-damped reconstruction of C_n(tau) exactly as the DOS (gtbo_dos).
//   V6  the time integral is the trapezoid rule on the grid tau_j = j dt, sigma(E, 0) = 0.
// Every step is written in that order; the only parallel loops are over independent rows.
#include "gtbo.h"

#include <cmath>
#include <complex>
#include <cstring>
#include <vector>

namespace {

using cd = std::complex<double>;

// y = A x for the ELL pattern of H with the values `vals` ([width][n]) and an optional diagonal
void ell_apply(const gtbo_ell* H, const double* vals, const double* diag, const cd* x, cd* y) {
  const int64_t n = H->n;
#pragma omp parallel for schedule(static) if (n > 16384)
  for (int64_t i = 0; i < n; ++i) {
    double re = 0.0, im = 0.0;
    for (int32_t k = 0; k < H->width; ++k) {
      const double v = vals[(size_t)k * n + i];
      const int32_t j = H->cols[(size_t)k * n + i];
      re = re + v * x[j].real();
      im = im + v * x[j].imag();
    }
    if (diag) {
      re = re + diag[i] * x[i].real();
      im = im + diag[i] * x[i].imag();
    }
    y[i] = cd(re, im);
  }
}

// y = V x,  V = i * vvals  (V1):  i (re + i im) = -im + i re
void velocity(const gtbo_ell* H, const double* vvals, const cd* x, cd* y) {
  ell_apply(H, vvals, nullptr, x, y);
  for (int64_t i = 0; i < H->n; ++i) y[i] = cd(-y[i].imag(), y[i].real());
}

// y = H~ x = (H x - b x)/a   and   z = 2 H~ y - x
void cheb_first(const gtbo_ell* H, double a, double b, const cd* x, cd* y) {
  ell_apply(H, H->vals, H->diag, x, y);
  const double s = 1.0 / a;
  for (int64_t i = 0; i < H->n; ++i)
    y[i] = cd((y[i].real() - b * x[i].real()) * s, (y[i].imag() - b * x[i].imag()) * s);
}
void cheb_next(const gtbo_ell* H, double a, double b, const cd* xm, const cd* x, cd* y) {
  ell_apply(H, H->vals, H->diag, x, y);
  const double s = 2.0 / a;
  for (int64_t i = 0; i < H->n; ++i)
    y[i] = cd((y[i].real() - b * x[i].real()) * s - xm[i].real(),
              (y[i].imag() - b * x[i].imag()) * s - xm[i].imag());
}

double re_dot(const cd* x, const cd* y, int64_t n) {  // Re <x|y>
  double s = 0.0;
  for (int64_t i = 0; i < n; ++i) s += x[i].real() * y[i].real() + x[i].imag() * y[i].imag();
  return s;
}

// V4: c_m = (2 - delta_m0) (-i)^m J_m(z), m = 0..P-1
std::vector<cd> bessel_coeffs(double z) {
  std::vector<cd> c;
  const cd mi[4] = {cd(1, 0), cd(0, -1), cd(-1, 0), cd(0, 1)};  // (-i)^m
  for (int m = 0; m < 100000; ++m) {
    const double j = std::cyl_bessel_j((double)m, z);
    if ((double)m > z && std::fabs(j) < 1e-18) break;
    c.push_back((m == 0 ? 1.0 : 2.0) * j * mi[m & 3]);
  }
  return c;
}

// y = U(dt) x  (V4)
int evolve(const gtbo_ell* H, double a, double b, double dt, const std::vector<cd>& x,
           std::vector<cd>& y) {
  const int64_t n = H->n;
  const std::vector<cd> c = bessel_coeffs(a * dt);
  std::vector<cd> tm(x), t(n), tp(n), acc(n);
  for (int64_t i = 0; i < n; ++i) acc[i] = c[0] * tm[i];
  if (c.size() > 1) {
    cheb_first(H, a, b, tm.data(), t.data());
    for (int64_t i = 0; i < n; ++i) acc[i] += c[1] * t[i];
  }
  for (size_t m = 2; m < c.size(); ++m) {
    cheb_next(H, a, b, tm.data(), t.data(), tp.data());
    for (int64_t i = 0; i < n; ++i) acc[i] += c[m] * tp[i];
    tm.swap(t);
    t.swap(tp);
  }
  const cd phase(std::cos(b * dt), -std::sin(b * dt));
  y.resize(n);
  for (int64_t i = 0; i < n; ++i) y[i] = phase * acc[i];
  return (int)c.size();
}

void load(const double* p, int64_t n, int32_t R, int32_t r, std::vector<cd>& v) {
  v.resize(n);
  for (int64_t i = 0; i < n; ++i) v[i] = cd(p[((size_t)i * R + r) * 2], p[((size_t)i * R + r) * 2 + 1]);
}
void store(const std::vector<cd>& v, int32_t R, int32_t r, double* p) {
  for (size_t i = 0; i < v.size(); ++i) {
    p[(i * R + r) * 2] = v[i].real();
    p[(i * R + r) * 2 + 1] = v[i].imag();
  }
}

}  // namespace

// V1: vvals[k][i] = vals[k][i] * (x_j - x_i)_axis, j = cols[k][i]; minimum image d -= L rint(d/L).
extern "C" int gtbo_velocity_ell(const gtbo_ell* H, const double* pos, const double box[3],
                                 const int32_t pbc[3], int32_t axis, double* vvals) {
  if (!H || !pos || !box || !pbc || !vvals || axis < 0 || axis > 2) return GTBO_ERR_INVALID_ARG;
  const int64_t n = H->n;
  for (int32_t k = 0; k < H->width; ++k)
    for (int64_t i = 0; i < n; ++i) {
      const int64_t j = H->cols[(size_t)k * n + i];
      double d = pos[(size_t)j * 3 + axis] - pos[(size_t)i * 3 + axis];
      if (pbc[axis]) d = d - box[axis] * std::nearbyint(d / box[axis]);
      vvals[(size_t)k * n + i] = H->vals[(size_t)k * n + i] * d;
    }
  return GTBO_OK;
}

// y = V x for R interleaved vectors ([n][R][2])
extern "C" int gtbo_velocity_apply(const gtbo_ell* H, const double* vvals, int32_t R, const double* x,
                                   double* y) {
  if (!H || !vvals || !x || !y || R <= 0) return GTBO_ERR_INVALID_ARG;
  std::vector<cd> a, b(H->n);
  for (int32_t r = 0; r < R; ++r) {
    load(x, H->n, R, r, a);
    velocity(H, vvals, a.data(), b.data());
    store(b, R, r, y);
  }
  return GTBO_OK;
}

// y = e^{-i H dt} x for R interleaved vectors; *terms = number of Chebyshev terms used
extern "C" int gtbo_evolve(const gtbo_ell* H, double a, double b, double dt, int32_t R,
                           const double* x, double* y, int32_t* terms) {
  if (!H || !x || !y || R <= 0 || !(a > 0.0)) return GTBO_ERR_INVALID_ARG;
  std::vector<cd> u, v;
  for (int32_t r = 0; r < R; ++r) {
    load(x, H->n, R, r, u);
    const int p = evolve(H, a, b, dt, u, v);
    if (terms) *terms = p;
    store(v, R, r, y);
  }
  return GTBO_OK;
}

// V2/V3: C[j][n], j = 0..n_steps-1 (tau_j = j dt), n = 0..M-1.  mode as gtbo_kpm_moments.
extern "C" int gtbo_vac_moments(const gtbo_ell* H, const double* vvals, double a, double b,
                                int32_t M, int32_t n_steps, double dt, int32_t R, uint64_t seed,
                                int32_t mode, double* C) {
  if (!H || !vvals || !C || M <= 0 || n_steps <= 0 || !(a > 0.0) || (mode == 0 && R <= 0) ||
      (mode != 0 && mode != 1))
    return GTBO_ERR_INVALID_ARG;
  const int64_t n = H->n;
  const int64_t n_vec = mode == 0 ? R : n;
  std::vector<double> sum((size_t)n_steps * M, 0.0);
  for (int64_t r = 0; r < n_vec; ++r) {
    std::vector<cd> phi(n, cd(0, 0));
    if (mode == 0) {
      for (int64_t i = 0; i < n; ++i) {
        const double th = 6.283185307179586 * gtbo_uniform(seed, (uint32_t)r, (uint64_t)i);
        phi[i] = cd(std::cos(th), std::sin(th));
      }
    } else {
      phi[r] = cd(1, 0);
    }
    std::vector<cd> psiL(phi), psiR(n), tmp, cm(n), c0(n), cp(n);
    velocity(H, vvals, phi.data(), psiR.data());
    for (int32_t j = 0; j < n_steps; ++j) {
      if (j > 0) {
        evolve(H, a, b, dt, psiL, tmp);
        psiL.swap(tmp);
        evolve(H, a, b, dt, psiR, tmp);
        psiR.swap(tmp);
      }
      double* out = &sum[(size_t)j * M];
      velocity(H, vvals, psiR.data(), cm.data());  // chi_0
      out[0] += re_dot(psiL.data(), cm.data(), n);
      if (M == 1) continue;
      cheb_first(H, a, b, cm.data(), c0.data());  // chi_1
      out[1] += re_dot(psiL.data(), c0.data(), n);
      for (int32_t k = 2; k < M; ++k) {
        cheb_next(H, a, b, cm.data(), c0.data(), cp.data());
        out[k] += re_dot(psiL.data(), cp.data(), n);
        cm.swap(c0);
        c0.swap(cp);
      }
    }
  }
  const double norm = mode == 0 ? (double)n * (double)R : (double)n;
  for (size_t q = 0; q < sum.size(); ++q) C[q] = sum[q] / norm;
  return GTBO_OK;
}

// V5/V6: rho_vv[j][g] = reconstruction of C[j][:] at E_g (as gtbo_dos, scale 1);
// sigma[0][g] = 0, sigma[j][g] = sigma[j-1][g] + scale dt (rho_vv[j-1][g] + rho_vv[j][g])/2.
extern "C" int gtbo_vac_conductivity(const double* C, int32_t M, int32_t n_steps, double a, double b,
                                     int32_t kernel, const double* energies, int32_t G, double dt,
                                     double scale, double* rho_vv, double* sigma) {
  if (!C || !energies || !sigma || M <= 0 || n_steps <= 0 || G < 0) return GTBO_ERR_INVALID_ARG;
  std::vector<double> rv((size_t)n_steps * G);
  for (int32_t j = 0; j < n_steps; ++j) {
    const int rc = gtbo_dos(C + (size_t)j * M, M, a, b, kernel, energies, G, 1.0, &rv[(size_t)j * G]);
    if (rc != GTBO_OK) return rc;
  }
  for (int32_t g = 0; g < G; ++g) {
    sigma[g] = 0.0;
    for (int32_t j = 1; j < n_steps; ++j)
      sigma[(size_t)j * G + g] =
          sigma[(size_t)(j - 1) * G + g] +
          scale * dt * (rv[(size_t)(j - 1) * G + g] + rv[(size_t)j * G + g]) / 2.0;
  }
  if (rho_vv) std::memcpy(rho_vv, rv.data(), sizeof(double) * rv.size());
  return GTBO_OK;
}

// --- post-processing of Fig. 4b: carrier density and mobility --------------------
// The paper plots mobility against carrier concentration and prints no formula; readings (DESIGN.md
// sec. 11, V7-V8): V7 carrier density relative to the reference energy E_ref (the charge-neutrality
// point), n(E_j) = int_{E_ref}^{E_j} rho(E) dE by the trapezoid rule on the given grid, with rho
// interpolated linearly at E_ref; negative below E_ref (holes).  V8 semiclassical mobility
// mu(E_j) = sigma(E_j) / (e |n(E_j)|) with e folded into `scale`; where |n| <= n_min the mobility is
// reported as 0 (the neutrality point itself has no carriers to carry it).
extern "C" int gtbo_carrier_density(const double* rho, const double* energies, int32_t G, double e_ref,
                                    double* n_out) {
  if (!rho || !energies || !n_out || G < 2) return GTBO_ERR_INVALID_ARG;
  for (int32_t j = 1; j < G; ++j)
    if (!(energies[j] > energies[j - 1])) return GTBO_ERR_INVALID_ARG;
  if (!(e_ref >= energies[0] && e_ref <= energies[G - 1])) return GTBO_ERR_INVALID_ARG;
  std::vector<double> cum(G, 0.0);   // int_{E_0}^{E_j}
  for (int32_t j = 1; j < G; ++j)
    cum[j] = cum[j - 1] + (energies[j] - energies[j - 1]) * (rho[j - 1] + rho[j]) / 2.0;
  int32_t k = 0;                      // E_k <= e_ref <= E_{k+1}
  while (k + 2 < G && energies[k + 1] < e_ref) ++k;
  const double h = energies[k + 1] - energies[k];
  const double t = (e_ref - energies[k]) / h;
  const double rho_ref = rho[k] + t * (rho[k + 1] - rho[k]);
  const double cum_ref = cum[k] + (e_ref - energies[k]) * (rho[k] + rho_ref) / 2.0;
  for (int32_t j = 0; j < G; ++j) n_out[j] = cum[j] - cum_ref;
  return GTBO_OK;
}

extern "C" int gtbo_mobility(const double* sigma, const double* n, int32_t G, double scale, double n_min,
                             double* mu) {
  if (!sigma || !n || !mu || G < 0 || !(n_min >= 0.0)) return GTBO_ERR_INVALID_ARG;
  for (int32_t j = 0; j < G; ++j) {
    const double a = std::fabs(n[j]);
    mu[j] = a > n_min ? scale * sigma[j] / a : 0.0;
  }
  return GTBO_OK;
}
