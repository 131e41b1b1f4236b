// Jackson-damped density of states from Chebyshev moments (K9).
//
// Eq. 4 of the paper (printed garbled, read rho(E) = (2/Omega) Tr delta(E - H)) in
// its kernel-polynomial form (BASELINE.json:north_star (4); reading C6 in DESIGN.md):
//   rho(E) = scale * [g_0 mu_0 + 2 sum_{n>=1} g_n mu_n T_n(x)] / (pi a sqrt(1 - x^2)),  x = (E-b)/a,
// zero for |x| >= 1 - 8 eps (reading A13b: a grid end point E = b +- a comes out of fl((fl(b +- a) - b)/a)
// as +-1 or one or two ulps inside, where 1/sqrt(1 - x^2) ~ 10^8 only amplifies the rounding noise of the
// cancelling sum; such points are the end points and get rho = 0 on both sides).  The Chebyshev sum is evaluated by the Clenshaw recurrence
//   b_n = c_n + 2 x b_{n+1} - b_{n+2},  sum = c_0 + x b_1 - b_2,
// one thread per energy point, with the damped coefficients c_n = 2 g_n mu_n staged through shared
// memory in chunks from the highest order down.
#include <cmath>

#include "common.cuh"

namespace gtb {
namespace {

constexpr int kDosThreads = 128;
constexpr int kChunk = 2048;

// g_n = [(M-n+1) cos(pi n/(M+1)) + sin(pi n/(M+1)) cot(pi/(M+1))] / (M+1)   (reading A13)
__device__ __forceinline__ double jackson_g(int n, int M) {
  const double inv = 1.0 / (double)(M + 1);
  const double q = (double)n * inv;
  const double cot = cospi(inv) / sinpi(inv);
  return ((double)(M - n + 1) * cospi(q) + sinpi(q) * cot) * inv;
}

__global__ void __launch_bounds__(kDosThreads) jackson_kernel(int32_t M, double* g) {
  const int n = blockIdx.x * kDosThreads + threadIdx.x;
  if (n < M) g[n] = jackson_g(n, M);
}

__global__ void __launch_bounds__(kDosThreads)
dos_kernel(const double* __restrict__ mu, int32_t M, double a, double b, int32_t kernel,
           const double* __restrict__ energies, int32_t G, double scale, double* __restrict__ rho) {
  __shared__ double coef[kChunk];
  const int j = blockIdx.x * kDosThreads + threadIdx.x;
  const double x = j < G ? (energies[j] - b) / a : 0.0;
  const double x2 = 2.0 * x;
  double b1 = 0.0, b2 = 0.0;
  for (int hi = M; hi > 1; hi -= kChunk) {
    const int lo = max(1, hi - kChunk);
    __syncthreads();
    for (int n = lo + threadIdx.x; n < hi; n += kDosThreads)
      coef[n - lo] = 2.0 * (kernel == 1 ? jackson_g(n, M) : 1.0) * mu[n];
    __syncthreads();
    for (int n = hi - 1; n >= lo; --n) {
      const double t = fma(x2, b1, coef[n - lo]) - b2;
      b2 = b1;
      b1 = t;
    }
  }
  if (j < G) {
    double r = 0.0;
    if (fabs(x) < 1.0 - 8.0 * 2.220446049250313e-16) {   // reading A13b
      const double c0 = (kernel == 1 ? jackson_g(0, M) : 1.0) * mu[0];
      const double sum = fma(x, b1, c0) - b2;
      r = scale * sum / (3.14159265358979323846 * a * sqrt((1.0 - x) * (1.0 + x)));
    }
    rho[j] = r;
  }
}

}  // namespace
}  // namespace gtb

using namespace gtb;

extern "C" int gtb_dos(const double* mu, int32_t M, double a, double b, int32_t kernel,
                       const double* energies, int32_t G, double scale, double* rho, void* stream) {
  if (!mu || !energies || !rho || M <= 0 || G < 0 || !(a > 0.0) || (kernel != 0 && kernel != 1))
    return GTB_ERR_INVALID_ARG;
  if (G == 0) return GTB_OK;
  dos_kernel<<<(G + kDosThreads - 1) / kDosThreads, kDosThreads, 0,
               static_cast<cudaStream_t>(stream)>>>(mu, M, a, b, kernel, energies, G, scale, rho);
  GTB_LAUNCHED();
  return GTB_OK;
}

extern "C" int gtb_jackson(int32_t M, double* g, void* stream) {
  if (M <= 0 || !g) return GTB_ERR_INVALID_ARG;
  jackson_kernel<<<(M + kDosThreads - 1) / kDosThreads, kDosThreads, 0,
                   static_cast<cudaStream_t>(stream)>>>(M, g);
  GTB_LAUNCHED();
  return GTB_OK;
}
