// Internal interface of the fused Chebyshev pass (K6/K7/K7t, defined in kpm.cu) for the other
// translation units of libgtb_kpm.so (vac.cu).  Product code; nothing here is used by oracle/.
#pragma once

#include "common.cuh"

namespace gtb {

constexpr int kBlock = 256;
constexpr int kMaxBlocksPerSm = 8;
constexpr int kMaxGrid = kSmCount * kMaxBlocksPerSm;

struct StepArgs {
  const int32_t* cols;
  const double* vals;
  const double* diag;
  int64_t n;
  int32_t width;
  int32_t T;              // threads per row = R*2/VW
  const double* phi_cur;  // phi_n           [n][R][2]
  double* phi_io;         // phi_{n-1} in, phi_{n+1} out
  double scale;           // 1/a (first pass) or 2/a
  double b;
  double2* partial;       // [gridDim.x]: (sum |phi_n|^2, sum Re conj(phi_{n+1}) phi_n), or with
  const double* dot_with; // dot_with = L:  (sum Re conj(L) phi_n, sum Re conj(L) phi_{n+1})
  double* axpy_acc;       // propagation passes (plan mode 2): axpy_acc += (axpy_cr + i axpy_ci) * phi_{n+1},
  double axpy_cr, axpy_ci;  // fused into the pass; no dot products are taken
  int32_t aux;              // K7w: blocks of the largest window (sizes the shared-memory stage)
};

using StepFn = void (*)(const StepArgs);
using TileFn = void (*)(const StepArgs, const int);

struct StepPlan {
  StepFn first = nullptr, next = nullptr;   // register path (K6/K7)
  TileFn tfirst = nullptr, tnext = nullptr; // TMA-staged path (K7t); used when stages > 0
  int vw = 0, T = 0;
  int grid = 0;
  int stages = 0;
  size_t smem = 0;
  int block = 0;   // threads per CTA of the staged kernel (0: the default of K7t)
};

// dot = 0: the DOS pass (dot products with phi_n itself); 1: with StepArgs::dot_with; 2: no dot products,
// the Chebyshev-Bessel accumulation StepArgs::axpy_acc += c * phi_{n+1} fused into the pass instead.
// opt (may be NULL) pins a kernel; GTB_ERR_INVALID_ARG when the pinned kernel cannot take (H, R).
int make_plan(const gtb_ell* H, int R, int dot, const gtb_kpm_options* opt, StepPlan* p);
int check_options(const gtb_kpm_options* opt);
void launch_step(const StepPlan& p, bool first, const StepArgs& sa, cudaStream_t st);
// K7b plan for an orbital-blocked matrix (B = 4: gtb_sk_hamiltonian's, B = 9: gtb_spd_hamiltonian's);
// false when H or R does not fit
bool make_plan_orb(const gtb_ell* H, int R, int B, bool dot, bool direct, StepPlan* p);
// s,p,d Hamiltonian held as 9x9 blocks (rep = 1: gtb_spd_blocks) or as bonds (rep = 2: gtb_spd_bonds);
// H->n counts atoms, the vectors have 9 H->n rows.  false when R is not 2, 4 or 8.
bool make_plan_rep9(const gtb_ell* H, int R, int rep, StepPlan* p);

// packed narrow rows (gtb_pack_ell); mode as make_plan's dot; false when (P, R) does not fit
bool make_plan_packed(const gtb_ell* P, int R, int mode, StepPlan* p);

// windowed wide rows (gtb_window_ell, built for this R); mode as make_plan's dot
bool make_plan_window(const gtb_ell* Wd, int R, int mode, int stages, StepPlan* p);

int check_ell(const gtb_ell* H);
int check_ws(const void* ws, size_t ws_bytes, size_t need);
// mode 0: random phases of (seed, r0..r0+R-1); mode 1: basis vectors e_{r0}..e_{r0+R-1}
// row_offset: global index of the first row written (a strip of the vectors)
void launch_fill(int mode, uint64_t seed, int64_t r0, int R, int64_t n, double* phi, cudaStream_t st,
                 int64_t row_offset = 0);
// mu[n] from the pass sums by the doubling identities (K8b); status: the non-finite flag
void launch_finish_moments(const double2* sums, int M, double norm, double* mu, int32_t* status, cudaStream_t st);
// sums[s] += sum_{k<grid} partial[s*stride + k]   for s = 0..nslots-1, fixed order
void launch_reduce_partials(const double2* partial, int stride, int grid, double2* sums, int nslots,
                            cudaStream_t st);

}  // namespace gtb
