// 1-D strip decomposition of the Chebyshev recursion, exercised on
// ONE device: the rows are cut into P contiguous strips; every strip owns its rows of the vectors plus two halo
// buffers holding the phi_n rows of its ring neighbours that its columns reach, and per pass there is ONE
// exchange step -- each halo is one contiguous copy from the neighbour's owned rows -- followed by the fused pass
// on the strip's own rows with the strip's own (column-localised) ELL.  On several GPUs the copies become peer
// copies over NVLink (one per side and pass: 2 x halo x R x 16 bytes, 1.3 MB at config 5) and the partial sums
// are all-reduced once at the end; that is the route past one GPU's memory.  Nothing here has been measured
// on more than one GPU ("unmeasured on hardware"); what is tested is that the partitioned
// run reproduces the unpartitioned one: bit-identical vectors, moments equal to the order of the block sums.
//
// Strip-local numbering: [ own rows | lo halo (the `halo` rows before row0 on the ring) | hi halo (after) ].
// The fused-pass kernels use H->n only as the row count and slot stride and gather by column index, so a strip
// runs on the unmodified kernels with H_p->n = its row count and vectors of rows + 2 halo rows.
#include <algorithm>
#include <vector>

#include "cheb.cuh"

namespace gtb {
namespace {

struct Strip {
  int64_t row0, rows;       // owned rows [row0, row0 + rows)
  int64_t lo_first, hi_first;   // global index of the first lo / hi halo row (ring)
  int32_t lo_owner, hi_owner;   // strips owning them
};

// even split in multiples of 4 rows (the staged kernels want n % 4 == 0); the last strip takes the rest
bool strip_of(int64_t n, int P, int64_t halo, int p, Strip* s) {
  if (P < 1 || p < 0 || p >= P || n <= 0 || halo < 0) return false;
  const int64_t base = n / P / 4 * 4;
  if (base <= 0) return false;
  s->row0 = base * p;
  s->rows = p == P - 1 ? n - base * (P - 1) : base;
  if (P > 1 && halo > base) return false;   // a halo must come from ONE neighbour
  if (P == 1 && halo > 0 && 2 * halo > n) return false;
  s->lo_first = ((s->row0 - halo) % n + n) % n;
  s->hi_first = (s->row0 + s->rows) % n;
  s->lo_owner = (p + P - 1) % P;
  s->hi_owner = (p + 1) % P;
  return true;
}

// largest ring distance min(|c - i|, n - |c - i|) over the genuine entries -> *out (zeroed before)
__global__ void __launch_bounds__(kBlock) ring_halo_kernel(const int32_t* __restrict__ cols, int64_t n,
                                                           int32_t width, int32_t* out) {
  const int64_t total = n * width;
  int m = 0;
  for (int64_t e = (int64_t)blockIdx.x * kBlock + threadIdx.x; e < total; e += (int64_t)gridDim.x * kBlock) {
    const int64_t i = e % n;
    int64_t d = (int64_t)cols[e] - i;
    d = d < 0 ? -d : d;
    d = min(d, n - d);
    m = max(m, (int)d);
  }
  m = warp_max_i(m);
  if ((threadIdx.x & 31) == 0 && m > 0) atomicMax(out, m);
}

// the strip's ELL in strip-local column numbering (slot stride = the strip's row count)
__global__ void __launch_bounds__(kBlock) strip_localize_kernel(const int32_t* __restrict__ cols,
                                                                const double* __restrict__ vals,
                                                                const double* __restrict__ diag, int64_t n,
                                                                int32_t width, Strip s, int64_t halo,
                                                                int32_t* __restrict__ lc, double* __restrict__ lv,
                                                                double* __restrict__ ld, int32_t* flag) {
  const int64_t total = s.rows * width;
  for (int64_t e = (int64_t)blockIdx.x * kBlock + threadIdx.x; e < total; e += (int64_t)gridDim.x * kBlock) {
    const int64_t k = e / s.rows, il = e - k * s.rows;
    const int64_t g = cols[(size_t)k * n + s.row0 + il];
    int64_t loc;
    if (g >= s.row0 && g < s.row0 + s.rows) {
      loc = g - s.row0;
    } else {
      const int64_t dlo = ((g - s.lo_first) % n + n) % n, dhi = ((g - s.hi_first) % n + n) % n;
      if (dlo < halo) loc = s.rows + dlo;
      else if (dhi < halo) loc = s.rows + halo + dhi;
      else { loc = il; atomicOr(flag, 1); }   // cannot happen when halo is the matrix's ring halo
    }
    lc[e] = (int32_t)loc;
    lv[e] = vals[(size_t)k * n + s.row0 + il];
  }
  if (ld)
    for (int64_t il = (int64_t)blockIdx.x * kBlock + threadIdx.x; il < s.rows; il += (int64_t)gridDim.x * kBlock)
      ld[il] = diag[s.row0 + il];
}

int grid_of(int64_t total) {
  return (int)std::max<int64_t>(1, std::min<int64_t>((total + kBlock - 1) / kBlock, kMaxGrid));
}

}  // namespace
}  // namespace gtb

using namespace gtb;

// HOST only.  out = { row0, rows, lo_first, hi_first, lo_owner, hi_owner } of strip p.
extern "C" int gtb_strip_plan(int64_t n, int32_t n_strips, int64_t halo, int32_t p, int64_t out[6]) {
  Strip s;
  if (!out || !strip_of(n, n_strips, halo, p, &s)) return GTB_ERR_INVALID_ARG;
  out[0] = s.row0;
  out[1] = s.rows;
  out[2] = s.lo_first;
  out[3] = s.hi_first;
  out[4] = s.lo_owner;
  out[5] = s.hi_owner;
  return GTB_OK;
}

// workspace: per strip the localised ELL, two vector sets with halos and the per-pass partial sums
extern "C" size_t gtb_strips_workspace_bytes(int64_t n, int32_t width, int32_t with_diag, int32_t n_strips,
                                             int64_t halo, int32_t M, int32_t R_batch) {
  if (n <= 0 || width < 0 || n_strips < 1 || halo < 0 || M <= 0 || R_batch <= 0) return 0;
  const size_t S = (size_t)(M + 1) / 2;
  size_t bytes = align_up(64 * sizeof(int32_t)) + align_up(S * sizeof(double2));
  for (int p = 0; p < n_strips; ++p) {
    Strip s;
    if (!strip_of(n, n_strips, halo, p, &s)) return 0;
    bytes += align_up((size_t)s.rows * width * 4) + align_up((size_t)s.rows * width * 8) +
             (with_diag ? align_up((size_t)s.rows * 8) : 0) +
             2 * align_up((size_t)(s.rows + 2 * halo) * R_batch * 16) + align_up(S * kMaxGrid * sizeof(double2));
  }
  return bytes;
}

// SYNC.  *halo (HOST) = largest ring distance |col - row| of H's genuine entries.  scratch: DEVICE int32.
extern "C" int gtb_ring_halo(const gtb_ell* H, int32_t* scratch, void* stream, int64_t* halo) {
  int rc = check_ell(H);
  if (rc != GTB_OK) return rc;
  if (!scratch || !halo) return GTB_ERR_INVALID_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  GTB_CUDA_TRY(cudaMemsetAsync(scratch, 0, sizeof(int32_t), st));
  if (H->width > 0) {
    ring_halo_kernel<<<grid_of(H->n * H->width), kBlock, 0, st>>>(H->cols, H->n, H->width, scratch);
    GTB_LAUNCHED();
  }
  int32_t h = 0;
  GTB_CUDA_TRY(cudaMemcpyAsync(&h, scratch, sizeof(h), cudaMemcpyDeviceToHost, st));
  GTB_CUDA_TRY(cudaStreamSynchronize(st));
  *halo = h;
  return GTB_OK;
}

// ASYNC.  gtb_kpm_moments on n_strips row strips with one halo exchange per pass (see the file header).
// halo: from gtb_ring_halo (or larger).  mode: 0 random phases, 1 exact trace.  R_batch: 1..64.
// phi_out (DEVICE [n][R_batch][2] or NULL): receives the LAST Chebyshev vector of the last batch, gathered
// from the strips (for the bit-identity test).  gtb_kpm_status(ws) reports non-finite moments.
extern "C" int gtb_kpm_moments_strips(const gtb_ell* H, int32_t n_strips, int64_t halo, double a, double b,
                                      int32_t M, int32_t R_total, int32_t R_batch, uint64_t seed,
                                      int32_t mode, double* mu, double* phi_out, void* ws, size_t ws_bytes,
                                      void* stream, const gtb_kpm_options* opt) {
  int rc = check_ell(H);
  if (rc != GTB_OK) return rc;
  rc = check_options(opt);
  if (rc != GTB_OK) return rc;
  if (!mu || M <= 0 || !(a > 0.0) || R_batch <= 0 || R_batch > 64 || (mode != 0 && mode != 1) ||
      (mode == 0 && R_total <= 0) || n_strips < 1 || n_strips > 64 || halo < 0)
    return GTB_ERR_INVALID_ARG;
  const int64_t n = H->n;
  const int K = H->width;
  const bool has_diag = H->diag != nullptr;
  const size_t need = gtb_strips_workspace_bytes(n, K, has_diag, n_strips, halo, M, R_batch);
  if (need == 0) return GTB_ERR_INVALID_ARG;   // strips narrower than the halo
  rc = check_ws(ws, ws_bytes, need);
  if (rc != GTB_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int S = (M + 1) / 2;
  Carver c(ws);
  int32_t* flags = c.take<int32_t>(64);
  double2* sums = c.take<double2>((size_t)S);
  struct Local {
    Strip s;
    gtb_ell H;
    double *pa, *pb;
    double2* partial;
    StepPlan plan;
  };
  std::vector<Local> L(n_strips);
  GTB_CUDA_TRY(cudaMemsetAsync(flags, 0, 64 * sizeof(int32_t), st));
  GTB_CUDA_TRY(cudaMemsetAsync(sums, 0, sizeof(double2) * (size_t)S, st));
  for (int p = 0; p < n_strips; ++p) {
    Local& l = L[p];
    strip_of(n, n_strips, halo, p, &l.s);
    l.H.n = l.s.rows;
    l.H.width = K;
    l.H.cols = c.take<int32_t>((size_t)l.s.rows * K);
    l.H.vals = c.take<double>((size_t)l.s.rows * K);
    l.H.diag = has_diag ? c.take<double>((size_t)l.s.rows) : nullptr;
    l.pa = c.take<double>((size_t)(l.s.rows + 2 * halo) * R_batch * 2);
    l.pb = c.take<double>((size_t)(l.s.rows + 2 * halo) * R_batch * 2);
    l.partial = c.take<double2>((size_t)S * kMaxGrid);
    if (K > 0 || has_diag) {
      strip_localize_kernel<<<grid_of(std::max<int64_t>(l.s.rows * std::max(K, 1), 1)), kBlock, 0, st>>>(
          H->cols, H->vals, H->diag, n, K, l.s, halo, l.H.cols, l.H.vals, l.H.diag, flags + 1);
      GTB_LAUNCHED();
    }
  }
  const int64_t n_vec = mode == 0 ? (int64_t)R_total : n;
  for (int64_t r0 = 0; r0 < n_vec; r0 += R_batch) {
    const int R = (int)std::min<int64_t>(R_batch, n_vec - r0);
    const size_t row_bytes = (size_t)R * 16;
    for (int p = 0; p < n_strips; ++p) {
      rc = make_plan(&L[p].H, R, 0, opt, &L[p].plan);
      if (rc != GTB_OK) return rc;
      launch_fill(mode, seed, r0, R, L[p].s.rows, L[p].pa, st, L[p].s.row0);
      GTB_LAUNCHED();
    }
    bool cur_is_a = true;
    for (int k = 0; k < S; ++k) {
      // the exchange step: both halos of phi_k, one contiguous copy per side, from the neighbours' owned rows
      if (halo > 0)
        for (int p = 0; p < n_strips; ++p) {
          Local& l = L[p];
          const Local& lo = L[l.s.lo_owner];
          const Local& hi = L[l.s.hi_owner];
          double* cur = cur_is_a ? l.pa : l.pb;
          const double* lo_src = (cur_is_a ? lo.pa : lo.pb) + (size_t)(lo.s.rows - halo) * R * 2;
          const double* hi_src = cur_is_a ? hi.pa : hi.pb;
          GTB_CUDA_TRY(cudaMemcpyAsync(cur + (size_t)l.s.rows * R * 2, lo_src, halo * row_bytes,
                                       cudaMemcpyDeviceToDevice, st));
          GTB_CUDA_TRY(cudaMemcpyAsync(cur + (size_t)(l.s.rows + halo) * R * 2, hi_src, halo * row_bytes,
                                       cudaMemcpyDeviceToDevice, st));
        }
      for (int p = 0; p < n_strips; ++p) {
        Local& l = L[p];
        StepArgs sa{l.H.cols, l.H.vals, l.H.diag, l.s.rows, K, l.plan.T, cur_is_a ? l.pa : l.pb,
                    cur_is_a ? l.pb : l.pa, (k == 0 ? 1.0 : 2.0) / a, b, l.partial + (size_t)k * kMaxGrid};
        launch_step(l.plan, k == 0, sa, st);
        GTB_LAUNCHED();
      }
      cur_is_a = !cur_is_a;
    }
    for (int p = 0; p < n_strips; ++p) {   // strip after strip into the same sums: a fixed order
      launch_reduce_partials(L[p].partial, kMaxGrid, L[p].plan.grid, sums, S, st);
      GTB_LAUNCHED();
    }
    if (phi_out && r0 + R_batch >= n_vec)
      for (int p = 0; p < n_strips; ++p)
        GTB_CUDA_TRY(cudaMemcpyAsync(phi_out + (size_t)L[p].s.row0 * R * 2, cur_is_a ? L[p].pa : L[p].pb,
                                     (size_t)L[p].s.rows * row_bytes, cudaMemcpyDeviceToDevice, st));
  }
  const double norm = mode == 0 ? (double)n * (double)R_total : (double)n;
  launch_finish_moments(sums, M, norm, mu, flags, st);
  GTB_LAUNCHED();
  return GTB_OK;
}
