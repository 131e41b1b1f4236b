// Hamiltonian assembly on the device: cell binning (K1/K2), neighbour search + sort +
// hopping -> ELL (K3), Gershgorin bounds (K4).
//
// Computes Eq. 1 of the paper, H = sum_i eps_i c+_i c_i + sum_{j in N(i)} t_ij
// c+_i c_j, for one p_z orbital per atom (BASELINE.json:north_star (1)), with N(i) the atoms
// inside the cutoff radius.  The distance rule is reading C2/A14/A15 of
// raw differences of the unwrapped coordinates, minimum image by rint, r2 summed left
// to right in fp64 WITHOUT fused multiply-add (the *_rn intrinsics below forbid contraction), and
// a strict r2 < cutoff^2 test -- this is what makes the column indices bit-reproducible.
#include <algorithm>
#include <cmath>

#include "common.cuh"

namespace gtb {
namespace {

constexpr int kThreads = 256;
constexpr int kScanThreads = 512;
constexpr int kScanItems = 4;
constexpr int kScanTile = kScanThreads * kScanItems;
constexpr int kPartialBlocks = kSmCount * 8;

struct CellGrid {
  int nc[3];
  int pbc[3];
  double lo[3];   // origin of the grid on a non-periodic axis
  double h[3];    // cell edge
  double box[3];
};

struct ModelParams {
  int n_species;
  double onsite[GTB_MAX_SPECIES];
  double t0[GTB_MAX_SPECIES * GTB_MAX_SPECIES];
  double r0, beta;
  const double* onsite_shift;
};

__device__ __forceinline__ int cell_coord(const CellGrid& g, double x, int a) {
  double w;
  if (g.pbc[a]) {
    w = x - g.box[a] * floor(x / g.box[a]);  // wrapped copy: used ONLY to choose the cell
  } else {
    w = x - g.lo[a];
  }
  int c = (int)floor(w / g.h[a]);
  c = max(c, 0);
  c = min(c, g.nc[a] - 1);
  return c;
}

__device__ __forceinline__ int64_t cell_index(const CellGrid& g, int cx, int cy, int cz) {
  return ((int64_t)cz * g.nc[1] + cy) * g.nc[0] + cx;
}

// ---- K0: bounding box of the positions (needed for non-periodic axes) -------------
__global__ void __launch_bounds__(kThreads) bounds_partial_kernel(const double* __restrict__ pos,
                                                                  int64_t n, double* partial) {
  double mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
  for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < n;
       i += (int64_t)gridDim.x * kThreads) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const double x = pos[3 * i + a];
      mn[a] = fmin(mn[a], x);
      mx[a] = fmax(mx[a], x);
    }
  }
  __shared__ double s[kThreads / 32][6];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double lo = warp_min(mn[a]), hi = warp_max(mx[a]);
    if (lane == 0) {
      s[wid][a] = lo;
      s[wid][3 + a] = hi;
    }
  }
  __syncthreads();
  if (threadIdx.x < 6) {
    double v = s[0][threadIdx.x];
    for (int w = 1; w < kThreads / 32; ++w)
      v = threadIdx.x < 3 ? fmin(v, s[w][threadIdx.x]) : fmax(v, s[w][threadIdx.x]);
    partial[(size_t)blockIdx.x * 6 + threadIdx.x] = v;
  }
}

__global__ void bounds_final_kernel(const double* partial, int blocks, double* out6) {
  const int k = threadIdx.x;
  if (k < 6) {
    double v = partial[k];
    for (int b = 1; b < blocks; ++b)
      v = k < 3 ? fmin(v, partial[(size_t)b * 6 + k]) : fmax(v, partial[(size_t)b * 6 + k]);
    out6[k] = v;
  }
}

// ---- K1: cell of each atom, running count per cell ----------------------------------
__global__ void __launch_bounds__(kThreads) bin_kernel(const double* __restrict__ pos, int64_t n,
                                                       CellGrid g, int32_t* __restrict__ cell_of,
                                                       int32_t* __restrict__ local_off,
                                                       int32_t* cell_count) {
  const int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x;
  if (i >= n) return;
  const int cx = cell_coord(g, pos[3 * i + 0], 0);
  const int cy = cell_coord(g, pos[3 * i + 1], 1);
  const int cz = cell_coord(g, pos[3 * i + 2], 2);
  const int32_t c = (int32_t)cell_index(g, cx, cy, cz);
  cell_of[i] = c;
  // the order of atoms inside a cell is irrelevant: K3 sorts each row by column
  local_off[i] = atomicAdd(&cell_count[c], 1);
}

// ---- K2: exclusive scan (in place) over the cell counts ---------------------------
__device__ __forceinline__ int block_exclusive_scan(int v, int* total) {
  // v: this thread's value; returns the exclusive prefix inside the block
  __shared__ int warp_tot[kScanThreads / 32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) warp_tot[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    int w = lane < kScanThreads / 32 ? warp_tot[lane] : 0;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, w, o);
      if (lane >= o) w += t;
    }
    if (lane < kScanThreads / 32) warp_tot[lane] = w;  // inclusive over warps
  }
  __syncthreads();
  const int base = wid == 0 ? 0 : warp_tot[wid - 1];
  *total = warp_tot[kScanThreads / 32 - 1];
  return base + inc - v;
}

__global__ void __launch_bounds__(kScanThreads) scan_tile_sums_kernel(const int32_t* data,
                                                                      int64_t count,
                                                                      int32_t* sums) {
  const int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
  int v = 0;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k)
    if (base + k < count) v += data[base + k];
  int total;
  block_exclusive_scan(v, &total);
  if (threadIdx.x == 0) sums[blockIdx.x] = total;
}

__global__ void __launch_bounds__(kScanThreads) scan_tile_apply_kernel(int32_t* data, int64_t count,
                                                                       const int32_t* sums) {
  const int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
  int x[kScanItems];
  int v = 0;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    x[k] = base + k < count ? data[base + k] : 0;
    v += x[k];
  }
  int total;
  int run = block_exclusive_scan(v, &total) + (sums ? sums[blockIdx.x] : 0);
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    if (base + k < count) data[base + k] = run;
    run += x[k];
  }
}

int exclusive_scan_inplace(int32_t* data, int64_t count, int32_t* sums_ws, cudaStream_t st) {
  const int64_t tiles = (count + kScanTile - 1) / kScanTile;
  if (tiles <= 1) {
    scan_tile_apply_kernel<<<1, kScanThreads, 0, st>>>(data, count, nullptr);
    GTB_LAUNCHED();
    return GTB_OK;
  }
  scan_tile_sums_kernel<<<(unsigned)tiles, kScanThreads, 0, st>>>(data, count, sums_ws);
  GTB_LAUNCHED();
  int rc = exclusive_scan_inplace(sums_ws, tiles, sums_ws + align_up(tiles * 4) / 4, st);
  if (rc != GTB_OK) return rc;
  scan_tile_apply_kernel<<<(unsigned)tiles, kScanThreads, 0, st>>>(data, count, sums_ws);
  GTB_LAUNCHED();
  return GTB_OK;
}

size_t scan_ws_ints(int64_t count) {
  size_t total = 0;
  int64_t c = count;
  while (c > kScanTile) {
    c = (c + kScanTile - 1) / kScanTile;
    total += align_up((size_t)c * 4) / 4;
  }
  return total + 64;
}

// ---- K2b: atoms sorted by cell: record = (x, y, z, id) ------------------------------
__global__ void __launch_bounds__(kThreads) fill_kernel(const double* __restrict__ pos, int64_t n,
                                                        const int32_t* __restrict__ cell_of,
                                                        const int32_t* __restrict__ local_off,
                                                        const int32_t* __restrict__ cell_start,
                                                        double4* __restrict__ rec) {
  const int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x;
  if (i >= n) return;
  const int64_t slot = (int64_t)cell_start[cell_of[i]] + local_off[i];
  rec[slot] = make_double4(pos[3 * i + 0], pos[3 * i + 1], pos[3 * i + 2],
                           __longlong_as_double((long long)i));
}

// ---- K3: neighbour search, sort by column, hopping, ELL rows ------------------------
// distinct neighbouring cell coordinates along one axis (a periodic axis with fewer than three
// cells would otherwise visit the same cell twice)
__device__ __forceinline__ int axis_cells(const CellGrid& g, int a, int c, int out[3]) {
  int m = 0;
  for (int s = -1; s <= 1; ++s) {
    int k = c + s;
    if (g.pbc[a]) {
      if (k < 0) k += g.nc[a];
      if (k >= g.nc[a]) k -= g.nc[a];
    } else if (k < 0 || k >= g.nc[a]) {
      continue;
    }
    bool seen = false;
    for (int q = 0; q < m; ++q) seen |= (out[q] == k);
    if (!seen) out[m++] = k;
  }
  return m;
}

__device__ __forceinline__ double min_image(double d, double L, int periodic) {
  if (periodic) {
    const double q = __ddiv_rn(d, L);
    const double k = rint(q);  // ties to even
    d = __dsub_rn(d, __dmul_rn(L, k));
  }
  return d;
}

template <bool kCountOnly>
__global__ void __launch_bounds__(kThreads)
neighbor_kernel(const double* __restrict__ pos, const int32_t* __restrict__ species, int64_t n,
                CellGrid g, double rc2, const int32_t* __restrict__ cell_start,
                const double4* __restrict__ rec, ModelParams m, int32_t width,
                int32_t* __restrict__ cols, double* __restrict__ vals, double* __restrict__ diag,
                int32_t* __restrict__ counts, int32_t* flags /* [0]=max count, [1]=bad species */) {
  const int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x;
  int cnt = 0;
  if (i < n) {
    const double xi = pos[3 * i + 0], yi = pos[3 * i + 1], zi = pos[3 * i + 2];
    int ax[3][3], na[3];
    na[0] = axis_cells(g, 0, cell_coord(g, xi, 0), ax[0]);
    na[1] = axis_cells(g, 1, cell_coord(g, yi, 1), ax[1]);
    na[2] = axis_cells(g, 2, cell_coord(g, zi, 2), ax[2]);
    int32_t cj[GTB_MAX_WIDTH];
    double cr[GTB_MAX_WIDTH];
    for (int iz = 0; iz < na[2]; ++iz)
      for (int iy = 0; iy < na[1]; ++iy)
        for (int ix = 0; ix < na[0]; ++ix) {
          const int64_t c = cell_index(g, ax[0][ix], ax[1][iy], ax[2][iz]);
          const int32_t beg = cell_start[c], end = cell_start[c + 1];
          for (int32_t s = beg; s < end; ++s) {
            const double4 p = rec[s];
            const int64_t j = __double_as_longlong(p.w);
            if (j == i) continue;
            const double dx = min_image(__dsub_rn(p.x, xi), g.box[0], g.pbc[0]);
            const double dy = min_image(__dsub_rn(p.y, yi), g.box[1], g.pbc[1]);
            const double dz = min_image(__dsub_rn(p.z, zi), g.box[2], g.pbc[2]);
            const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)),
                                        __dmul_rn(dz, dz));
            if (r2 < rc2) {
              if (!kCountOnly && cnt < GTB_MAX_WIDTH) {
                cj[cnt] = (int32_t)j;
                cr[cnt] = r2;
              }
              ++cnt;
            }
          }
        }
    if (counts) counts[i] = cnt;
    if (!kCountOnly) {
      const int si = species[i];
      bool ok = si >= 0 && si < m.n_species;
      if (cnt <= width && cnt <= GTB_MAX_WIDTH && ok) {
        for (int p = 1; p < cnt; ++p) {  // insertion sort by column
          const int32_t j = cj[p];
          const double r = cr[p];
          int q = p - 1;
          while (q >= 0 && cj[q] > j) {
            cj[q + 1] = cj[q];
            cr[q + 1] = cr[q];
            --q;
          }
          cj[q + 1] = j;
          cr[q + 1] = r;
        }
        for (int k = 0; k < width; ++k) {
          int32_t col = (int32_t)i;
          double t = 0.0;
          if (k < cnt) {
            col = cj[k];
            const int sj = species[col];
            if (sj < 0 || sj >= m.n_species) {
              ok = false;
            } else {
              t = m.t0[si * m.n_species + sj];
              if (m.beta != 0.0) {
                const double r = sqrt(cr[k]);
                const double arg = __dmul_rn(-m.beta, __dsub_rn(__ddiv_rn(r, m.r0), 1.0));
                t = __dmul_rn(t, exp(arg));
              }
            }
          }
          cols[(size_t)k * n + i] = col;
          vals[(size_t)k * n + i] = t;
        }
        if (diag) {
          double e = ok ? m.onsite[si] : 0.0;
          if (m.onsite_shift) e = __dadd_rn(e, m.onsite_shift[i]);
          diag[i] = e;
        }
      }
      if (!ok) atomicOr(&flags[1], 1);
    }
  }
  const int wmax = warp_max_i(cnt);
  if ((threadIdx.x & 31) == 0 && wmax > 0) atomicMax(&flags[0], wmax);
}

// ---- K4: Gershgorin bounds -----------------------------------------------------------
__global__ void __launch_bounds__(kThreads)
gershgorin_partial_kernel(const int32_t width, const int64_t n, const double* __restrict__ vals,
                          const double* __restrict__ diag, double* partial) {
  double lo = INFINITY, hi = -INFINITY;
  for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < n;
       i += (int64_t)gridDim.x * kThreads) {
    double off = 0.0;
    for (int k = 0; k < width; ++k) off += fabs(vals[(size_t)k * n + i]);
    const double d = diag ? diag[i] : 0.0;
    lo = fmin(lo, d - off);
    hi = fmax(hi, d + off);
  }
  __shared__ double s[kThreads / 32][2];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  lo = warp_min(lo);
  hi = warp_max(hi);
  if (lane == 0) {
    s[wid][0] = lo;
    s[wid][1] = hi;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < kThreads / 32; ++w) {
      lo = fmin(lo, s[w][0]);
      hi = fmax(hi, s[w][1]);
    }
    partial[2 * blockIdx.x + 0] = lo;
    partial[2 * blockIdx.x + 1] = hi;
  }
}

__global__ void gershgorin_final_kernel(const double* partial, int blocks, double* lo_hi) {
  if (threadIdx.x == 0) {
    double lo = partial[0], hi = partial[1];
    for (int b = 1; b < blocks; ++b) {
      lo = fmin(lo, partial[2 * b]);
      hi = fmax(hi, partial[2 * b + 1]);
    }
    lo_hi[0] = lo;
    lo_hi[1] = hi;
  }
}

// ---- host side -------------------------------------------------------------------------
// cell indices are int32: the cap never exceeds INT32_MAX - 64 (beyond n ~ 1.07e9 atoms the grid is
// simply coarser than two cells per atom)
int64_t cell_cap(int64_t n) { return std::min<int64_t>(2 * n + 1024, (int64_t)INT32_MAX - 64); }

struct BuildWs {
  int32_t* cell_of;
  int32_t* local_off;
  double4* rec;
  int32_t* cell_start;  // [cap + 2]
  int32_t* scan_sums;
  double* bounds_partial;  // [kPartialBlocks][6] + 6
  int32_t* flags;          // [16]
  size_t bytes;
};

BuildWs carve_build(void* ws, int64_t n) {
  Carver c(ws);
  BuildWs w;
  w.rec = c.take<double4>((size_t)n);
  w.cell_of = c.take<int32_t>((size_t)n);
  w.local_off = c.take<int32_t>((size_t)n);
  w.cell_start = c.take<int32_t>((size_t)cell_cap(n) + 2);
  w.scan_sums = c.take<int32_t>(scan_ws_ints(cell_cap(n) + 2));
  w.bounds_partial = c.take<double>((size_t)kPartialBlocks * 6 + 6);
  w.flags = c.take<int32_t>(16);
  w.bytes = c.off;
  return w;
}

int check_geometry(const double* pos, int64_t n, const double box[3], const int32_t pbc[3],
                   double cutoff) {
  if (!pos || n < 0 || !box || !pbc || !(cutoff > 0.0)) return GTB_ERR_INVALID_ARG;
  if (n > (int64_t)INT32_MAX - 64) return GTB_ERR_INDEX_RANGE;
  for (int a = 0; a < 3; ++a)
    if (pbc[a]) {
      if (!(box[a] > 0.0)) return GTB_ERR_INVALID_ARG;
      if (box[a] < 2.0 * cutoff) return GTB_ERR_BOX_TOO_SMALL;
    }
  return GTB_OK;
}

int check_ws(const void* ws, size_t ws_bytes, size_t need) {
  if (!ws || (reinterpret_cast<uintptr_t>(ws) & 255u) || ws_bytes < need) return GTB_ERR_WORKSPACE;
  return GTB_OK;
}

// Chooses the cell grid (host) and bins the atoms (device).  Cells are at least 1.001*cutoff
// wide so that the 3x3x3 block around an atom's cell covers its cutoff sphere even when the
// wrapped coordinate used for binning is off by a rounding error; the grid is coarsened until it
// has at most cell_cap(n) cells (a 2-D sheet in a 3-D box must not create empty cell layers).
int make_cells(const double* pos, int64_t n, const double box[3], const int32_t pbc[3],
               double cutoff, const BuildWs& w, cudaStream_t st, CellGrid* g) {
  double lohi[6] = {0, 0, 0, 0, 0, 0};
  if (!(pbc[0] && pbc[1] && pbc[2])) {
    const int blocks = (int)std::min<int64_t>(kPartialBlocks, (n + kThreads - 1) / kThreads);
    bounds_partial_kernel<<<blocks, kThreads, 0, st>>>(pos, n, w.bounds_partial);
    GTB_LAUNCHED();
    double* out6 = w.bounds_partial + (size_t)kPartialBlocks * 6;
    bounds_final_kernel<<<1, 32, 0, st>>>(w.bounds_partial, blocks, out6);
    GTB_LAUNCHED();
    GTB_CUDA_TRY(cudaMemcpyAsync(lohi, out6, sizeof(lohi), cudaMemcpyDeviceToHost, st));
    GTB_CUDA_TRY(cudaStreamSynchronize(st));
  }
  double edge = cutoff * 1.001;
  for (int iter = 0; iter < 64; ++iter) {
    double total = 1.0;
    int active = 0;
    for (int a = 0; a < 3; ++a) {
      g->pbc[a] = pbc[a] ? 1 : 0;
      g->box[a] = box[a];
      if (pbc[a]) {
        g->lo[a] = 0.0;
        g->nc[a] = std::max(1, (int)std::floor(box[a] / edge));
        g->h[a] = box[a] / g->nc[a];
      } else {
        const double extent = lohi[3 + a] - lohi[a];
        if (!std::isfinite(extent)) return GTB_ERR_INVALID_ARG;  // NaN/inf coordinates
        g->lo[a] = lohi[a];
        g->nc[a] = std::max(1, (int)std::floor(extent / edge) + 1);
        g->h[a] = edge;
      }
      total *= g->nc[a];
      active += g->nc[a] > 1;
    }
    if (total <= (double)cell_cap(n) || active == 0) break;
    edge *= std::max(1.05, std::pow(total / (double)cell_cap(n), 1.0 / active));
  }
  const int64_t ncell = (int64_t)g->nc[0] * g->nc[1] * g->nc[2];
  if (ncell > cell_cap(n)) return GTB_ERR_INVALID_ARG;
  GTB_CUDA_TRY(cudaMemsetAsync(w.cell_start, 0, (size_t)(ncell + 2) * sizeof(int32_t), st));
  GTB_CUDA_TRY(cudaMemsetAsync(w.flags, 0, 16 * sizeof(int32_t), st));
  const unsigned blocks = (unsigned)((n + kThreads - 1) / kThreads);
  bin_kernel<<<blocks, kThreads, 0, st>>>(pos, n, *g, w.cell_of, w.local_off, w.cell_start);
  GTB_LAUNCHED();
  int rc = exclusive_scan_inplace(w.cell_start, ncell + 1, w.scan_sums, st);
  if (rc != GTB_OK) return rc;
  fill_kernel<<<blocks, kThreads, 0, st>>>(pos, n, w.cell_of, w.local_off, w.cell_start, w.rec);
  GTB_LAUNCHED();
  return GTB_OK;
}

}  // namespace
}  // namespace gtb

using namespace gtb;

extern "C" size_t gtb_build_workspace_bytes(int64_t n) {
  if (n < 0) return 0;
  return carve_build(nullptr, n).bytes;
}

extern "C" int gtb_neighbor_width(const double* pos, int64_t n, const double box[3],
                                  const int32_t pbc[3], double cutoff, int32_t* counts, void* ws,
                                  size_t ws_bytes, void* stream, int32_t* width_out) {
  int rc = check_geometry(pos, n, box, pbc, cutoff);
  if (rc != GTB_OK) return rc;
  if (!width_out) return GTB_ERR_INVALID_ARG;
  *width_out = 0;
  if (n == 0) return GTB_OK;
  rc = check_ws(ws, ws_bytes, gtb_build_workspace_bytes(n));
  if (rc != GTB_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const BuildWs w = carve_build(ws, n);
  CellGrid g;
  rc = make_cells(pos, n, box, pbc, cutoff, w, st, &g);
  if (rc != GTB_OK) return rc;
  ModelParams m{};
  const unsigned blocks = (unsigned)((n + kThreads - 1) / kThreads);
  neighbor_kernel<true><<<blocks, kThreads, 0, st>>>(pos, nullptr, n, g, cutoff * cutoff,
                                                      w.cell_start, w.rec, m, 0, nullptr, nullptr,
                                                      nullptr, counts, w.flags);
  GTB_LAUNCHED();
  int32_t flags[2] = {0, 0};
  GTB_CUDA_TRY(cudaMemcpyAsync(flags, w.flags, sizeof(flags), cudaMemcpyDeviceToHost, st));
  GTB_CUDA_TRY(cudaStreamSynchronize(st));
  *width_out = flags[0];
  return GTB_OK;
}

extern "C" int gtb_build_hamiltonian(const double* pos, const int32_t* species, int64_t n,
                                     const double box[3], const int32_t pbc[3], double cutoff,
                                     const gtb_hopping_model* model, gtb_ell* H, void* ws,
                                     size_t ws_bytes, void* stream, int32_t* width_needed) {
  int rc = check_geometry(pos, n, box, pbc, cutoff);
  if (rc != GTB_OK) return rc;
  if (!species || !model || !H || H->n != n || H->width < 0 || H->width > GTB_MAX_WIDTH ||
      model->n_species <= 0 || model->n_species > GTB_MAX_SPECIES || !model->onsite || !model->t0)
    return GTB_ERR_INVALID_ARG;
  if (H->width > 0 && (!H->cols || !H->vals)) return GTB_ERR_INVALID_ARG;
  if (model->beta != 0.0 && !(model->r0 > 0.0)) return GTB_ERR_INVALID_ARG;
  if (width_needed) *width_needed = 0;
  if (n == 0) return GTB_OK;
  rc = check_ws(ws, ws_bytes, gtb_build_workspace_bytes(n));
  if (rc != GTB_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const BuildWs w = carve_build(ws, n);
  CellGrid g;
  rc = make_cells(pos, n, box, pbc, cutoff, w, st, &g);
  if (rc != GTB_OK) return rc;
  ModelParams m{};
  m.n_species = model->n_species;
  for (int s = 0; s < m.n_species; ++s) m.onsite[s] = model->onsite[s];
  for (int s = 0; s < m.n_species * m.n_species; ++s) m.t0[s] = model->t0[s];
  m.r0 = model->r0;
  m.beta = model->beta;
  m.onsite_shift = model->onsite_shift;
  const unsigned blocks = (unsigned)((n + kThreads - 1) / kThreads);
  neighbor_kernel<false><<<blocks, kThreads, 0, st>>>(pos, species, n, g, cutoff * cutoff,
                                                       w.cell_start, w.rec, m, H->width, H->cols,
                                                       H->vals, H->diag, nullptr, w.flags);
  GTB_LAUNCHED();
  int32_t flags[2] = {0, 0};
  GTB_CUDA_TRY(cudaMemcpyAsync(flags, w.flags, sizeof(flags), cudaMemcpyDeviceToHost, st));
  GTB_CUDA_TRY(cudaStreamSynchronize(st));
  if (width_needed) *width_needed = flags[0];
  if (flags[1]) return GTB_ERR_INVALID_ARG;  // a species index outside [0, n_species)
  if (flags[0] > H->width) return GTB_ERR_ELL_OVERFLOW;
  return GTB_OK;
}

extern "C" size_t gtb_bounds_workspace_bytes(int64_t n) {
  (void)n;
  return align_up((size_t)kPartialBlocks * 2 * sizeof(double));
}

extern "C" int gtb_spectral_bounds(const gtb_ell* H, double* lo_hi, void* ws, size_t ws_bytes,
                                   void* stream) {
  if (!H || !lo_hi || H->n <= 0 || H->width < 0 || (H->width > 0 && !H->vals))
    return GTB_ERR_INVALID_ARG;
  int rc = check_ws(ws, ws_bytes, gtb_bounds_workspace_bytes(H->n));
  if (rc != GTB_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int blocks = (int)std::min<int64_t>(kPartialBlocks, (H->n + kThreads - 1) / kThreads);
  double* partial = static_cast<double*>(ws);
  gershgorin_partial_kernel<<<blocks, kThreads, 0, st>>>(H->width, H->n, H->vals, H->diag, partial);
  GTB_LAUNCHED();
  gershgorin_final_kernel<<<1, 32, 0, st>>>(partial, blocks, lo_hi);
  GTB_LAUNCHED();
  return GTB_OK;
}
