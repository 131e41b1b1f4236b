// Status strings, CUDA error capture and the launch counter of libgtb_kpm.so.
#include <atomic>
#include <cstdio>

#include "common.cuh"

namespace gtb {

static thread_local char g_cuda_error[512] = "";
static std::atomic<int64_t> g_launches{0};

void note_cuda_error(cudaError_t e, const char* where) {
  std::snprintf(g_cuda_error, sizeof(g_cuda_error), "%s: %s (%s)", where, cudaGetErrorName(e),
                cudaGetErrorString(e));
  cudaGetLastError();  // clear the sticky-less error state so later calls report their own
}

void count_launch(int64_t k) { g_launches.fetch_add(k, std::memory_order_relaxed); }

}  // namespace gtb

extern "C" const char* gtb_status_string(int status) {
  switch (status) {
    case GTB_OK: return "ok";
    case GTB_ERR_INVALID_ARG: return "invalid argument";
    case GTB_ERR_BOX_TOO_SMALL: return "a periodic box length is smaller than twice the cutoff";
    case GTB_ERR_ELL_OVERFLOW: return "a row needs more ELL slots than the width provided";
    case GTB_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
    case GTB_ERR_DIVERGED: return "non-finite Chebyshev moments (spectrum outside [b-a, b+a])";
    case GTB_ERR_CUDA: return "CUDA runtime error";
    case GTB_ERR_INDEX_RANGE: return "too many atoms for int32 indices";
    case GTB_ERR_NOT_PACKABLE: return "matrix does not fit the packed-row format (width, offsets or distinct values)";
    case GTB_ERR_STATIC_LIMIT:
      return "the run needs more scratch than the static array holds (GTB_STATIC_WS_BYTES); use gtb_kpm_moments "
             "with a caller-owned workspace";
    default: return "unknown status";
  }
}

extern "C" const char* gtb_last_cuda_error(void) { return gtb::g_cuda_error; }

extern "C" int gtb_version(void) { return 200; }

extern "C" int64_t gtb_launch_count(void) {
  return gtb::g_launches.load(std::memory_order_relaxed);
}
