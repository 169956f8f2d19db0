// noalloc.cu - pepo_gram_static: the Gram kernel (eq. (10)) for callers that may not
// allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc).  Same kernels and the same split plan as pepo_gram; the split-K partial sums go to a
// file-scope device array of a fixed size instead of a caller-provided workspace.
//
// The array (PEPO_STATIC_SCRATCH_BYTES = 8 MiB) is part of the library image: every GPU that loads the
// library holds it until the process exits.  All calls on a device share it, so
//   * two calls that overlap on the GPU (different streams, no event between them) RACE on it: keep the
//     calls of one device on one stream or order them with events;
//   * it keeps the previous call's contents.  Nothing in it has to start at zero: every partial entry the
//     reduction reads (upper triangle of each split) is written by the product kernel of the same call
//     first, in stream order, so there is nothing to clear.
// In host code the array's name is only a stand-in for the symbol; the device address is looked up once
// per device with cudaGetSymbolAddress (that device current) and passed to the kernels.
#include "../../include/pepo.h"
#include "common.cuh"

#include <mutex>

namespace pepo {
namespace {

static __device__ __align__(256) unsigned char g_static_scratch[PEPO_STATIC_SCRATCH_BYTES];

std::mutex g_scratch_mu;
double* g_scratch_ptr[PEPO_MAX_DEVICES] = {nullptr};

// device address of the scratch array on the CURRENT device (looked up on the first call per device)
int static_scratch(double** out) {
  int dev = 0;
  PEPO_CUDA_OK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= PEPO_MAX_DEVICES) { set_error("gram_static: device index %d out of range", dev); return -3; }
  std::lock_guard<std::mutex> lock(g_scratch_mu);
  if (!g_scratch_ptr[dev]) {
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess || !p) { set_error("gram_static: cudaGetSymbolAddress failed: %s", cudaGetErrorString(e)); return -3; }
    g_scratch_ptr[dev] = (double*)p;
  }
  *out = g_scratch_ptr[dev];
  return 0;
}

}  // namespace
}  // namespace pepo

using namespace pepo;

extern "C" size_t pepo_static_scratch_bytes(void) { return (size_t)PEPO_STATIC_SCRATCH_BYTES; }

extern "C" int pepo_gram_static(const double* d_A, long long m, int n, long long lda, double* d_C, void* stream) {
  if (!d_A || !d_C || m < 1 || n < 1 || lda < m || m >= (1ll << 31)) { set_error("gram_static: bad argument"); return -1; }
  int ks, kc;
  gram_plan(m, n, &ks, &kc);
  const size_t need = ks > 1 ? (size_t)ks * n * n * 8 : 0;
  if (need > (size_t)PEPO_STATIC_SCRATCH_BYTES) {
    set_error("gram_static: %lld x %d needs %zu bytes of split-K scratch, the built-in array holds %zu "
              "(use pepo_gram with a workspace of pepo_gram_ws_bytes)", m, n, need, (size_t)PEPO_STATIC_SCRATCH_BYTES);
    return -2;
  }
  double* part = nullptr;
  int rc = static_scratch(&part);
  if (rc) return rc;
  GemmProb gp;
  gp.A = d_A; gp.B = d_A; gp.C = d_C; gp.lda = lda; gp.ldb = lda; gp.ldc = n; gp.M = n; gp.N = n; gp.K = (int)m;
  cudaStream_t st = (cudaStream_t)stream;
  rc = launch_dgemm(st, 1, 0, gp, ks, kc, part, true);
  if (rc) return rc;
  return launch_gram_reduce(st, ks > 1 ? (const double*)part : d_C, ks, n, d_C, n);
}
