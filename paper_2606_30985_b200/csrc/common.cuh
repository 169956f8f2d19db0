// common.cuh - shared declarations of the pepo_b200 CUDA sources (product path only; the
// CPU oracle under oracle/ shares nothing with these files).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

namespace pepo {

#define PEPO_MAX_RANK 8

// ---- error plumbing (host) ---------------------------------------------------------------
void set_error(const char* fmt, ...);
#define PEPO_CUDA_OK(expr)                                                          \
  do {                                                                              \
    cudaError_t _e = (expr);                                                        \
    if (_e != cudaSuccess) {                                                        \
      pepo::set_error("CUDA error %s at %s:%d", cudaGetErrorString(_e), __FILE__,   \
                      __LINE__);                                                    \
      return -3;                                                                    \
    }                                                                               \
  } while (0)

// Kernel-launch counter of the context the calling thread is working for (every extern "C" entry
// that takes a pepo_ctx points it at that context's counter; the kernel-level entry points count
// into a per-thread scratch counter).  No process-global mutable state: two contexts on two host
// threads do not interfere.
extern thread_local long long* t_launch_counter;
#define PEPO_COUNT_LAUNCH() (++*pepo::t_launch_counter)

// One-time per-device setup (cudaFuncSetAttribute): flags[dev] is set on first use on that device.
#define PEPO_MAX_DEVICES 64
inline bool first_use_on_device(char* flags) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= PEPO_MAX_DEVICES) return true;
  if (flags[dev]) return false;
  flags[dev] = 1;
  return true;
}

// ---- fast division by a runtime constant (index arithmetic of the permute kernels) -------
struct FastDiv {
  uint32_t d, mul, shift;   // n / d = (umulhi(n, mul) + n) >> shift  (n < 2^31)
};
inline FastDiv make_fastdiv(uint32_t d) {
  FastDiv f; f.d = d;
  if (d == 1) { f.mul = 0; f.shift = 0; return f; }
  uint32_t s = 0;
  while ((1ull << s) < d) ++s;                       // s = ceil(log2 d)
  uint64_t m = ((1ull << 32) * ((1ull << s) - d)) / d + 1;
  f.mul = (uint32_t)m; f.shift = s;
  return f;
}
__device__ __forceinline__ uint32_t fd_div(uint32_t n, const FastDiv& f) {
  return (uint32_t)(((uint64_t)__umulhi(n, f.mul) + n) >> f.shift);
}

// ---- DMMA GEMM ---------------------------------------------------------------------------
// C (M x N, ldc) = op(A) op(B); column-major operands.  transA: 0 -> A is M x K (lda),
// 1 -> A is K x M.  transB: 0 -> B is K x N, 1 -> B is N x K.
struct GemmProb {
  const double* A; const double* B; double* C;
  long long lda, ldb, ldc;
  long long M; int N; int K;
};
// ksplit > 1: CTA (tile, s) handles K range [s*kchunk, (s+1)*kchunk) and writes its partial
// tile to part + s*M*N (packed ld = M); the caller reduces.  upper_only: skip tiles whose
// column-tile index < row-tile index (Gram).  probs_dev != nullptr: batched over grid.z with
// per-problem descriptors in device memory (max_M / max_N size the grid).
int launch_dgemm(cudaStream_t st, int transA, int transB, const GemmProb& p, int ksplit,
                 int kchunk, double* part, bool upper_only);
int launch_dgemm_batched(cudaStream_t st, int transA, int transB, const GemmProb* probs_dev,
                         int batch, long long max_M, int max_N);
// C[i,j] = C[j,i] = sum_s part[s][i + j*n], j >= i (fixed order: deterministic).
int launch_gram_reduce(cudaStream_t st, const double* part, int ksplit, int n, double* C,
                       long long ldc);
void gram_plan(long long m, int n, int* ksplit, int* kchunk);

// ---- permutation -------------------------------------------------------------------------
// dst[sum_j o_j * dst_stride[j]] = src[sum_d i_d * src_stride[d]] * prod_d scale_d(i_d),
// o_j = i_perm[j].  Strides in elements.  scale[d] device pointers (may be null); the factor
// is pow(scale, power) with power in {1, 0.5, -0.5}.
struct PermuteDesc {
  int rank;
  int shape[PEPO_MAX_RANK];          // input dims (first fastest)
  int perm[PEPO_MAX_RANK];
  long long src_stride[PEPO_MAX_RANK];
  long long dst_stride[PEPO_MAX_RANK];   // stride of OUTPUT dim j
  const double* scale[PEPO_MAX_RANK];    // per INPUT dim
  double power;
};
int launch_permute(cudaStream_t st, const double* src, double* dst, const PermuteDesc& d);

}  // namespace pepo
