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
// ---- gathered operands (permute-on-load GEMMs of the bond gate) -----------------------------
// A site tensor psi[U,D,L,R,P] (column-major) read as the matrix cv[rows = environment legs,
// cols = (cut, P)] WITHOUT materialising the permuted copy (section 4.1 describes the
// explicit permutation; the irreducible traffic of a gate is 2 reads + 1 write of
// psi): every GEMM index maps to an element offset through a two-level function
//     off(i) = s * (i mod E) + T * (i div E)            (E = 0: off(i) = s * i)
// which covers all four cut legs: the row index splits into a contiguous run and a strided
// remainder, the column index into (cut index, Pauli slab).
struct Idx2 {
  FastDiv E; long long s, T;
};
inline Idx2 make_idx2(long long E, long long s, long long T) {
  Idx2 r; r.E = make_fastdiv(E > 0 ? (uint32_t)E : 1u); if (E <= 0) r.E.d = 0; r.s = s; r.T = T; return r;
}
__host__ __device__ __forceinline__ long long idx2_off_host(const Idx2& f, long long i) {
  if (f.E.d == 0) return f.s * i;
  return f.s * (i % f.E.d) + f.T * (i / f.E.d);
}
struct GemmGather {
  Idx2 a_outer, a_k, b_outer, b_k, c_m, c_n;   // element (outer, k) of A at A + a_outer(outer) + a_k(k), etc.
  // row weights (Gram of the environment-weighted matrix, a3 fused): the A fragments are multiplied by
  // w(k) = wv[0][k mod wE0] * wv[1][(k div wE0) mod wE1] * wv[2][k div (wE0 wE1)]; nw = 0: none
  int nw; const double* wv[3]; FastDiv wE[2]; int wlen[3];
  int alignedA, alignedB;                      // 16-byte pairs along the contiguous direction are valid
  int ktabA;                                   // operand A not K-contiguous with a two-level k index: offsets from a per-CTA table
};
int launch_dgemm_gather(cudaStream_t st, int transA, int transB, const GemmProb& p, const GemmGather& g,
                        int ksplit, int kchunk, double* part, bool upper_only);

// A packed site tensor psi[leg_0, .., leg_{nlegs-1}, P] (column-major, P = 4 slowest) viewed as the
// matrix cv[rows = the legs other than `cut` in canonical order, cols = (cut, P)] of Algorithm 1
// (PAPER.md:L267-L269, L318-L319): m = prod of the other dims, n = 4 dims[cut].
struct SiteView {
  int nlegs, cut;
  int dims[4];
  long long m() const { long long r = 1; for (int l = 0; l < nlegs; l++) if (l != cut) r *= dims[l]; return r; }
  int n() const { return 4 * dims[cut]; }
};
// C (n x n, ld n, both triangles) = cv^T diag(w) cv with w(row) = prod over the environment legs of
// w2[leg][i_leg] (a3 fused into a5: w2 = lambda, the squared absorb factor); w2[leg] device pointers
// (entry `cut` ignored; NULL = no weight on that leg).  part: split-K workspace of gram_plan(m, n).
// psiB != nullptr: the cross Gram cv(psi)^T diag(w) cv(psiB) of two tensors of the same shape (norm-network
// BP); it must be symmetric by construction, only its upper triangle is computed and mirrored.
int launch_site_gram(cudaStream_t st, const double* psi, const SiteView& v, const double* const* w2,
                     double* C, double* part, const double* psiB = nullptr);
// out = the packed site tensor with dims[cut] replaced by chi_new: out[.., c', .., p'] =
// sum_{c,p} psi[.., c, .., p] W[(c,p),(c',p')], W column-major (4 dims[cut]) x (4 chi_new), ld ldw
// (a10-a13 fused: reconstruction GEMM that reads and writes the canonical layout).
int launch_site_apply(cudaStream_t st, const double* psi, const SiteView& v, const double* W, long long ldw,
                      int chi_new, double* out);

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
// largest split count gram_plan returns for any row count <= m (sizing of a shared split-K workspace)
int gram_max_splits(long long m, int n);
// register-only DMMA loop (fp64 tensor-pipe yardstick of bench.py); *flops = flops of the launch
int launch_dmma_peak(cudaStream_t st, int iters, int ctas_per_sm, double* sink, double* flops);

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
