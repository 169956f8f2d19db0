// normbp.cu - small kernels of the norm-network belief propagation with chi x chi matrix messages
// ("approximate Vidal gauge maintained by BP", L146-L150 message storage,
// L315-L317 PSEUDO_SQRT, L318 / L336 absorb / de-absorb as chi x chi GEMMs, Table 1 L373-L380 Bethe norm).
// The heavy contractions (a site tensor times a matrix on one leg; the cross Gram of two site tensors)
// run on the DMMA GEMM kernels of gemm.cu through launch_site_apply / launch_site_gram; this file holds
// what is left: building I_4 (x) M, folding the Pauli trace of a Gram matrix into a message, the
// Frobenius scalar products and the PSEUDO_SQRT assembly from a Jacobi eigen-decomposition.
#include "normbp.cuh"

namespace pepo {
namespace {

__device__ __forceinline__ double nb_warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ double nb_block_sum(double v, double* sred) {      // blockDim.x = 256, fixed order
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  v = nb_warp_sum(v);
  __syncthreads();
  if (lane == 0) sred[warp] = v;
  __syncthreads();
  double s = 0.0;
  for (int w = 0; w < 8; w++) s += sred[w];
  return s;
}

// W[(c + ci p), (c' + co p')] = delta_{p p'} M[c, c']      (M: ci x co, ld ldm; W: 4 ci x 4 co, ld 4 ci)
__global__ void kron_i4_kernel(const double* M, int ci, int co, int ldm, double* W) {
  const long long tot = 16ll * ci * co;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < tot; e += (long long)gridDim.x * blockDim.x) {
    const int row = (int)(e % (4 * ci)), col = (int)(e / (4 * ci));
    const int c = row % ci, p = row / ci, c2 = col % co, p2 = col / co;
    W[e] = (p == p2) ? M[c + (long long)c2 * ldm] : 0.0;
  }
}

// Message update from the cross Gram G (n x n, n = 4 chi) of B = psi x_{u != w} M_u and psi over the legs
// other than w: Mhat[k,k'] = sum_p G[k + chi p, k' + chi p]; symmetrise; raw (optional) keeps the
// unnormalised matrix; new = d old + (1 - d) Mhat / ||Mhat||_F; delta = max |new - old| (eq. (14), (19)).
__global__ void __launch_bounds__(256) norm_msg_kernel(const double* G, int chi, const double* old, double damping,
                                                       double* out, double* raw, unsigned long long* delta_bits,
                                                       int* flag) {
  __shared__ double sred[8];
  extern __shared__ double mh[];                      // chi * chi
  const int n = 4 * chi;
  double nrm2 = 0.0;
  for (int e = threadIdx.x; e < chi * chi; e += blockDim.x) {
    const int k = e % chi, k2 = e / chi;
    double a = 0.0, b = 0.0;
#pragma unroll
    for (int p = 0; p < 4; p++) {
      a += G[(k + chi * p) + (long long)(k2 + chi * p) * n];
      b += G[(k2 + chi * p) + (long long)(k + chi * p) * n];
    }
    const double v = 0.5 * (a + b);
    mh[e] = v;
    if (raw) raw[e] = v;
    nrm2 += v * v;
  }
  nrm2 = nb_block_sum(nrm2, sred);
  const double nrm = sqrt(nrm2);
  if (!(nrm > 0.0) || !isfinite(nrm)) {
    for (int e = threadIdx.x; e < chi * chi; e += blockDim.x) out[e] = old[e];
    if (threadIdx.x == 0) { atomicOr(flag, isfinite(nrm) ? 1 : 2); if (!isfinite(nrm)) atomicMax(delta_bits, 0x7ff0000000000000ull); }
    return;
  }
  double dmax = 0.0;
  for (int e = threadIdx.x; e < chi * chi; e += blockDim.x) {
    const double o = old[e];
    const double mn = damping * o + (1.0 - damping) * (mh[e] / nrm);
    out[e] = mn;
    const double ch = fabs(mn - o);
    dmax = (ch == ch) ? fmax(dmax, ch) : INFINITY;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) dmax = fmax(dmax, __shfl_xor_sync(0xffffffffu, dmax, o));
  if ((threadIdx.x & 31) == 0) atomicMax(delta_bits, (unsigned long long)__double_as_longlong(dmax));
}

// out[0] = sum_e A[e] B[e]
__global__ void __launch_bounds__(256) frob_dot_kernel(const double* A, const double* B, int n, double* out) {
  __shared__ double sred[8];
  double s = 0.0;
  for (int e = threadIdx.x; e < n; e += blockDim.x) s += A[e] * B[e];
  s = nb_block_sum(s, sred);
  if (threadIdx.x == 0) out[0] = s;
}

// PSEUDO_SQRT from M = U diag(s) V^T (symmetric PSD: U = V up to rounding): S = U sqrt(s) V^T and
// Sinv = U s^-1/2 V^T over the eigenvalues s_k > eps s_0 (s sorted descending).
__global__ void psqrt_build_kernel(const double* U, const double* V, const double* s, int chi, double eps,
                                   double* S, double* Sinv) {
  const double cut = eps * s[0];
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < chi * chi; e += gridDim.x * blockDim.x) {
    const int i = e % chi, j = e / chi;
    double a = 0.0, b = 0.0;
    for (int k = 0; k < chi; k++) {
      const double sk = s[k];
      if (!(sk > cut) || !(sk > 0.0)) break;
      const double r = sqrt(sk), uv = U[i + (long long)k * chi] * V[j + (long long)k * chi];
      a += uv * r; b += uv / r;
    }
    S[e] = a; Sinv[e] = b;
  }
}

// M = diag(v) (chi x chi); power: 1 -> v, 0.5 -> sqrt(v), -0.5 -> 1/sqrt(v)
__global__ void set_diag_kernel(const double* v, int chi, int mode, double* M) {
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < chi * chi; e += gridDim.x * blockDim.x) {
    const int i = e % chi, j = e / chi;
    double x = 0.0;
    if (i == j) { x = v[i]; if (mode == 1) x = sqrt(x); else if (mode == 2) x = 1.0 / sqrt(x); }
    M[e] = x;
  }
}

}  // namespace

int launch_kron_i4(cudaStream_t st, const double* M, int ci, int co, int ldm, double* W) {
  const long long tot = 16ll * ci * co;
  const int g = (int)std::min<long long>((tot + 255) / 256, 148 * 8);
  kron_i4_kernel<<<g, 256, 0, st>>>(M, ci, co, ldm, W);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}
int launch_norm_msg(cudaStream_t st, const double* G, int chi, const double* old, double damping, double* out,
                    double* raw, unsigned long long* delta_bits, int* flag) {
  const size_t smem = (size_t)chi * chi * sizeof(double);
  static char attr[PEPO_MAX_DEVICES] = {0};
  if (first_use_on_device(attr))
    PEPO_CUDA_OK(cudaFuncSetAttribute(norm_msg_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
  if (smem > (size_t)200 * 1024) { set_error("norm_bp: chi %d too large for the matrix-message kernels (chi <= 160)", chi); return -1; }
  norm_msg_kernel<<<1, 256, smem, st>>>(G, chi, old, damping, out, raw, delta_bits, flag);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}
int launch_frob_dot(cudaStream_t st, const double* A, const double* B, int n, double* out) {
  frob_dot_kernel<<<1, 256, 0, st>>>(A, B, n, out);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}
int launch_psqrt_build(cudaStream_t st, const double* U, const double* V, const double* s, int chi, double eps,
                       double* S, double* Sinv) {
  const int g = std::min((chi * chi + 255) / 256, 148 * 4);
  psqrt_build_kernel<<<g, 256, 0, st>>>(U, V, s, chi, eps, S, Sinv);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}
int launch_set_diag(cudaStream_t st, const double* v, int chi, int mode, double* M) {
  const int g = std::min((chi * chi + 255) / 256, 148 * 4);
  set_diag_kernel<<<g, 256, 0, st>>>(v, chi, mode, M);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

}  // namespace pepo
