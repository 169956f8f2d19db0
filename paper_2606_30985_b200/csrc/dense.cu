// dense.cu - batched small dense fp64 kernels of Algorithm 1:
//   Cholesky of the (dressed) Gram matrix and its triangular inverse (a5, eq. (10)),
//   Householder QR (a6, L223-L229), gate dressing (a7/a8, L96-L99) and the bridge matrices
//   (a10, L102).  The Jacobi SVD lives in svd.cu.
#include "dense.cuh"
#include <algorithm>
#include <cooperative_groups.h>
namespace cg = cooperative_groups;

namespace pepo {
namespace {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// =============================== Cholesky =====================================================
constexpr int PB = 32;   // block size

struct InfoPtrs { int* p[PEPO_MAXT]; };

// Footprint: 256 threads x 128 registers = half of an SM's register file.  The kernel is latency-bound
// and was 10 % faster alone with 512 threads, but a CTA that needs the whole register file can only
// start on an SM that has drained completely, and in a Trotter step the GEMM CTAs of the other pieces
// keep refilling every SM: measured in the pipelined 4x4 chi = 60 step, POTRF 0.58 ms against 0.40 ms
// alone, and the step 36.2 ms against 34.6 ms with this footprint (128 threads: 35.4).  Any thread count
// gives the same bits (every entry is computed by one thread in a fixed order).
constexpr int POTRF_THREADS = 256;
__global__ void __launch_bounds__(POTRF_THREADS, 2) potrf_upper_kernel(MatBatch b, InfoPtrs info, double tau) {
  extern __shared__ double sm[];
  const int t = blockIdx.x;
  double* A = b.A[t];
  const long long ld = b.ld[t];
  const int n = b.n[t];
  double* D = sm;                 // PB x (PB+1)
  double* Ps = sm + PB * (PB + 1);  // PB x pitch (pitch = n rounded)
  double* dg = Ps + (size_t)PB * max(n, 1);   // original diagonal G_jj = ||column j||^2
  __shared__ int s_fail;
  __shared__ double s_rmin;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) { s_fail = 0; s_rmin = 1e300; }
  for (int j = tid; j < n; j += blockDim.x) dg[j] = A[j + (long long)j * ld];
  __syncthreads();
  for (int jb = 0; jb < n; jb += PB) {
    const int nb = min(PB, n - jb);
    // load diagonal block (upper part)
    for (int e = tid; e < nb * nb; e += blockDim.x) {
      int i = e % nb, j = e / nb;
      D[i * (PB + 1) + j] = (i <= j) ? A[(jb + i) + (long long)(jb + j) * ld] : 0.0;
    }
    __syncthreads();
    // right-looking Cholesky of the nb x nb block with the whole CTA: per column k one pass that
    // scales row k and one rank-1 update of the trailing (i, j) entries (two barriers per column;
    // one warp doing the update row by row was half of the kernel's time)
    for (int k = 0; k < nb; k++) {
      const double piv = D[k * (PB + 1) + k];
      if (!(piv > 0.0) || !isfinite(piv)) {               // uniform: every thread reads the same value
        if (tid == 0 && s_fail == 0) s_fail = jb + k + 1;
        break;
      }
      const double rkk = sqrt(piv);
      // scale-invariant conditioning measure (R9): R_kk / ||column k|| = sine of the angle between
      // column k and the span of the previous columns
      if (tid == 0) s_rmin = fmin(s_rmin, rkk / sqrt(dg[jb + k]));
      __syncthreads();
      if (tid >= k && tid < nb) D[k * (PB + 1) + tid] = (tid == k) ? rkk : D[k * (PB + 1) + tid] / rkk;
      __syncthreads();
      for (int e = tid; e < nb * nb; e += blockDim.x) {
        const int i = e / nb, j = e % nb;
        if (i > k && j >= i) D[i * (PB + 1) + j] -= D[k * (PB + 1) + i] * D[k * (PB + 1) + j];
      }
      __syncthreads();
    }
    __syncthreads();
    if (s_fail) break;
    // write back factored diagonal block
    for (int e = tid; e < nb * nb; e += blockDim.x) {
      int i = e % nb, j = e / nb;
      if (i <= j) A[(jb + i) + (long long)(jb + j) * ld] = D[i * (PB + 1) + j];
    }
    const int rest = n - jb - nb;
    if (rest > 0) {
      const int c0 = jb + nb;
      // panel row: solve R_jj^T P = A[jb:jb+nb, c0:n], one thread per column
      for (int c = tid; c < rest; c += blockDim.x) {
        double x[PB];
#pragma unroll
        for (int i = 0; i < PB; i++) {
          if (i < nb) {
            double v = A[(jb + i) + (long long)(c0 + c) * ld];
#pragma unroll
            for (int l = 0; l < PB; l++)
              if (l < i) v -= D[l * (PB + 1) + i] * x[l];
            x[i] = v / D[i * (PB + 1) + i];
          }
        }
#pragma unroll
        for (int i = 0; i < PB; i++) {
          if (i < nb) {
            A[(jb + i) + (long long)(c0 + c) * ld] = x[i];
            Ps[i * rest + c] = x[i];
          }
        }
      }
      __syncthreads();
      // trailing update of the upper triangle: 4 x 4 register tiles (8 shared loads per 16 FMAs
      // instead of 2 per FMA; the old element-wise loop made the kernel instruction-bound), each
      // entry accumulated over l in ascending order and subtracted once, as before
      const int nt = (rest + 3) >> 2;
      const int ntile = nt * (nt + 1) / 2;
      for (int e = tid; e < ntile; e += blockDim.x) {
        int tj = (int)((sqrt(8.0 * e + 1.0) - 1.0) * 0.5);
        while ((tj + 1) * (tj + 2) / 2 <= e) tj++;
        while (tj * (tj + 1) / 2 > e) tj--;
        const int ti = e - tj * (tj + 1) / 2;
        const int i0 = 4 * ti, j0 = 4 * tj;
        double acc[4][4];
#pragma unroll
        for (int a = 0; a < 4; a++)
#pragma unroll
          for (int bq = 0; bq < 4; bq++) acc[a][bq] = 0.0;
        for (int l = 0; l < nb; l++) {
          const double* row = Ps + (size_t)l * rest;
          double pa[4], pb[4];
#pragma unroll
          for (int a = 0; a < 4; a++) { pa[a] = (i0 + a < rest) ? row[i0 + a] : 0.0; pb[a] = (j0 + a < rest) ? row[j0 + a] : 0.0; }
#pragma unroll
          for (int a = 0; a < 4; a++)
#pragma unroll
            for (int bq = 0; bq < 4; bq++) acc[a][bq] += pa[a] * pb[bq];
        }
#pragma unroll
        for (int bq = 0; bq < 4; bq++) {
          const int j = j0 + bq;
          if (j >= rest) continue;
          double* cj = A + c0 + (long long)(c0 + j) * ld;
#pragma unroll
          for (int a = 0; a < 4; a++) {
            const int i = i0 + a;
            if (i <= j) cj[i] = cj[i] - acc[a][bq];
          }
        }
      }
    }
    __syncthreads();
  }
  if (tid == 0) {
    int inf = s_fail;
    if (inf == 0 && n > 0 && s_rmin < tau) inf = -1;
    *info.p[t] = inf;
  }
}

__global__ void zero_lower_kernel(MatBatch b) {
  const int t = blockIdx.y;
  const int n = b.n[t];
  const long long m = b.m[t];
  double* A = b.A[t];
  const long long ld = b.ld[t];
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < m * n;
       e += (long long)gridDim.x * blockDim.x) {
    long long i = e % m; int j = (int)(e / m);
    if (i > j) A[i + j * ld] = 0.0;
  }
}

// =============================== triangular inverse ===========================================
// one CTA per (block column J, task); X block column kept in shared memory.
__global__ void __launch_bounds__(256) trtri_upper_kernel(MatBatch R, MatBatch X) {
  extern __shared__ double sm[];
  const int t = blockIdx.y;
  const int n = R.n[t];
  const int J = blockIdx.x;
  const int j0 = J * PB;
  if (j0 >= n) return;
  const int nbj = min(PB, n - j0);
  const double* Rm = R.A[t];
  const long long ldr = R.ld[t];
  double* Xm = X.A[t];
  const long long ldx = X.ld[t];
  double* XS = sm;                              // (J+1) blocks of PB x PB (column-major, pitch PB)
  double* Bs = sm + (size_t)(J + 1) * PB * PB;  // PB x PB accumulator
  double* Rd = Bs + PB * PB;                    // PB x (PB+1) diagonal block
  const int tid = threadIdx.x;
  // zero rows below the block column (strictly lower part of Rinv)
  for (long long e = tid; e < (long long)(n - j0) * nbj; e += blockDim.x) {
    int i = (int)(e % (n - j0)), c = (int)(e / (n - j0));
    if (i >= nbj || i > c) Xm[(j0 + i) + (long long)(j0 + c) * ldx] = 0.0;
  }
  for (int I = J; I >= 0; I--) {
    const int i0 = I * PB;
    const int nbi = PB;   // all blocks above the last are full
    const int nbi_eff = (I == J) ? nbj : nbi;
    // B = (I == J) ? Identity : -sum_{K=I+1..J} R_IK X_KJ
    for (int e = tid; e < PB * PB; e += blockDim.x) {
      int i = e % PB, c = e / PB;
      double s = 0.0;
      if (I == J) {
        s = (i == c && i < nbj) ? 1.0 : 0.0;
      } else if (c < nbj) {
        for (int K = I + 1; K <= J; K++) {
          const int k0 = K * PB;
          const int nbk = (K == J) ? nbj : PB;
          const double* xs = XS + (size_t)K * PB * PB + c * PB;
          for (int l = 0; l < nbk; l++) s -= Rm[(i0 + i) + (long long)(k0 + l) * ldr] * xs[l];
        }
      }
      Bs[i + c * PB] = s;
    }
    for (int e = tid; e < PB * PB; e += blockDim.x) {
      int i = e % PB, c = e / PB;
      Rd[i * (PB + 1) + c] = (i < nbi_eff && c < nbi_eff && i <= c)
                                 ? Rm[(i0 + i) + (long long)(i0 + c) * ldr] : (i == c ? 1.0 : 0.0);
    }
    __syncthreads();
    // back substitution R_II X_IJ = B, one thread per column c
    if (tid < nbj) {
      const int c = tid;
      double x[PB];
#pragma unroll
      for (int ii = PB - 1; ii >= 0; ii--) {
        double v = Bs[ii + c * PB];
#pragma unroll
        for (int l = PB - 1; l >= 0; l--)
          if (l > ii) v -= Rd[ii * (PB + 1) + l] * x[l];
        x[ii] = v / Rd[ii * (PB + 1) + ii];
      }
#pragma unroll
      for (int ii = 0; ii < PB; ii++) {
        XS[(size_t)I * PB * PB + c * PB + ii] = x[ii];
        if (ii < nbi_eff) Xm[(i0 + ii) + (long long)(j0 + c) * ldx] = x[ii];
      }
    }
    __syncthreads();
  }
}

// =============================== Householder ==================================================
// Reflector j of A (raw column kept): x = A[j:m, j]; beta = -sign(x_0)||x||; v = x - beta e_0;
// tau = 2/(v^T v) = 1/(||x|| (||x|| + |x_0|)); H y = y - tau v (v^T y).
// A group (warp or block) applies it to one target column y (rows j..m-1).
template <int GROUP>   // 32 = warp, otherwise block size
__device__ __forceinline__ double group_sum(double v, double* red) {
  v = warp_sum(v);
  if (GROUP == 32) return v;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  __syncthreads();
  if (lane == 0) red[warp] = v;
  __syncthreads();
  double s = 0.0;
  for (int w = 0; w < GROUP / 32; w++) s += red[w];
  return s;
}

template <int GROUP> __device__ __forceinline__ void group_sync() {
  if (GROUP == 32) __syncwarp(); else __syncthreads();
}

template <int GROUP>
__device__ void hh_reflect(const double* __restrict__ x, double* __restrict__ y, long long len,
                           int gtid, double* red, double* beta_out, double* tau_out) {
  // pass 1: ||x||^2 and x^T y
  double sxx = 0.0, sxy = 0.0;
  for (long long i = gtid; i < len; i += GROUP) {
    double xi = x[i];
    sxx += xi * xi;
    if (y) sxy += xi * y[i];
  }
  sxx = group_sum<GROUP>(sxx, red);
  if (y) sxy = group_sum<GROUP>(sxy, red);
  const double x0 = x[0];
  const double nrm = sqrt(sxx);
  double beta = (x0 >= 0.0) ? -nrm : nrm;
  double tau = 0.0;
  // tau = 2 / v^T v overflows for ||x|| < ~1e-154 (underflow-level columns occur at the light-cone
  // front, where entries are products of rounding noise): such a column is numerically zero, its
  // reflector is the identity and R_jj = x_0
  if (sxx > 1e-290) tau = 1.0 / (nrm * (nrm + fabs(x0)));
  else beta = x0;
  if (beta_out && gtid == 0) { *beta_out = beta; *tau_out = tau; }
  if (!y || tau == 0.0) return;
  const double y0 = y[0];
  const double w = tau * (sxy - beta * y0);     // tau * v^T y
  group_sync<GROUP>();
  for (long long i = gtid; i < len; i += GROUP) {
    double vi = x[i] - (i == 0 ? beta : 0.0);
    y[i] -= w * vi;
  }
}

// apply a stored reflector (beta, tau known) to y
template <int GROUP>
__device__ void hh_apply_stored(const double* __restrict__ x, double beta, double tau,
                                double* __restrict__ y, long long len, int gtid, double* red) {
  if (tau == 0.0) return;
  double sxy = 0.0;
  for (long long i = gtid; i < len; i += GROUP) sxy += x[i] * y[i];
  sxy = group_sum<GROUP>(sxy, red);
  const double w = tau * (sxy - beta * y[0]);
  group_sync<GROUP>();
  for (long long i = gtid; i < len; i += GROUP) {
    double vi = x[i] - (i == 0 ? beta : 0.0);
    y[i] -= w * vi;
  }
}

// single CTA per task: whole factorisation, column per warp
// hh_reflect<32> for the cluster kernel below: same arithmetic in the same order (bit-identical
// results), every load through L2 (__ldcg): the column a warp reads may have been written by a
// warp of another CTA of the cluster one step earlier, and L1 is not coherent between SMs.
__device__ void hh_reflect_cg(const double* x, double* y, long long len, int lane,
                              double* beta_out, double* tau_out) {
  double sxx = 0.0, sxy = 0.0;
  for (long long i = lane; i < len; i += 32) {
    double xi = __ldcg(x + i);
    sxx += xi * xi;
    if (y) sxy += xi * __ldcg(y + i);
  }
  sxx = warp_sum(sxx);
  if (y) sxy = warp_sum(sxy);
  const double x0 = __ldcg(x);
  const double nrm = sqrt(sxx);
  double beta = (x0 >= 0.0) ? -nrm : nrm;
  double tau = 0.0;
  if (sxx > 1e-290) tau = 1.0 / (nrm * (nrm + fabs(x0)));
  else beta = x0;
  if (beta_out && lane == 0) { *beta_out = beta; *tau_out = tau; }
  if (!y || tau == 0.0) return;
  const double y0 = __ldcg(y);
  const double w = tau * (sxy - beta * y0);
  __syncwarp();
  for (long long i = lane; i < len; i += 32) {
    double vi = __ldcg(x + i) - (i == 0 ? beta : 0.0);
    y[i] = __ldcg(y + i) - w * vi;
  }
}

// The small factorisation spread over a thread-block cluster: the warps of all CS CTAs take the
// columns c > j of step j (column per warp, as in the single-CTA kernel), a cluster barrier ends
// the step.  The matrix stays in global memory (<= 2 MB: L2-resident).  Growth phase of a run:
// the single-CTA kernel took up to 16 ms for a 1090 x 240 matrix (one SM, 240 dependent steps of
// 15 column updates per warp).
__global__ void __launch_bounds__(512) hh_factor_small_cluster_kernel(HHBatch b, int small_limit_log2, int CS) {
  cg::cluster_group cluster = cg::this_cluster();
  const int crank = (int)cluster.block_rank();
  const int t = blockIdx.x / CS;
  const long long m = b.m[t];
  const int n = b.n[t];
  if (m * (long long)n > (1ll << small_limit_log2)) return;      // uniform over the cluster
  double* A = b.A[t];
  const long long lda = b.lda[t];
  const int k = (int)min((long long)n, m);
  const int lane = threadIdx.x & 31, nw = blockDim.x >> 5;
  const int gw = crank * nw + (threadIdx.x >> 5), gnw = CS * nw;
  for (int j = 0; j < k; j++) {
    const double* x = A + j + (long long)j * lda;
    const long long len = m - j;
    if (j + 1 >= n) {
      if (gw == 0) hh_reflect_cg(x, nullptr, len, lane, b.beta[t] + j, b.tau[t] + j);
    } else {
      for (int c = j + 1 + gw; c < n; c += gnw)
        hh_reflect_cg(x, A + j + (long long)c * lda, len, lane,
                      (c == j + 1) ? b.beta[t] + j : nullptr, b.tau[t] + j);
    }
    __threadfence();
    cluster.sync();
  }
}

__global__ void __launch_bounds__(512) hh_factor_small_kernel(HHBatch b, int small_limit_log2) {
  const int t = blockIdx.x;
  const long long m = b.m[t];
  const int n = b.n[t];
  if (m * (long long)n > (1ll << small_limit_log2)) return;
  double* A = b.A[t];
  const long long lda = b.lda[t];
  const int k = (int)min((long long)n, m);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  for (int j = 0; j < k; j++) {
    const double* x = A + j + (long long)j * lda;
    const long long len = m - j;
    if (j + 1 >= n) {
      if (warp == 0) hh_reflect<32>(x, nullptr, len, lane, nullptr, b.beta[t] + j, b.tau[t] + j);
    } else {
      for (int c = j + 1 + warp; c < n; c += nw)
        hh_reflect<32>(x, A + j + (long long)c * lda, len, lane, nullptr,
                       (c == j + 1) ? b.beta[t] + j : nullptr, b.tau[t] + j);
    }
    __syncthreads();
  }
}

// multi-launch variant: one block per trailing column, launched once per column j
__global__ void __launch_bounds__(256) hh_factor_step_kernel(HHBatch b, int j, int small_limit_log2) {
  __shared__ double red[8];
  const int t = blockIdx.y;
  const long long m = b.m[t];
  const int n = b.n[t];
  if (m * (long long)n <= (1ll << small_limit_log2)) return;
  const int k = (int)min((long long)n, m);
  if (j >= k) return;
  double* A = b.A[t];
  const long long lda = b.lda[t];
  const double* x = A + j + (long long)j * lda;
  const long long len = m - j;
  if (j + 1 >= n) {
    if (blockIdx.x == 0) hh_reflect<256>(x, nullptr, len, threadIdx.x, red, b.beta[t] + j, b.tau[t] + j);
    return;
  }
  for (int c = j + 1 + blockIdx.x; c < n; c += gridDim.x)
    hh_reflect<256>(x, A + j + (long long)c * lda, len, threadIdx.x, red,
                    (c == j + 1) ? b.beta[t] + j : nullptr, b.tau[t] + j);
}

struct RPtrs { double* p[PEPO_MAXT]; long long ld[PEPO_MAXT]; };

__global__ void hh_extract_r_kernel(HHBatch b, RPtrs R) {
  const int t = blockIdx.y;
  const long long m = b.m[t];
  const int n = b.n[t];
  const int k = (int)min((long long)n, m);
  const double* A = b.A[t];
  const long long lda = b.lda[t];
  double* Ro = R.p[t];
  const long long ldr = R.ld[t];
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < (long long)k * n;
       e += (long long)gridDim.x * blockDim.x) {
    int i = (int)(e % k), j = (int)(e / k);
    double v = 0.0;
    if (i < j) v = A[i + (long long)j * lda];
    else if (i == j) v = b.beta[t][j];
    Ro[i + j * ldr] = v;
  }
}

__global__ void __launch_bounds__(512) hh_apply_small_kernel(HHApplyBatch b, int small_limit_log2) {
  const int t = blockIdx.x;
  const long long m = b.m[t];
  if (m * (long long)max(b.k[t], b.ncols[t]) > (1ll << small_limit_log2)) return;
  const int lane = threadIdx.x & 31, nw = blockDim.x >> 5;
  // columns are independent: each warp (of the gridDim.y CTAs of a task) runs all reflectors over its own columns
  for (int c = blockIdx.y * nw + (threadIdx.x >> 5); c < b.ncols[t]; c += gridDim.y * nw) {
    double* y = b.Y[t] + (long long)c * b.ldy[t];
    for (int j = b.k[t] - 1; j >= 0; j--) {
      hh_apply_stored<32>(b.A[t] + j + (long long)j * b.lda[t], b.beta[t][j], b.tau[t][j], y + j,
                          m - j, lane, nullptr);
      __syncwarp();
    }
  }
}

__global__ void __launch_bounds__(256) hh_apply_big_kernel(HHApplyBatch b, int small_limit_log2) {
  __shared__ double red[8];
  const int t = blockIdx.y;
  const long long m = b.m[t];
  if (m * (long long)max(b.k[t], b.ncols[t]) <= (1ll << small_limit_log2)) return;
  for (int c = blockIdx.x; c < b.ncols[t]; c += gridDim.x) {
    double* y = b.Y[t] + (long long)c * b.ldy[t];
    for (int j = b.k[t] - 1; j >= 0; j--) {
      hh_apply_stored<256>(b.A[t] + j + (long long)j * b.lda[t], b.beta[t][j], b.tau[t][j], y + j,
                           m - j, threadIdx.x, red);
      __syncthreads();
    }
  }
}

// =============================== gate dressing ================================================
__global__ void dress_gram_kernel(DressBatch b, GateTables g) {
  const int t = blockIdx.y;
  const int chi = b.chi[t], NA = b.NA;
  const int N = NA * chi;
  const double* C = b.in[t];
  const long long ldc = b.ld_in[t];
  double* S = b.out[t];
  const long long lds = b.ld_out[t];
  const double* Gam = g.Gamma[b.site[t]];
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < (long long)N * N;
       e += (long long)gridDim.x * blockDim.x) {
    int row = (int)(e % N), col = (int)(e / N);
    int c = row % chi, a = row / chi, c2 = col % chi, a2 = col / chi;
    const double* G = Gam + (a * NA + a2) * 16;
    double s = 0.0;
#pragma unroll
    for (int p = 0; p < 4; p++)
#pragma unroll
      for (int q = 0; q < 4; q++) s += G[p * 4 + q] * C[(c + chi * p) + (long long)(c2 + chi * q) * ldc];
    S[row + col * lds] = s;
  }
}

__global__ void dress_R_kernel(DressBatch b, GateTables g) {
  const int t = blockIdx.y;
  const int chi = b.chi[t], NA = b.NA, k = b.k[t];
  const int N = NA * chi;
  const double* R = b.in[t];
  const long long ldr = b.ld_in[t];
  double* X = b.out[t];
  const long long ldx = b.ld_out[t];
  const double* Ah = g.Ahat[b.site[t]];
  const long long rows = 4ll * k;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < rows * N;
       e += (long long)gridDim.x * blockDim.x) {
    int row = (int)(e % rows), col = (int)(e / rows);
    int kk = row % k, pp = row / k, c = col % chi, a = col / chi;
    double s = 0.0;
#pragma unroll
    for (int p = 0; p < 4; p++) s += Ah[(a * 4 + pp) * 4 + p] * R[kk + (long long)(c + chi * p) * ldr];
    X[row + col * ldx] = s;
  }
}

__global__ void scale_sigma_kernel(DressBatch b, GateTables g) {
  const int t = blockIdx.y;
  const int chi = b.chi[t], NA = b.NA, k = b.k[t];
  const int N = NA * chi;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < (long long)k * N;
       e += (long long)gridDim.x * blockDim.x) {
    int row = (int)(e % k), col = (int)(e / k);
    b.out[t][row + col * b.ld_out[t]] = b.in[t][row + col * b.ld_in[t]] * g.sigma[col / chi];
  }
}

struct IntPtrs { int* p[PEPO_MAXT]; };
struct LLVals { long long v[PEPO_MAXT]; };

__global__ void build_W_kernel(DressBatch b, GateTables g, IntPtrs chin_p) {
  const int t = blockIdx.y;
  const int chi = b.chi[t], NA = b.NA;
  const int chin = *chin_p.p[t];
  const int n = 4 * chi;
  const double* T = b.in[t];
  const long long ldt = b.ld_in[t];
  double* W = b.out[t];
  const long long ldw = b.ld_out[t];
  const double* Ah = g.Ahat[b.site[t]];
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < (long long)n * 4 * chin;
       e += (long long)gridDim.x * blockDim.x) {
    int row = (int)(e % n), col = (int)(e / n);
    int c = row % chi, p = row / chi, c2 = col % chin, pp = col / chin;
    double s = 0.0;
    for (int a = 0; a < NA; a++) s += Ah[(a * 4 + pp) * 4 + p] * T[(c + chi * a) + (long long)c2 * ldt];
    W[row + col * ldw] = s;
  }
}

__global__ void reshuffle_M_kernel(DressBatch b, IntPtrs chin_p, LLVals mrows) {
  const int t = blockIdx.y;
  const int k = b.k[t];
  const int chin = *chin_p.p[t];
  const long long m = mrows.v[t];
  const double* Mx = b.in[t];
  const long long ldm = b.ld_in[t];
  double* Mp = b.out[t];
  const long long ldo = b.ld_out[t];
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < m * 4 * chin;
       e += (long long)gridDim.x * blockDim.x) {
    long long row = e % m; int col = (int)(e / m);
    int c2 = col % chin, pp = col / chin;
    double v = 0.0;
    if (row < k) v = Mx[(row + (long long)k * pp) + (long long)c2 * ldm];
    Mp[row + col * ldo] = v;
  }
}

__global__ void copy_pad_kernel(MatBatch src, HHApplyBatch dst) {
  const int t = blockIdx.y;
  const long long m = dst.m[t];
  const int nc = dst.ncols[t];
  const long long r = src.m[t];
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < m * nc;
       e += (long long)gridDim.x * blockDim.x) {
    long long i = e % m; int j = (int)(e / m);
    dst.Y[t][i + j * dst.ldy[t]] = (i < r) ? src.A[t][i + j * src.ld[t]] : 0.0;
  }
}

constexpr int SMALL_LOG2 = 18;   // <= 256K elements: single-CTA Householder

inline unsigned grid1d(long long work, int bs, unsigned cap = 148 * 8) {
  long long g = (work + bs - 1) / bs;
  if (g < 1) g = 1;
  if (g > cap) g = cap;
  return (unsigned)g;
}

}  // namespace

int launch_potrf(cudaStream_t st, const MatBatch& b, int* const* info, double tau) {
  if (b.count == 0) return 0;
  InfoPtrs ip;
  int nmax = 0;
  for (int t = 0; t < b.count; t++) { ip.p[t] = info[t]; nmax = std::max(nmax, b.n[t]); }
  size_t smem = (size_t)(PB * (PB + 1) + (PB + 1) * std::max(nmax, 1)) * sizeof(double);
  // largest shared-memory size the kernel may ask for (chi_max <= 256: n <= 1024), set once per device
  static char attr[PEPO_MAX_DEVICES] = {0};
  if (first_use_on_device(attr))
    PEPO_CUDA_OK(cudaFuncSetAttribute(potrf_upper_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
  if (smem > (size_t)200 * 1024) { set_error("potrf: matrix of order %d too large", nmax); return -1; }
  potrf_upper_kernel<<<b.count, POTRF_THREADS, smem, st>>>(b, ip, tau);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

int launch_zero_lower(cudaStream_t st, const MatBatch& R) {
  if (R.count == 0) return 0;
  long long w = 0;
  for (int t = 0; t < R.count; t++) w = std::max(w, R.m[t] * R.n[t]);
  dim3 grid(grid1d(w, 256), R.count);
  zero_lower_kernel<<<grid, 256, 0, st>>>(R);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

int launch_trtri(cudaStream_t st, const MatBatch& R, const MatBatch& Rinv) {
  if (R.count == 0) return 0;
  int nmax = 0;
  for (int t = 0; t < R.count; t++) nmax = std::max(nmax, R.n[t]);
  int nblk = (nmax + PB - 1) / PB;
  size_t smem = ((size_t)(nblk + 1) * PB * PB + PB * (PB + 1)) * sizeof(double);
  static char attr[PEPO_MAX_DEVICES] = {0};
  if (first_use_on_device(attr))
    PEPO_CUDA_OK(cudaFuncSetAttribute(trtri_upper_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
  if (smem > (size_t)200 * 1024) { set_error("trtri: matrix of order %d too large", nmax); return -1; }
  dim3 grid(nblk, R.count);
  trtri_upper_kernel<<<grid, 256, smem, st>>>(R, Rinv);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

int launch_hh_factor(cudaStream_t st, const HHBatch& b) {
  if (b.count == 0) return 0;
  bool any_small = false; int kbig = 0, nbig = 0;
  for (int t = 0; t < b.count; t++) {
    if (b.m[t] * (long long)b.n[t] <= (1ll << SMALL_LOG2)) any_small = true;
    else {
      kbig = std::max(kbig, (int)std::min((long long)b.n[t], b.m[t]));
      nbig = std::max(nbig, b.n[t]);
    }
  }
  if (any_small) {
    // matrices of more than a few columns: the cluster form (8 CTAs share the columns of a step)
    int nsmall = 0; long long wsmall = 0;
    for (int t = 0; t < b.count; t++)
      if (b.m[t] * (long long)b.n[t] <= (1ll << SMALL_LOG2)) { nsmall = std::max(nsmall, b.n[t]); wsmall = std::max(wsmall, b.m[t] * (long long)b.n[t]); }
    bool done = false;
    if (nsmall > 32 && wsmall > 4096) {
      const int CS = 8;
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3((unsigned)(b.count * CS));
      cfg.blockDim = dim3(512);
      cfg.dynamicSmemBytes = 0;
      cfg.stream = st;
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeClusterDimension;
      at[0].val.clusterDim.x = CS; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
      cfg.attrs = at; cfg.numAttrs = 1;
      cudaError_t e = cudaLaunchKernelEx(&cfg, hh_factor_small_cluster_kernel, b, (int)SMALL_LOG2, CS);
      if (e == cudaSuccess) done = true; else (void)cudaGetLastError();
    }
    if (!done) hh_factor_small_kernel<<<b.count, 512, 0, st>>>(b, SMALL_LOG2);
    PEPO_COUNT_LAUNCH();
  }
  for (int j = 0; j < kbig; j++) {
    dim3 grid(std::max(1, std::min(nbig - j - 1, 1024)), b.count);
    hh_factor_step_kernel<<<grid, 256, 0, st>>>(b, j, SMALL_LOG2);
    PEPO_COUNT_LAUNCH();
  }
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

int launch_hh_extract_r(cudaStream_t st, const HHBatch& b, double* const* Rout, const long long* ldr) {
  if (b.count == 0) return 0;
  RPtrs R;
  long long w = 0;
  for (int t = 0; t < b.count; t++) {
    R.p[t] = Rout[t]; R.ld[t] = ldr[t];
    w = std::max(w, std::min((long long)b.n[t], b.m[t]) * b.n[t]);
  }
  dim3 grid(grid1d(w, 256), b.count);
  hh_extract_r_kernel<<<grid, 256, 0, st>>>(b, R);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

int launch_hh_apply_q(cudaStream_t st, const HHApplyBatch& b) {
  if (b.count == 0) return 0;
  bool any_small = false, any_big = false; int cbig = 0;
  for (int t = 0; t < b.count; t++) {
    if (b.m[t] * (long long)std::max(b.k[t], b.ncols[t]) <= (1ll << SMALL_LOG2)) any_small = true;
    else { any_big = true; cbig = std::max(cbig, b.ncols[t]); }
  }
  if (any_small) {
    int csmall = 1;
    for (int t = 0; t < b.count; t++)
      if (b.m[t] * (long long)std::max(b.k[t], b.ncols[t]) <= (1ll << SMALL_LOG2)) csmall = std::max(csmall, b.ncols[t]);
    hh_apply_small_kernel<<<dim3(b.count, std::min((csmall + 15) / 16, 16)), 512, 0, st>>>(b, SMALL_LOG2);
    PEPO_COUNT_LAUNCH();
  }
  if (any_big) {
    dim3 grid(std::max(1, std::min(cbig, 2048)), b.count);
    hh_apply_big_kernel<<<grid, 256, 0, st>>>(b, SMALL_LOG2);
    PEPO_COUNT_LAUNCH();
  }
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

int launch_copy_pad(cudaStream_t st, const MatBatch& src, const HHApplyBatch& dst) {
  if (dst.count == 0) return 0;
  long long w = 0;
  for (int t = 0; t < dst.count; t++) w = std::max(w, dst.m[t] * dst.ncols[t]);
  dim3 grid(grid1d(w, 256), dst.count);
  copy_pad_kernel<<<grid, 256, 0, st>>>(src, dst);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

int launch_dress_gram(cudaStream_t st, const DressBatch& b, const GateTables& g) {
  if (b.count == 0) return 0;
  long long w = 0;
  for (int t = 0; t < b.count; t++) { long long N = (long long)b.NA * b.chi[t]; w = std::max(w, N * N); }
  dim3 grid(grid1d(w, 256), b.count);
  dress_gram_kernel<<<grid, 256, 0, st>>>(b, g);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}
int launch_dress_R(cudaStream_t st, const DressBatch& b, const GateTables& g) {
  if (b.count == 0) return 0;
  long long w = 0;
  for (int t = 0; t < b.count; t++) w = std::max(w, 4ll * b.k[t] * b.NA * b.chi[t]);
  dim3 grid(grid1d(w, 256), b.count);
  dress_R_kernel<<<grid, 256, 0, st>>>(b, g);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}
int launch_scale_sigma(cudaStream_t st, const DressBatch& b, const GateTables& g) {
  if (b.count == 0) return 0;
  long long w = 0;
  for (int t = 0; t < b.count; t++) w = std::max(w, (long long)b.k[t] * b.NA * b.chi[t]);
  dim3 grid(grid1d(w, 256), b.count);
  scale_sigma_kernel<<<grid, 256, 0, st>>>(b, g);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}
int launch_build_W(cudaStream_t st, const DressBatch& b, const GateTables& g, int* const* chi_new) {
  if (b.count == 0) return 0;
  IntPtrs ip;
  long long w = 0;
  for (int t = 0; t < b.count; t++) { ip.p[t] = chi_new[t]; w = std::max(w, 16ll * b.chi[t] * b.k[t]); }
  dim3 grid(grid1d(w, 256), b.count);
  build_W_kernel<<<grid, 256, 0, st>>>(b, g, ip);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}
int launch_reshuffle_M(cudaStream_t st, const DressBatch& b, int* const* chi_new, const long long* mrows) {
  if (b.count == 0) return 0;
  IntPtrs ip; LLVals mv;
  long long w = 0;
  for (int t = 0; t < b.count; t++) {
    ip.p[t] = chi_new[t]; mv.v[t] = mrows[t];
    w = std::max(w, mrows[t] * 4 * b.chi[t]);   // chi[t] carries the chi_new cap here
  }
  dim3 grid(grid1d(w, 256, 148 * 16), b.count);
  reshuffle_M_kernel<<<grid, 256, 0, st>>>(b, ip, mv);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

}  // namespace pepo
