// dense.cuh - batched small dense kernels of the bond update (Cholesky, triangular inverse,
// Householder QR, one-sided Jacobi SVD, gate dressing).  Batches are passed BY VALUE (no
// descriptor upload): at most PEPO_MAXT problems per launch.
#pragma once
#include "common.cuh"

namespace pepo {

#define PEPO_MAXT 32

struct MatBatch {             // generic batch of column-major matrices
  int count;
  double* A[PEPO_MAXT];
  long long ld[PEPO_MAXT];
  long long m[PEPO_MAXT];
  int n[PEPO_MAXT];
};

// ---- Cholesky (upper, in place): C = R^T R.  info[t] = 0 ok / j+1 = pivot j <= 0 or NaN;
// if ok and min diag < tau*max diag -> info = -1 (ill-conditioned, R still valid). ----------
int launch_potrf(cudaStream_t st, const MatBatch& b, int* const* info, double tau);
// Rinv = R^{-1} for upper-triangular R (n x n); strictly-lower part of Rinv zeroed.
int launch_trtri(cudaStream_t st, const MatBatch& R, const MatBatch& Rinv);
// zero the strictly lower triangle
int launch_zero_lower(cudaStream_t st, const MatBatch& R);

// ---- Householder QR (in place, raw columns kept; beta = R_jj, tau = 2/(v^T v), v = x - beta e_j)
struct HHBatch {
  int count;
  double* A[PEPO_MAXT]; long long lda[PEPO_MAXT]; long long m[PEPO_MAXT]; int n[PEPO_MAXT];
  double* beta[PEPO_MAXT]; double* tau[PEPO_MAXT];
};
int launch_hh_factor(cudaStream_t st, const HHBatch& b);
// extract R (k x n, k = min(m,n)) from the factored A into Rout (ld = ldr), zero below diag
int launch_hh_extract_r(cudaStream_t st, const HHBatch& b, double* const* Rout, const long long* ldr);
// Y <- Q Y for Y (m x ncols, ldy) using reflectors k-1..0
struct HHApplyBatch {
  int count;
  const double* A[PEPO_MAXT]; long long lda[PEPO_MAXT]; long long m[PEPO_MAXT]; int k[PEPO_MAXT];
  const double* beta[PEPO_MAXT]; const double* tau[PEPO_MAXT];
  double* Y[PEPO_MAXT]; long long ldy[PEPO_MAXT]; int ncols[PEPO_MAXT];
};
int launch_hh_apply_q(cudaStream_t st, const HHApplyBatch& b);
// Y[t] (m x ncols) <- [src[t] (rows src.m x ncols) ; 0]
int launch_copy_pad(cudaStream_t st, const MatBatch& src, const HHApplyBatch& dst);

// ---- one-sided Jacobi SVD --------------------------------------------------------------------
// K (r1 x r2, ldk).  Work: G (max(r1,r2) x min(r1,r2)) and V (min x min), caller-provided.
// Outputs after launch_svd_finish: s sorted descending in sv[0..r), order[] permutation,
// Us (r1 x chi_new) = U sqrt(s), Vs (r2 x chi_new) = V sqrt(s), chi_new, lambda, stats.
struct SvdBatch {
  int count;
  const double* K[PEPO_MAXT]; int ldk[PEPO_MAXT]; int r1[PEPO_MAXT]; int r2[PEPO_MAXT];
  double* G[PEPO_MAXT]; double* V[PEPO_MAXT];       // G: M x Nc (ld M), V: Nc x Nc (ld Nc)
  double* sv[PEPO_MAXT];                            // Nc singular values (sorted, descending)
  int* order[PEPO_MAXT];                            // Nc ints scratch
  int* sweeps[PEPO_MAXT];                           // device int
  // device int or nullptr, OUT: 1 = a square core (r1 == r2) was iterated as K^T (see `orient` below)
  int* orient[PEPO_MAXT] = {};
};
// with_v = false: V is not accumulated (launch_svd_bridge then derives it from K, SvdFinishBatch::K)
// precond_min > 0 (only with_v = false): problems with min(r1,r2) >= precond_min are QR-preconditioned
// (the Jacobi iteration runs on R^T); launch_svd_bridge must get the same value.
// early: cosine below which a sweep counts as the last one (jacobi_c16_kernel; 0 = always run the
// confirming sweep)
// keep_hint > 0 and theta > 0 (hot-path kernel only): only the leading keep_hint triplets are needed
// (truncation to chi_max); after 3 full sweeps the columns with norm < theta x the keep_hint-th largest
// norm are set aside and the iteration continues on the rest (svd.cu "deflation")
// orient (hot-path kernel, preconditioned SQUARE cores only; needs SvdBatch::orient): which of K, K^T
// gets the QR preconditioner.  0 = K; 1 = the one whose column norms are more graded (larger variance
// of ln ||col||^2: an unpivoted QR then leaves an L = R^T that is closer to diagonal, 9 Jacobi sweeps
// instead of 19-21 on the far-corner cores of the 4x4 chi 60 step); 2 = K^T.  The choice is a function
// of K alone; launch_svd_bridge reads it back through SvdFinishBatch::orient.
int launch_svd_jacobi(cudaStream_t st, const SvdBatch& b, double tol, int max_sweeps, bool with_v,
                      int precond_min, double early, int keep_hint = 0, double theta = 0.0, int orient = 0);

struct SvdFinishBatch {
  int count;
  int r1[PEPO_MAXT]; int r2[PEPO_MAXT];
  const double* G[PEPO_MAXT]; const double* V[PEPO_MAXT]; const double* sv[PEPO_MAXT];
  const int* order[PEPO_MAXT];
  const int* orient[PEPO_MAXT] = {};                // as written by launch_svd_jacobi (nullptr = 0)
  int with_v;                                       // 1: V accumulated by the Jacobi kernel; 0: derive from K
  int precond_min;                                  // as passed to launch_svd_jacobi (with_v = 0)
  const double* K[PEPO_MAXT]; int ldk[PEPO_MAXT];   // the core (needed when with_v = 0)
  double* Us[PEPO_MAXT]; int ldus[PEPO_MAXT];       // r1 x chi_new
  double* Vs[PEPO_MAXT]; int ldvs[PEPO_MAXT];       // r2 x chi_new
  double* lambda[PEPO_MAXT]; double* sqrt_l[PEPO_MAXT]; double* isqrt_l[PEPO_MAXT];
  int* chi_new[PEPO_MAXT];                          // device int
  double* gate_stats[PEPO_MAXT];                    // [0] discarded weight, [1] relative cut gap
};
// truncation rule eq. (11), Vidal normalisation eq. (12)
int launch_svd_truncate(cudaStream_t st, const SvdFinishBatch& b, int chi_max, double eps_cut);
int launch_svd_bridge(cudaStream_t st, const SvdFinishBatch& b, int chi_cap);
// plain singular vectors of an m x n problem solved by launch_svd_jacobi: U (m x r, ld m),
// Vout (n x r, ld n), r = min(m,n); columns of zero singular values are zero in the tall factor
int launch_svd_vectors(cudaStream_t st, const double* G, const double* V, const double* s,
                       const int* order, int m, int n, double* U, double* Vout);
// Q (m x k, ld m) <- [I_k ; 0]
int launch_set_identity(cudaStream_t st, double* Q, long long m, int k);

// ---- gate dressing ---------------------------------------------------------------------------
// S[(a,c),(a',c')] = sum_{p,q} Gamma[((a*NA+a')*4+p)*4+q] C[(c,p),(c',q)]  (index (c,p) = c + chi*p,
// (a,c) = c + chi*a).
struct DressBatch {
  int count; int NA;
  const double* in[PEPO_MAXT]; double* out[PEPO_MAXT];
  int chi[PEPO_MAXT]; int k[PEPO_MAXT];             // k: rows of R (dress_R only)
  int site[PEPO_MAXT];                              // 0 -> first Schmidt factor, 1 -> second
  long long ld_in[PEPO_MAXT]; long long ld_out[PEPO_MAXT];
};
struct GateTables {           // device pointers
  const double* Gamma[2];     // NA*NA*16
  const double* Ahat[2];      // NA*16: Ahat[a][p'][p]
  const double* sigma;        // NA
};
int launch_dress_gram(cudaStream_t st, const DressBatch& b, const GateTables& g);
// X[(kk + k*p'), (c + chi*a)] = sum_p Ahat[a][p'][p] R[kk, c + chi*p]
int launch_dress_R(cudaStream_t st, const DressBatch& b, const GateTables& g);
// out[:, (c + chi*a)] = in[:, (c + chi*a)] * sigma[a]   (rows = k[t])
int launch_scale_sigma(cudaStream_t st, const DressBatch& b, const GateTables& g);
// W[(c + chi*p), (c' + chin*p')] = sum_a Ahat[a][p'][p] T[(c + chi*a), c']   (T: N x chin, ld_in)
int launch_build_W(cudaStream_t st, const DressBatch& b, const GateTables& g, int* const* chi_new);
// Mp[kk, c' + chin*p'] = Mx[kk + k*p', c'] for kk<k ; rows k..m-1 of Mp (m = mrows) zeroed
int launch_reshuffle_M(cudaStream_t st, const DressBatch& b, int* const* chi_new, const long long* mrows);

}  // namespace pepo
