// api.cu - kernel-level entry points of include/pepo.h (BASELINE config 3 microbenchmarks and
// the parity tests): permutation, Gram, Cholesky-QR, Householder QR, Jacobi SVD, DGEMM.
#include "../../include/pepo.h"
#include "common.cuh"
#include "dense.cuh"
#include <algorithm>
#include <vector>

using namespace pepo;

namespace {
inline size_t al(size_t b) { return (b + 255) & ~(size_t)255; }
struct Carver {
  char* p; size_t left;
  void* take(size_t bytes) {
    bytes = al(bytes);
    if (bytes > left) return nullptr;
    void* r = p; p += bytes; left -= bytes; return r;
  }
};
}  // namespace

static int permute_common(const double* d_src, double* d_dst, const int* shape, const int* perm,
                          int rank, const double* const* scale, void* stream) {
  if (!shape || !perm || rank < 1 || rank > PEPO_MAX_RANK) {
    set_error("permute: bad argument"); return -1;
  }
  bool seen[PEPO_MAX_RANK] = {false};
  for (int j = 0; j < rank; j++) {
    if (perm[j] < 0 || perm[j] >= rank || seen[perm[j]]) { set_error("permute: perm is not a permutation"); return -1; }
    seen[perm[j]] = true;
    if (shape[j] < 0) { set_error("permute: negative extent"); return -1; }
  }
  long long total = 1;
  for (int j = 0; j < rank; j++) total *= shape[j];
  if (total == 0) return 0;                 // empty tensor: nothing to move
  if (!d_src || !d_dst) { set_error("permute: NULL tensor pointer"); return -1; }
  PermuteDesc pd;
  pd.rank = rank; pd.power = 1.0;
  long long s = 1;
  for (int d = 0; d < rank; d++) { pd.shape[d] = shape[d]; pd.src_stride[d] = s; s *= shape[d]; pd.scale[d] = scale ? scale[d] : nullptr; }
  long long t = 1;
  for (int j = 0; j < rank; j++) { pd.perm[j] = perm[j]; pd.dst_stride[j] = t; t *= shape[perm[j]]; }
  return launch_permute((cudaStream_t)stream, d_src, d_dst, pd);
}

extern "C" int pepo_permute(const double* d_src, double* d_dst, const int* h_shape,
                            const int* h_perm, int rank, void* stream) {
  return permute_common(d_src, d_dst, h_shape, h_perm, rank, nullptr, stream);
}
extern "C" int pepo_permute_scaled(const double* d_src, double* d_dst, const int* h_shape,
                                   const int* h_perm, int rank, const double* const* h_scale,
                                   void* stream) {
  return permute_common(d_src, d_dst, h_shape, h_perm, rank, h_scale, stream);
}

extern "C" size_t pepo_gram_ws_bytes(long long m, int n) {
  if (m < 0 || n < 1) return 0;
  int ks, kc;
  gram_plan(std::max(m, 1ll), n, &ks, &kc);
  return al((size_t)ks * n * n * 8);
}
extern "C" int pepo_gram(const double* d_A, long long m, int n, long long lda, double* d_C,
                         void* d_ws, size_t ws_bytes, void* stream) {
  if (!d_A || !d_C || m < 1 || n < 1 || lda < m || m >= (1ll << 31)) { set_error("gram: bad argument"); return -1; }
  if (ws_bytes < pepo_gram_ws_bytes(m, n) || !d_ws) { set_error("gram: workspace too small (%zu needed)", pepo_gram_ws_bytes(m, n)); return -2; }
  int ks, kc;
  gram_plan(m, n, &ks, &kc);
  GemmProb gp;
  gp.A = d_A; gp.B = d_A; gp.C = d_C; gp.lda = lda; gp.ldb = lda; gp.ldc = n; gp.M = n; gp.N = n; gp.K = (int)m;
  cudaStream_t st = (cudaStream_t)stream;
  int rc = launch_dgemm(st, 1, 0, gp, ks, kc, (double*)d_ws, true);
  if (rc) return rc;
  return launch_gram_reduce(st, ks > 1 ? (const double*)d_ws : d_C, ks, n, d_C, n);
}

extern "C" int pepo_dmma_peak(int iters, int ctas_per_sm, double* d_sink, double* h_flops, void* stream) {
  if (!d_sink) { set_error("dmma_peak: NULL sink"); return -1; }
  return launch_dmma_peak((cudaStream_t)stream, iters, ctas_per_sm, d_sink, h_flops);
}

// ---- permute-on-load contractions of the bond gate --------------------------------------------
static int site_view(const int* h_dims, int nlegs, int cut_leg, SiteView& v, const char* who) {
  if (!h_dims || nlegs < 1 || nlegs > 4 || cut_leg < 0 || cut_leg >= nlegs) { set_error("%s: bad legs", who); return -1; }
  v.nlegs = nlegs; v.cut = cut_leg;
  long long tot = 4;
  for (int l = 0; l < nlegs; l++) {
    if (h_dims[l] < 1 || h_dims[l] > 256) { set_error("%s: bond dimension %d out of range 1..256", who, h_dims[l]); return -1; }
    v.dims[l] = h_dims[l]; tot *= h_dims[l];
  }
  if (v.m() >= (1ll << 31) || tot >= (1ll << 40)) { set_error("%s: tensor too large", who); return -1; }
  return 0;
}
extern "C" size_t pepo_site_gram_ws_bytes(const int* h_dims, int nlegs, int cut_leg) {
  SiteView v;
  if (site_view(h_dims, nlegs, cut_leg, v, "site_gram_ws_bytes")) return 0;
  return pepo_gram_ws_bytes(v.m(), v.n());
}
extern "C" int pepo_site_gram(const double* d_psi, const int* h_dims, int nlegs, int cut_leg,
                              const double* const* h_w2, double* d_C, void* d_ws, size_t ws_bytes, void* stream) {
  SiteView v;
  if (site_view(h_dims, nlegs, cut_leg, v, "site_gram")) return -1;
  if (!d_psi || !d_C) { set_error("site_gram: NULL pointer"); return -1; }
  const size_t need = pepo_gram_ws_bytes(v.m(), v.n());
  if (!d_ws || ws_bytes < need) { set_error("site_gram: workspace too small (%zu needed)", need); return -2; }
  return launch_site_gram((cudaStream_t)stream, d_psi, v, h_w2, d_C, (double*)d_ws);
}
extern "C" int pepo_site_apply(const double* d_psi, const int* h_dims, int nlegs, int cut_leg, const double* d_W,
                               int chi_new, double* d_out, void* stream) {
  SiteView v;
  if (site_view(h_dims, nlegs, cut_leg, v, "site_apply")) return -1;
  if (!d_psi || !d_W || !d_out || chi_new < 1 || chi_new > 256) { set_error("site_apply: bad argument"); return -1; }
  return launch_site_apply((cudaStream_t)stream, d_psi, v, d_W, v.n(), chi_new, d_out);
}

extern "C" size_t pepo_cholqr_ws_bytes(long long m, int n) {
  if (m < 0 || n < 1) return 0;
  return pepo_gram_ws_bytes(m, n) + al((size_t)n * n * 8) + 256;
}
extern "C" int pepo_cholqr(const double* d_A, long long m, int n, long long lda, double* d_Q,
                           double* d_R, int* d_info, void* d_ws, size_t ws_bytes, void* stream) {
  if (!d_A || !d_Q || !d_R || !d_info || m < 1 || n < 1 || lda < m) { set_error("cholqr: bad argument"); return -1; }
  if (!d_ws || ws_bytes < pepo_cholqr_ws_bytes(m, n)) { set_error("cholqr: workspace too small (%zu needed)", pepo_cholqr_ws_bytes(m, n)); return -2; }
  cudaStream_t st = (cudaStream_t)stream;
  Carver cv{(char*)d_ws, ws_bytes};
  size_t gws = pepo_gram_ws_bytes(m, n);
  void* gram_ws = cv.take(gws);
  double* Rinv = (double*)cv.take((size_t)n * n * 8);
  if (!gram_ws || !Rinv) { set_error("cholqr: workspace carve failed"); return -2; }
  int rc = pepo_gram(d_A, m, n, lda, d_R, gram_ws, gws, stream);
  if (rc) return rc;
  MatBatch b; b.count = 1; b.A[0] = d_R; b.ld[0] = n; b.m[0] = n; b.n[0] = n;
  int* infos[1] = {d_info};
  rc = launch_potrf(st, b, infos, 0.0); if (rc) return rc;
  rc = launch_zero_lower(st, b); if (rc) return rc;
  MatBatch bi = b; bi.A[0] = Rinv;
  rc = launch_trtri(st, b, bi); if (rc) return rc;
  GemmProb gp;
  gp.A = d_A; gp.lda = lda; gp.B = Rinv; gp.ldb = n; gp.C = d_Q; gp.ldc = lda; gp.M = m; gp.N = n; gp.K = n;
  return launch_dgemm(st, 0, 0, gp, 1, 0, nullptr, false);
}

extern "C" size_t pepo_householder_ws_bytes(long long m, int n) {
  if (m < 0 || n < 1) return 0;
  return al((size_t)m * n * 8) + 2 * al((size_t)n * 8) + 256;
}
extern "C" int pepo_householder_qr(const double* d_A, long long m, int n, long long lda,
                                   double* d_Q, double* d_R, void* d_ws, size_t ws_bytes,
                                   void* stream) {
  if (!d_A || !d_Q || !d_R || m < 1 || n < 1 || lda < m) { set_error("householder_qr: bad argument"); return -1; }
  if (!d_ws || ws_bytes < pepo_householder_ws_bytes(m, n)) { set_error("householder_qr: workspace too small"); return -2; }
  cudaStream_t st = (cudaStream_t)stream;
  Carver cv{(char*)d_ws, ws_bytes};
  double* F = (double*)cv.take((size_t)m * n * 8);
  double* beta = (double*)cv.take((size_t)n * 8);
  double* tau = (double*)cv.take((size_t)n * 8);
  if (!F || !beta || !tau) { set_error("householder_qr: workspace carve failed"); return -2; }
  PEPO_CUDA_OK(cudaMemcpy2DAsync(F, (size_t)m * 8, d_A, (size_t)lda * 8, (size_t)m * 8, n, cudaMemcpyDeviceToDevice, st));
  const int k = (int)std::min<long long>(m, n);
  HHBatch h; h.count = 1; h.A[0] = F; h.lda[0] = m; h.m[0] = m; h.n[0] = n; h.beta[0] = beta; h.tau[0] = tau;
  int rc = launch_hh_factor(st, h); if (rc) return rc;
  double* Ro[1] = {d_R}; long long ldr[1] = {k};
  rc = launch_hh_extract_r(st, h, Ro, ldr); if (rc) return rc;
  // Q = H_0 ... H_{k-1} [I_k ; 0]
  HHApplyBatch a; a.count = 1; a.A[0] = F; a.lda[0] = m; a.m[0] = m; a.k[0] = k; a.beta[0] = beta; a.tau[0] = tau;
  a.Y[0] = d_Q; a.ldy[0] = m; a.ncols[0] = k;
  rc = launch_set_identity(st, d_Q, m, k); if (rc) return rc;
  return launch_hh_apply_q(st, a);
}

extern "C" size_t pepo_svd_ws_bytes(int m, int n) {
  if (m < 1 || n < 1) return 0;
  size_t M = std::max(m, n), Nc = std::min(m, n);
  return al(M * Nc * 8) + al((Nc * Nc + Nc) * 8) + al(Nc * 8) + al(Nc * 4) + 4 * 256 + al(16) + al(3 * Nc * 8) + al(16);
}
extern "C" int pepo_svd_jacobi(const double* d_A, int m, int n, int lda, double* d_U, double* d_s,
                               double* d_V, int* d_sweeps, void* d_ws, size_t ws_bytes,
                               void* stream) {
  if (!d_A || !d_U || !d_s || !d_V || m < 1 || n < 1 || lda < m) { set_error("svd_jacobi: bad argument"); return -1; }
  if (!d_ws || ws_bytes < pepo_svd_ws_bytes(m, n)) { set_error("svd_jacobi: workspace too small"); return -2; }
  cudaStream_t st = (cudaStream_t)stream;
  const int Nc = std::min(m, n), M = std::max(m, n);
  Carver cv{(char*)d_ws, ws_bytes};
  double* G = (double*)cv.take((size_t)M * Nc * 8);
  double* V = (double*)cv.take(((size_t)Nc * Nc + Nc) * 8);
  int* order = (int*)cv.take((size_t)Nc * 4);
  int* ints = (int*)cv.take(16);
  double* lam3 = (double*)cv.take((size_t)3 * Nc * 8);
  double* gs = (double*)cv.take(16);
  if (!G || !V || !order || !ints || !lam3 || !gs) { set_error("svd_jacobi: workspace carve failed"); return -2; }
  SvdBatch sb; sb.count = 1;
  sb.K[0] = d_A; sb.ldk[0] = lda; sb.r1[0] = m; sb.r2[0] = n; sb.G[0] = G; sb.V[0] = V; sb.sv[0] = d_s;
  sb.order[0] = order; sb.sweeps[0] = d_sweeps ? d_sweeps : ints + 1;
  int rc = launch_svd_jacobi(st, sb, 1e-15, 60, true, 0, 0.0); if (rc) return rc;
  return launch_svd_vectors(st, G, V, d_s, order, m, n, d_U, d_V);
}

extern "C" int pepo_dgemm(int transA, int transB, long long M, int N, int K, const double* d_A,
                          long long lda, const double* d_B, long long ldb, double* d_C,
                          long long ldc, void* stream) {
  if (!d_A || !d_B || !d_C || M < 0 || N < 0 || K < 0 || (transA & ~1) || (transB & ~1)) { set_error("dgemm: bad argument"); return -1; }
  GemmProb gp;
  gp.A = d_A; gp.B = d_B; gp.C = d_C; gp.lda = lda; gp.ldb = ldb; gp.ldc = ldc; gp.M = M; gp.N = N; gp.K = K;
  return launch_dgemm((cudaStream_t)stream, transA, transB, gp, 1, 0, nullptr, false);
}
