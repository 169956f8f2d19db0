// ctx.cu - the context behind the C ABI of include/pepo.h: lattice bookkeeping, the single
// pre-sized device arena ("zero-malloc"), the analytic memory model
// (eq. (15)-(17) L292-L304 re-derived for this layout), the Trotter step scheduler (Fig. 1
// L310-L342; colour classes L87) and the BP / Bethe drivers.
//
// Schedule of one bond-gate batch (<= max_inflight gates of one colour class, disjoint sites):
//   A. per site: cv = permute(psi * sqrt(lambda_env))             (a2-a4, fused)
//   B. tall sites (m >= ratio*n): C = cv^T cv on DMMA, S = dressed Gram, Rx = chol(S)   (a5)
//      -> host reads the potrf flags of the batch (the paper's potrf_info, L221)
//   C. rejected / short sites: Householder cv = Q R, X = dress(R), Householder X = Qx Rx (a6)
//   D. per gate: K = Rx1 (Sigma x I) Rx2^T, Jacobi SVD, truncation, lambda           (a7-a9)
//      -> host reads chi_new of the batch (the paper's host threshold, L344)
//   E. per site: Cholesky path  W = dress(Rx^-1 U sqrt(S)), cv_new = cv W (DMMA)
//                Householder    cv_new = Q [dress(Qx [U sqrt(S); 0]); 0]              (a10)
//   F. per site: psi = inverse-permute(cv_new) / sqrt(lambda_env)  (a11-a13, fused)
// The gate is applied in Schmidt-dressed form: G = sum_a sigma_a Ahat_a (x) Bhat_a (operator-
// Schmidt decomposition of the 16x16 Pauli-transfer matrix, rank 4 for ZZ), so that the core
// the Jacobi SVD sees is (NA chi) x (NA chi) instead of the literal (16 chi)^2.
#include "../../include/pepo.h"
#include "bp.cuh"
#include "common.cuh"
#include "dense.cuh"
#include "normbp.cuh"

#include <algorithm>
#include <chrono>
#include <cmath>
#include <complex>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <string>
#include <deque>
#include <vector>
#include <thread>

namespace pepo {

static thread_local long long t_scratch_launches = 0;
thread_local long long* t_launch_counter = &t_scratch_launches;
static thread_local char g_err[512] = "";
void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}
const char* last_error() { return g_err; }

// ------------------------------------------------------------------------------------------
// host-side gate tables
// ------------------------------------------------------------------------------------------
typedef std::complex<double> cplx;
static void pauli(int p, cplx m[2][2]) {
  static const cplx I(0, 1);
  cplx z(0, 0), o(1, 0);
  switch (p) {
    case 0: m[0][0] = o; m[0][1] = z; m[1][0] = z; m[1][1] = o; break;
    case 1: m[0][0] = z; m[0][1] = o; m[1][0] = o; m[1][1] = z; break;
    case 2: m[0][0] = z; m[0][1] = -I; m[1][0] = I; m[1][1] = z; break;
    default: m[0][0] = o; m[0][1] = z; m[1][0] = z; m[1][1] = -o; break;
  }
}
// dense d x d helpers
static void matmul(const std::vector<cplx>& A, const std::vector<cplx>& B, std::vector<cplx>& C, int d) {
  C.assign((size_t)d * d, cplx(0, 0));
  for (int i = 0; i < d; i++)
    for (int k = 0; k < d; k++)
      for (int j = 0; j < d; j++) C[i * d + j] += A[i * d + k] * B[k * d + j];
}
static std::vector<cplx> dagger(const std::vector<cplx>& A, int d) {
  std::vector<cplx> R((size_t)d * d);
  for (int i = 0; i < d; i++)
    for (int j = 0; j < d; j++) R[i * d + j] = std::conj(A[j * d + i]);
  return R;
}
static std::vector<cplx> kron2(int a, int b) {
  cplx A[2][2], B[2][2];
  pauli(a, A); pauli(b, B);
  std::vector<cplx> R(16);
  for (int i = 0; i < 2; i++) for (int j = 0; j < 2; j++)
    for (int k = 0; k < 2; k++) for (int l = 0; l < 2; l++) R[(i * 2 + k) * 4 + (j * 2 + l)] = A[i][j] * B[k][l];
  return R;
}
// PTM of conjugation by U = exp(+i theta P): G[a][b] = Tr[P_a U^dag P_b U]/2  (R2)
static void ptm_one_site(double theta, int fp, double G[16]) {
  cplx P[2][2]; pauli(fp, P);
  std::vector<cplx> U(4), Pa(4), Pb(4), T1, T2, T3;
  for (int i = 0; i < 2; i++) for (int j = 0; j < 2; j++)
    U[i * 2 + j] = (i == j ? cplx(std::cos(theta), 0) : cplx(0, 0)) + cplx(0, std::sin(theta)) * P[i][j];
  std::vector<cplx> Ud = dagger(U, 2);
  for (int a = 0; a < 4; a++) for (int b = 0; b < 4; b++) {
    cplx A[2][2], B[2][2]; pauli(a, A); pauli(b, B);
    for (int i = 0; i < 2; i++) for (int j = 0; j < 2; j++) { Pa[i * 2 + j] = A[i][j]; Pb[i * 2 + j] = B[i][j]; }
    matmul(Pa, Ud, T1, 2); matmul(T1, Pb, T2, 2); matmul(T2, U, T3, 2);
    G[a * 4 + b] = (T3[0] + T3[3]).real() / 2.0;
  }
}
// 16x16 PTM of exp(+i theta P (x) P); row p1'*4+p2', column p1*4+p2 (R15)
static void ptm_two_site(double theta, int bp, double G[256]) {
  std::vector<cplx> PP = kron2(bp, bp), U(16), T1, T2, T3;
  for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++)
    U[i * 4 + j] = (i == j ? cplx(std::cos(theta), 0) : cplx(0, 0)) + cplx(0, std::sin(theta)) * PP[i * 4 + j];
  std::vector<cplx> Ud = dagger(U, 4);
  for (int a1 = 0; a1 < 4; a1++) for (int a2 = 0; a2 < 4; a2++) {
    std::vector<cplx> Pa = kron2(a1, a2);
    for (int b1 = 0; b1 < 4; b1++) for (int b2 = 0; b2 < 4; b2++) {
      std::vector<cplx> Pb = kron2(b1, b2);
      matmul(Pa, Ud, T1, 4); matmul(T1, Pb, T2, 4); matmul(T2, U, T3, 4);
      cplx tr(0, 0);
      for (int i = 0; i < 4; i++) tr += T3[i * 4 + i];
      G[(a1 * 4 + a2) * 16 + (b1 * 4 + b2)] = tr.real() / 4.0;
    }
  }
}
// one-sided Jacobi SVD of a 16x16 host matrix (column-major A = U S V^T); returns sorted.
static void host_svd16(const double* Ain, double* U, double* s, double* V) {
  const int n = 16;
  double G[256], W[256];
  memcpy(G, Ain, sizeof(G));
  for (int i = 0; i < 256; i++) W[i] = (i % n == i / n) ? 1.0 : 0.0;
  for (int sweep = 0; sweep < 100; sweep++) {
    bool rot = false;
    for (int p = 0; p < n; p++) for (int q = p + 1; q < n; q++) {
      double al = 0, be = 0, ga = 0;
      for (int k = 0; k < n; k++) { al += G[p * n + k] * G[p * n + k]; be += G[q * n + k] * G[q * n + k]; ga += G[p * n + k] * G[q * n + k]; }
      if (al < 1e-300 || be < 1e-300) continue;
      if (std::fabs(ga) <= 1e-16 * std::sqrt(al * be)) continue;
      rot = true;
      double zeta = (be - al) / (2 * ga);
      double t = (zeta >= 0 ? 1.0 : -1.0) / (std::fabs(zeta) + std::sqrt(1 + zeta * zeta));
      double c = 1 / std::sqrt(1 + t * t), sn = c * t;
      for (int k = 0; k < n; k++) {
        double x = G[p * n + k], y = G[q * n + k];
        G[p * n + k] = c * x - sn * y; G[q * n + k] = sn * x + c * y;
        x = W[p * n + k]; y = W[q * n + k];
        W[p * n + k] = c * x - sn * y; W[q * n + k] = sn * x + c * y;
      }
    }
    if (!rot) break;
  }
  double nr[16]; int ord[16];
  for (int j = 0; j < n; j++) { double a = 0; for (int k = 0; k < n; k++) a += G[j * n + k] * G[j * n + k]; nr[j] = std::sqrt(a); ord[j] = j; }
  std::stable_sort(ord, ord + n, [&](int a, int b) { return nr[a] > nr[b]; });
  for (int c = 0; c < n; c++) {
    int j = ord[c];
    s[c] = nr[j];
    for (int k = 0; k < n; k++) { U[c * n + k] = nr[j] > 0 ? G[j * n + k] / nr[j] : 0.0; V[c * n + k] = W[j * n + k]; }
  }
}

// ------------------------------------------------------------------------------------------
// lattice
// ------------------------------------------------------------------------------------------
static const int DXY[4][2] = {{0, -1}, {0, 1}, {-1, 0}, {1, 0}};   // U, D, L, R
static const int OPP[4] = {1, 0, 3, 2};

struct SiteInfo {
  int x, y;
  int nlegs;
  int leg_dir[4];     // canonical order, present legs only
  int leg_bond[4];
  int nbr[4];         // per direction: neighbour site or -1
  int bond_of_dir[4];
  double* psi;        // device slot
  size_t cap;         // doubles
};
struct BondInfo { int v1, d1, v2, d2; };

struct SiteWs {       // per lane, per site-slot
  double *cv, *out, *C, *Rx, *Rxinv, *Rbuf, *X, *T, *W, *Mx, *beta1, *tau1, *beta2, *tau2, *part;
  // spare[d]: a buffer of the size of a site slot with d legs.  On the Cholesky path the reconstruction
  // GEMM writes the new site tensor straight into spare[nlegs] in the canonical layout and the site
  // takes that buffer; its old slot becomes this lane's spare (stream-ordered: a lane belongs to one
  // piece stream).  `out` (work matrix of the Householder path) is the spare of the largest class.
  double* spare[5];
  int* info;          // device int (in the lane readback block)
};
struct LaneWs {
  SiteWs s[2];
  double *K, *Ks, *G, *V, *sv, *Us, *Vs;
  int* order;
  int* ints;          // [chi_new, sweeps, info0, info1]
  int* orient;        // device int: the Jacobi kernel iterated on K^T (square core, option "svd_orient")
  double* dbls;       // [discarded, gap]
};

struct Arena {
  char* base = nullptr; size_t size = 0, top = 0;
  bool dry = false; size_t model = 0;     // dry run: only account (model = unaligned sum)
  // Every buffer is followed by a guard zone of PEPO_GUARD bytes holding a fixed pattern (the arena
  // canaries of SURVEY section 5): pepo_check_guards() finds a kernel that wrote past its buffer.
  std::vector<size_t> guards;             // offsets of the guard zones
  std::vector<const char*> names;         // which buffer each guard follows (layout()'s name of it)
  void* take(const char* name, size_t bytes) {
    names.push_back(name);
    model += bytes;
    size_t off = (top + 255) & ~(size_t)255;
    top = off + bytes;
    const size_t g = (top + 7) & ~(size_t)7;
    guards.push_back(g);
    top = g + 64;
    if (dry) return nullptr;
    return base ? base + off : nullptr;
  }
};

// ---- optional in-situ profiling: CUDA-event pairs around every launch group, accumulated per
// category at the existing host sync points (option "profile").  Events are created at init.
enum ProfCat { PC_PERMUTE = 0, PC_GRAM, PC_APPLY, PC_SMALL_GEMM, PC_CHOL, PC_HOUSEHOLDER, PC_DRESS,
               PC_SVD, PC_FIELD, PC_BP, PC_COUNT };
struct Prof {
  bool on = false;
  std::vector<cudaEvent_t> ev;
  std::vector<int> cat;          // category of pair i
  std::vector<int> strm;         // stream id of pair i (trace)
  int trace = 0;                 // option "trace": print (category, stream, start, end) of every pair at the flush
  size_t used = 0;               // pairs in flight
  double ms[PC_COUNT] = {0}, flops[PC_COUNT] = {0}, bytes[PC_COUNT] = {0};
  long long cnt[PC_COUNT] = {0};
};

}  // namespace pepo

using namespace pepo;

constexpr int BP_GROUP = 8;            // delta slots (sweeps per read-back, upper bound)

struct pepo_ctx {
  int Lx, Ly, cx, cy, center;
  double J, h, dt, bp_tol, bp_damping;
  int chi_max, B;      // B = max inflight gates
  int bondP, fieldP, obsP;
  double eps_cut = 1e-11, chol_ratio = 4.0, chol_tau = 1e-7, jacobi_tol = 1e-15;
  int bp_max_sweeps = 100, bp_max_sweeps_damped = 1000, jacobi_max_sweeps = 60;
  int force_hh = 0;
  int direct = 1;                      // option "direct_gemm": Cholesky-path GEMMs read / write psi in place (no permute passes)
  int svd_precond_min = 32;            // QR-precondition core SVDs with min(r1,r2) >= this (0: off)
  cudaStream_t st;
  cudaStream_t cur_st = nullptr;       // stream the profiling events of the current launches go to
  // pipelined schedule of a Trotter step (option "pipeline" = number of piece streams, 0/1 = serial):
  // pieces of the colour classes on the streams ps[], their Jacobi kernels on the high-priority
  // streams hp[]; pev: per stream [svd fork, svd join, read-back], then [fork, join per stream]
  int pipeline = 4;
  static constexpr int NSMAX = 4;
  cudaStream_t ps[NSMAX] = {nullptr}, hp[NSMAX] = {nullptr};
  cudaEvent_t pev[5 * NSMAX + 1] = {nullptr};
  int bp_group = 8;                    // option "bp_group": BP sweeps enqueued per delta read-back (1..BP_GROUP)
  int bp_init = 0;                     // option "bp_init": 0 = uniform init of R7, 1 = leading Schmidt vector e_0
  int bp_ladder = 0;                   // option "bp_ladder": third BP stage with damping bp_damping2 (alpha-retry, L451-L457)
  double bp_damping2 = 0.2;            // option "bp_damping2": alpha = 0.8
  double obs_prev_C = 1.0, obs_prev_gerr = 0.0;   // last C(t) / gate_err accepted by pepo_observe (C(0) = 1)
  int svd_orient = 1;                  // option "svd_orient": 0 QR of K, 1 of the more graded of K / K^T (default), 2 of K^T (square cores)
  double svd_deflate = 0.0;            // option "svd_deflate": theta of the truncation-aware deflation of the Jacobi SVD (0: off, default)
  double jacobi_early = 1e-7;          // option "jacobi_early": cosine below which a Jacobi sweep counts as the last one
  std::vector<cudaEvent_t> done_ev;    // completion events of the pieces of a pipelined step
  int n_sites, n_bonds, n_hb;
  std::vector<SiteInfo> sites;
  std::vector<BondInfo> bonds;
  std::vector<std::vector<int>> classes;
  std::vector<int> chi;
  // device
  Arena arena;
  double *lambda, *sqrt_l, *isqrt_l;     // n_bonds * chi_max each
  double *msgs[2];                        // 2*n_bonds*chi_max each
  int* chi_of_msg;                        // device 2*n_bonds
  double* ones;                           // [1.0]
  double* vs;                             // n_sites
  double* bp_scalars;                     // [C]
  unsigned long long* delta_bits;
  int* bp_ints;                           // [flag, status]
  std::vector<double*> partU, partD, partS;
  // NEXT-1: norm-network BP with chi x chi matrix messages (option "env" = 1 feeds them to the gates).
  // Indexed like msgs: 2e = sent by v1 of bond e, 2e + 1 = sent by v2; packed, ld = live chi of the bond.
  int env_mode = 0;
  double* nM[2] = {nullptr, nullptr};     // two sets of 2 n_bonds messages (chi_max^2 each)
  double *nS = nullptr, *nSinv = nullptr; // PSEUDO_SQRT and its pseudo-inverse of the current messages
  double *nG = nullptr, *nraw = nullptr;  // cross Gram (4 chi)^2; unnormalised message chi^2
  double *nEg = nullptr, *nEv = nullptr, *nEu = nullptr, *nEw = nullptr, *nEs = nullptr;   // eigen workspace
  int* nEo = nullptr;                     // order (chi ints) + sweeps
  double* nscal = nullptr;                // n_sites + n_bonds scalars (f_v, Z_e)
  int n_cur = 0;
  bool n_valid = false, n_sqrt_valid = false;
  double psqrt_eps = 1e-12;               // option "psqrt_eps"
  double* sw_part = nullptr;              // n_sites x PEPO_SW_CHUNKS x 4 partials of pepo_site_weights
  double* sw_out = nullptr;               // n_sites x 4
  double *dG1, *dGamma[2], *dAhat[2], *dSigma;
  int NA;
  double G1[16], G1h[16];              // field PTM at h dt and at h dt / 2 (symmetric step, eq. (6))
  int f_row_mask, f_col_mask;
  // asynchronous site uploads (pepo_set_site_async): copies on copy_st, one event per site; the
  // first kernels that touch a site wait for its event (field gate of the piece that owns it)
  cudaStream_t copy_st = nullptr;
  cudaEvent_t copy_ev = nullptr;
  bool lazy_field = false, lazy_half = false;   // this step applies the field gate piece by piece
  std::vector<cudaEvent_t> site_ev;
  std::vector<char> site_pending, field_todo;
  bool copy_forked = false;            // copy_st already ordered after the compute queued so far
  int n_pending = 0;
  int trotter_order = 1;               // option "trotter_order": 1 = R2 (BASELINE), 2 = symmetric step of eq. (6)
  std::vector<LaneWs> lanes;
  int* lane_orient = nullptr;             // B ints (LaneWs::orient)
  size_t part_cap = 0;                    // doubles of every SiteWs::part
  int* lane_ints; double* lane_dbls;      // device readback blocks (B*4 ints, B*2 doubles)
  // pinned host
  int* h_ints = nullptr; double* h_dbls = nullptr; int* h_chi_msg = nullptr; double* h_scal = nullptr;
  unsigned long long* h_delta = nullptr; int* h_bpints = nullptr;
  int cur_msg = 0;
  bool msgs_valid = false;
  long long launches = 0;              // kernels launched for this context (PEPO_COUNT_LAUNCH via t_launch_counter)
  pepo_stats stats;
  size_t model_bytes = 0;
  Prof prof;
};

namespace {
// Kernel launches made while an API call works for a context are counted into that context.
struct CtxScope {
  long long* prev;
  explicit CtxScope(pepo_ctx* c) : prev(pepo::t_launch_counter) { pepo::t_launch_counter = &c->launches; }
  ~CtxScope() { pepo::t_launch_counter = prev; }
};

void prof_flush(pepo_ctx* c) {        // call only after a stream synchronize
  Prof& P = c->prof;
  for (size_t i = 0; i < P.used; i++) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, P.ev[2 * i], P.ev[2 * i + 1]) == cudaSuccess) P.ms[P.cat[i]] += ms;
    if (P.trace) {
      float t0 = 0.f, t1 = 0.f;
      cudaEventElapsedTime(&t0, P.ev[0], P.ev[2 * i]);
      cudaEventElapsedTime(&t1, P.ev[0], P.ev[2 * i + 1]);
      fprintf(stderr, "TRACE %d %d %.3f %.3f\n", P.cat[i], P.strm[i], t0, t1);
    }
  }
  P.used = 0;
}
struct ProfScope {
  pepo_ctx* c; bool active; cudaStream_t st = nullptr;
  ProfScope(pepo_ctx* c_, int cat, double flops, double bytes) : c(c_), active(false) {
    Prof& P = c->prof;
    if (!P.on) return;
    if (2 * (P.used + 1) > P.ev.size()) {
      cudaStreamSynchronize(c->st);
      for (int i = 0; i < pepo_ctx::NSMAX; i++) if (c->ps[i]) { cudaStreamSynchronize(c->ps[i]); cudaStreamSynchronize(c->hp[i]); }
      prof_flush(c);
    }
    P.cat[P.used] = cat; P.cnt[cat]++; P.flops[cat] += flops; P.bytes[cat] += bytes;
    st = c->cur_st ? c->cur_st : c->st;
    P.strm[P.used] = 0;
    for (int i = 0; i < pepo_ctx::NSMAX; i++) { if (st == c->ps[i]) P.strm[P.used] = i; if (st == c->hp[i]) P.strm[P.used] = pepo_ctx::NSMAX + i; }
    cudaEventRecord(P.ev[2 * P.used], st);
    active = true;
  }
  ~ProfScope() {
    if (!active) return;
    Prof& P = c->prof;
    cudaEventRecord(P.ev[2 * P.used + 1], st);
    P.used++;
  }
};
}  // namespace

namespace {
int wait_pending_uploads(pepo_ctx* c, cudaStream_t st);
}

namespace {

size_t ipow(size_t b, int e) { size_t r = 1; while (e-- > 0) r *= b; return r; }

void build_lattice(int Lx, int Ly, std::vector<SiteInfo>& sites, std::vector<BondInfo>& bonds,
                   std::vector<std::vector<int>>& classes, int& n_hb) {
  const int ns = Lx * Ly;
  n_hb = Ly * (Lx - 1);
  const int nb = n_hb + (Ly - 1) * Lx;
  sites.assign(ns, SiteInfo());
  bonds.assign(nb, BondInfo());
  for (int e = 0; e < nb; e++) {
    if (e < n_hb) { int y = e / (Lx - 1), x = e % (Lx - 1); bonds[e] = {y * Lx + x, 3, y * Lx + x + 1, 2}; }
    else { int q = e - n_hb; int y = q / Lx, x = q % Lx; bonds[e] = {y * Lx + x, 1, (y + 1) * Lx + x, 0}; }
  }
  for (int v = 0; v < ns; v++) {
    SiteInfo& s = sites[v];
    s.x = v % Lx; s.y = v / Lx; s.nlegs = 0;
    for (int d = 0; d < 4; d++) {
      int x2 = s.x + DXY[d][0], y2 = s.y + DXY[d][1];
      s.nbr[d] = -1; s.bond_of_dir[d] = -1;
      if (x2 < 0 || x2 >= Lx || y2 < 0 || y2 >= Ly) continue;
      s.nbr[d] = y2 * Lx + x2;
      int e;
      if (d == 3) e = s.y * (Lx - 1) + s.x;
      else if (d == 2) e = s.y * (Lx - 1) + s.x - 1;
      else if (d == 1) e = n_hb + s.y * Lx + s.x;
      else e = n_hb + (s.y - 1) * Lx + s.x;
      s.bond_of_dir[d] = e;
      s.leg_dir[s.nlegs] = d; s.leg_bond[s.nlegs] = e; s.nlegs++;
    }
  }
  classes.assign(4, std::vector<int>());
  for (int y = 0; y < Ly; y++) for (int x = 0; x + 1 < Lx; x++) classes[x % 2].push_back(y * (Lx - 1) + x);
  for (int y = 0; y + 1 < Ly; y++) for (int x = 0; x < Lx; x++) classes[2 + y % 2].push_back(n_hb + y * Lx + x);
}

size_t gram_part_cap(int chi_max, size_t m_max) {
  size_t best = 0;
  for (int c = 1; c <= chi_max; c++) {
    const int n = 4 * c;
    // every m <= m_max occurs (mixed bond dimensions during growth): the bound over all of them
    const int ks = gram_max_splits((long long)m_max, n);
    best = std::max(best, (size_t)ks * n * n);
  }
  return best;
}

// Lays out (or, with arena.dry, only accounts) every device buffer.  The same routine is the
// memory model: arena.model = plain sum of the buffer sizes.
int layout(pepo_ctx* c) {
  Arena& A = c->arena;
  const size_t chi = c->chi_max;
  const int NA = c->NA;
  const size_t nmax = 4 * chi, Nmax = (size_t)NA * chi;
  int degmax = 0;
  for (auto& s : c->sites) degmax = std::max(degmax, s.nlegs);
  for (auto& s : c->sites) {
    s.cap = 4 * ipow(chi, s.nlegs);
    s.psi = (double*)A.take("s.psi", s.cap * 8);
  }
  const size_t nb = c->n_bonds;
  c->lambda = (double*)A.take("c->lambda", nb * chi * 8);
  c->sqrt_l = (double*)A.take("c->sqrt_l", nb * chi * 8);
  c->isqrt_l = (double*)A.take("c->isqrt_l", nb * chi * 8);
  c->msgs[0] = (double*)A.take("c->msgs[0]", 2 * nb * chi * 8 + 8);
  c->msgs[1] = (double*)A.take("c->msgs[1]", 2 * nb * chi * 8 + 8);
  c->chi_of_msg = (int*)A.take("c->chi_of_msg", 2 * nb * 4 + 4);
  c->ones = (double*)A.take("c->ones", 8);
  c->vs = (double*)A.take("c->vs", c->n_sites * 8);
  c->bp_scalars = (double*)A.take("c->bp_scalars", 16);
  c->delta_bits = (unsigned long long*)A.take("c->delta_bits", 8 * BP_GROUP);
  c->bp_ints = (int*)A.take("c->bp_ints", 16);
  c->partU.assign(c->n_sites, nullptr); c->partD.assign(c->n_sites, nullptr); c->partS.assign(c->n_sites, nullptr);
  for (int v = 0; v < c->n_sites; v++) {
    const SiteInfo& s = c->sites[v];
    // BP roles (fill_bp_site): the legs that exist, in storage order, play the roles (u, d, l, r) of the
    // sweep kernel; per-chunk partial vectors: <= d_l d_r chunks of d_u (d_d) entries, d_l d_r slice scalars
    const int nl = s.nlegs;
    c->partU[v] = (double*)A.take("c->partU[v]", ipow(chi, (nl >= 1) + (nl >= 3) + (nl >= 4)) * 8);
    c->partD[v] = (double*)A.take("c->partD[v]", ipow(chi, (nl >= 2) + (nl >= 3) + (nl >= 4)) * 8);
    c->partS[v] = (double*)A.take("c->partS[v]", ipow(chi, (nl >= 3) + (nl >= 4)) * 8);
  }
  {
    const size_t x2 = chi * chi;
    for (int i = 0; i < 2; i++) c->nM[i] = (double*)A.take("c->nM[i]", 2 * nb * x2 * 8 + 8);
    c->nS = (double*)A.take("c->nS", 2 * nb * x2 * 8 + 8);
    c->nSinv = (double*)A.take("c->nSinv", 2 * nb * x2 * 8 + 8);
    c->nG = (double*)A.take("c->nG", 16 * x2 * 8);
    c->nraw = (double*)A.take("c->nraw", x2 * 8);
    c->nEg = (double*)A.take("c->nEg", x2 * 8); c->nEv = (double*)A.take("c->nEv", (x2 + chi) * 8);
    c->nEu = (double*)A.take("c->nEu", x2 * 8); c->nEw = (double*)A.take("c->nEw", x2 * 8); c->nEs = (double*)A.take("c->nEs", chi * 8);
    c->nEo = (int*)A.take("c->nEo", (chi + 4) * 4);
    c->nscal = (double*)A.take("c->nscal", (c->n_sites + nb + 1) * 8);
  }
  c->sw_part = (double*)A.take("c->sw_part", (size_t)c->n_sites * PEPO_SW_CHUNKS * 4 * 8);
  c->sw_out = (double*)A.take("c->sw_out", (size_t)c->n_sites * 4 * 8);
  c->dG1 = (double*)A.take("c->dG1", 16 * 8);
  for (int i = 0; i < 2; i++) {
    c->dGamma[i] = (double*)A.take("c->dGamma[i]", (size_t)NA * NA * 16 * 8);
    c->dAhat[i] = (double*)A.take("c->dAhat[i]", (size_t)NA * 16 * 8);
  }
  c->dSigma = (double*)A.take("c->dSigma", NA * 8);
  c->lane_ints = (int*)A.take("c->lane_ints", (size_t)c->B * 4 * 4);
  c->lane_dbls = (double*)A.take("c->lane_dbls", (size_t)c->B * 2 * 8);
  c->lane_orient = (int*)A.take("c->lane_orient", (size_t)c->B * 4);
  const size_t m_max = ipow(chi, std::max(degmax - 1, 0));
  const size_t ld_max = (m_max + 1) & ~(size_t)1;
  const size_t cvcap = ld_max * nmax;
  const size_t partcap = (degmax >= 1) ? gram_part_cap(c->chi_max, m_max) : 0;
  c->part_cap = partcap;
  c->lanes.assign(c->B, LaneWs());
  for (int l = 0; l < c->B; l++) {
    LaneWs& L = c->lanes[l];
    L.ints = c->lane_ints ? c->lane_ints + 4 * l : nullptr;
    L.dbls = c->lane_dbls ? c->lane_dbls + 2 * l : nullptr;
    L.orient = c->lane_orient ? c->lane_orient + l : nullptr;
    for (int i = 0; i < 2; i++) {
      SiteWs& S = L.s[i];
      S.cv = (double*)A.take("S.cv", cvcap * 8);
      for (int d = 0; d < 5; d++) S.spare[d] = nullptr;
      for (int d = 1; d <= degmax; d++) {
        bool have = false;
        for (auto& sv : c->sites) have |= (sv.nlegs == d);
        if (!have) continue;
        // the largest class also serves as the Householder path's work matrix (even leading dimension)
        S.spare[d] = (double*)A.take("S.spare[d]", (d == degmax ? std::max(cvcap, 4 * ipow(chi, d)) : 4 * ipow(chi, d)) * 8);
      }
      S.out = degmax >= 1 ? S.spare[degmax] : (double*)A.take("S.out", cvcap * 8);
      S.C = (double*)A.take("S.C", nmax * nmax * 8);
      S.Rx = (double*)A.take("S.Rx", Nmax * Nmax * 8);
      S.Rxinv = (double*)A.take("S.Rxinv", Nmax * Nmax * 8);
      S.Rbuf = (double*)A.take("S.Rbuf", nmax * nmax * 8);
      S.X = (double*)A.take("S.X", 4 * nmax * Nmax * 8);
      S.T = (double*)A.take("S.T", Nmax * chi * 8);
      S.W = (double*)A.take("S.W", nmax * 4 * chi * 8);
      S.Mx = (double*)A.take("S.Mx", 4 * nmax * chi * 8);
      S.beta1 = (double*)A.take("S.beta1", nmax * 8); S.tau1 = (double*)A.take("S.tau1", nmax * 8);
      S.beta2 = (double*)A.take("S.beta2", Nmax * 8); S.tau2 = (double*)A.take("S.tau2", Nmax * 8);
      S.part = (double*)A.take("S.part", partcap * 8);
      S.info = L.ints ? L.ints + 2 + i : nullptr;
    }
    L.K = (double*)A.take("L.K", Nmax * Nmax * 8);
    L.Ks = (double*)A.take("L.Ks", Nmax * Nmax * 8);
    L.G = (double*)A.take("L.G", Nmax * Nmax * 8);
    L.V = (double*)A.take("L.V", (Nmax * Nmax + Nmax) * 8);     // + Nmax: unsorted norms scratch
    L.sv = (double*)A.take("L.sv", Nmax * 8);
    L.Us = (double*)A.take("L.Us", Nmax * chi * 8);
    L.Vs = (double*)A.take("L.Vs", Nmax * chi * 8);
    L.order = (int*)A.take("L.order", Nmax * 4);
  }
  return 0;
}

int max_class_size(int Lx, int Ly) {
  std::vector<SiteInfo> s; std::vector<BondInfo> b; std::vector<std::vector<int>> cl; int nh;
  build_lattice(Lx, Ly, s, b, cl, nh);
  size_t m = 1;
  for (auto& c : cl) m = std::max(m, c.size());
  return (int)m;
}

size_t model_bytes_for(int Lx, int Ly, int chi_max, int B, int NA, size_t* aligned_top) {
  pepo_ctx tmp;
  tmp.Lx = Lx; tmp.Ly = Ly; tmp.chi_max = chi_max; tmp.B = B; tmp.NA = NA;
  build_lattice(Lx, Ly, tmp.sites, tmp.bonds, tmp.classes, tmp.n_hb);
  tmp.n_sites = Lx * Ly; tmp.n_bonds = (int)tmp.bonds.size();
  tmp.arena.dry = true;
  layout(&tmp);
  if (aligned_top) *aligned_top = tmp.arena.top;
  return tmp.arena.model;
}

int default_inflight(int Lx, int Ly, int chi_max, int NA) {
  int B = std::min(max_class_size(Lx, Ly), 16);
  const double budget = 170e9;
  while (B > 1) {
    size_t top;
    model_bytes_for(Lx, Ly, chi_max, B, NA, &top);
    if ((double)top <= budget) break;
    B--;
  }
  return std::max(B, 1);
}

inline double* bond_vec(double* base, int e, int chi_max) { return base + (size_t)e * chi_max; }

}  // namespace

// ============================================================================================
// C ABI: lifetime
// ============================================================================================
extern "C" const char* pepo_last_error(void) { return pepo::last_error(); }

extern "C" size_t pepo_arena_bytes_ex(int Lx, int Ly, int chi_max, int max_inflight) {
  if (Lx < 1 || Ly < 1 || chi_max < 1) return 0;
  int B = max_inflight > 0 ? std::min(max_inflight, PEPO_MAXT / 2) : default_inflight(Lx, Ly, chi_max, 4);
  size_t top;
  model_bytes_for(Lx, Ly, chi_max, B, 4, &top);
  return top + 256;
}
extern "C" size_t pepo_arena_bytes(int Lx, int Ly, int chi_max) {
  return pepo_arena_bytes_ex(Lx, Ly, chi_max, 0);
}

static int upload(pepo_ctx* c, void* dst, const void* src, size_t bytes) {
  PEPO_CUDA_OK(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, c->st));
  PEPO_CUDA_OK(cudaStreamSynchronize(c->st));
  return 0;
}

static int reset_state(pepo_ctx* c) {
  // product operator: all bonds chi = 1, lambda = [1]
  std::fill(c->chi.begin(), c->chi.end(), 1);
  for (int v = 0; v < c->n_sites; v++) {
    double t[4] = {0, 0, 0, 0};
    t[v == c->center ? c->obsP : 0] = 1.0;
    int rc = upload(c, c->sites[v].psi, t, sizeof(t));
    if (rc) return rc;
  }
  std::vector<double> one((size_t)c->n_bonds * c->chi_max, 0.0);
  for (int e = 0; e < c->n_bonds; e++) one[(size_t)e * c->chi_max] = 1.0;
  if (c->n_bonds) {
    int rc = upload(c, c->lambda, one.data(), one.size() * 8); if (rc) return rc;
    rc = upload(c, c->sqrt_l, one.data(), one.size() * 8); if (rc) return rc;
    rc = upload(c, c->isqrt_l, one.data(), one.size() * 8); if (rc) return rc;
  }
  c->msgs_valid = false;
  return 0;
}

extern "C" int pepo_init_ex(pepo_ctx** out, int Lx, int Ly, int cx, int cy, double J, double h,
                            double dt, int chi_max, double bp_tol, double bp_damping,
                            void* d_arena, size_t arena_bytes, void* stream, int max_inflight,
                            int bond_pauli, int field_pauli, int obs_pauli) {
  if (!out) { set_error("init: out is NULL"); return -1; }
  *out = nullptr;
  if (chi_max > 256) {
    set_error("init: chi_max %d > 256 is not supported (the BP kernels hold a message in 256 lanes x 8 registers)", chi_max);
    return -1;
  }
  if (Lx < 1 || Ly < 1 || cx < 0 || cx >= Lx || cy < 0 || cy >= Ly || chi_max < 1 ||
      !(dt > 0.0) || bond_pauli < 1 || bond_pauli > 3 || field_pauli < 1 || field_pauli > 3 ||
      obs_pauli < 1 || obs_pauli > 3 || bp_damping < 0.0 || bp_damping >= 1.0 || !d_arena) {
    set_error("init: bad argument (grid %dx%d centre (%d,%d) chi_max %d dt %g)", Lx, Ly, cx, cy, chi_max, dt);
    return -1;
  }
  pepo_ctx* c = new pepo_ctx();
  c->Lx = Lx; c->Ly = Ly; c->cx = cx; c->cy = cy; c->center = cy * Lx + cx;
  c->J = J; c->h = h; c->dt = dt; c->bp_tol = bp_tol; c->bp_damping = bp_damping;
  c->chi_max = chi_max; c->bondP = bond_pauli; c->fieldP = field_pauli; c->obsP = obs_pauli;
  c->st = (cudaStream_t)stream;
  build_lattice(Lx, Ly, c->sites, c->bonds, c->classes, c->n_hb);
  c->n_sites = Lx * Ly; c->n_bonds = (int)c->bonds.size();
  c->chi.assign(c->n_bonds, 1);
  // gate tables: field PTM, bond PTM and its operator-Schmidt decomposition
  ptm_one_site(h * dt, field_pauli, c->G1);
  ptm_one_site(0.5 * h * dt, field_pauli, c->G1h);     // same sparsity pattern as G1
  c->f_row_mask = 0; c->f_col_mask = 0;
  for (int q = 0; q < 4; q++) {
    bool ident = true;
    for (int p = 0; p < 4; p++) if (std::fabs(c->G1[q * 4 + p] - (p == q ? 1.0 : 0.0)) > 0.0) ident = false;
    if (!ident) {
      c->f_row_mask |= 1 << q;
      for (int p = 0; p < 4; p++) if (c->G1[q * 4 + p] != 0.0) c->f_col_mask |= 1 << p;
    }
  }
  double G2[256];
  ptm_two_site(J * dt, bond_pauli, G2);
  // T[(p1',p1),(p2',p2)] = G2[(p1'p2'),(p1p2)], column-major 16x16
  double Tm[256], U[256], S[16], V[256];
  for (int a1 = 0; a1 < 4; a1++) for (int a2 = 0; a2 < 4; a2++) for (int b1 = 0; b1 < 4; b1++) for (int b2 = 0; b2 < 4; b2++)
    Tm[(a1 * 4 + b1) + 16 * (a2 * 4 + b2)] = G2[(a1 * 4 + a2) * 16 + (b1 * 4 + b2)];
  host_svd16(Tm, U, S, V);
  int NA = 0;
  for (int a = 0; a < 16; a++) if (S[a] > 1e-13 * S[0]) NA = a + 1;
  if (NA > 4) { set_error("init: gate with operator-Schmidt rank %d > 4 unsupported", NA); delete c; return -1; }
  c->NA = 4;     // fixed layout (N = 4 chi); unused components get sigma = 0
  std::vector<double> Ahat[2], Gam[2], sig(4, 0.0);
  for (int i = 0; i < 2; i++) {
    const double* F = i == 0 ? U : V;
    Ahat[i].assign(4 * 16, 0.0);
    for (int a = 0; a < NA; a++)
      for (int pp = 0; pp < 4; pp++) for (int p = 0; p < 4; p++) Ahat[i][(a * 4 + pp) * 4 + p] = F[a * 16 + (pp * 4 + p)];
    // unused components: keep an orthonormal completion so that the dressed Gram stays SPD
    for (int a = NA; a < 4; a++)
      for (int pp = 0; pp < 4; pp++) for (int p = 0; p < 4; p++) Ahat[i][(a * 4 + pp) * 4 + p] = F[a * 16 + (pp * 4 + p)];
    Gam[i].assign(4 * 4 * 16, 0.0);
    for (int a = 0; a < 4; a++) for (int a2 = 0; a2 < 4; a2++) for (int p = 0; p < 4; p++) for (int q = 0; q < 4; q++) {
      double s = 0;
      for (int pp = 0; pp < 4; pp++) s += Ahat[i][(a * 4 + pp) * 4 + p] * Ahat[i][(a2 * 4 + pp) * 4 + q];
      Gam[i][((a * 4 + a2) * 4 + p) * 4 + q] = s;
    }
  }
  for (int a = 0; a < NA; a++) sig[a] = S[a];
  // workspace sizing
  c->B = max_inflight > 0 ? std::min(max_inflight, PEPO_MAXT / 2) : default_inflight(Lx, Ly, chi_max, 4);
  size_t top;
  c->model_bytes = model_bytes_for(Lx, Ly, chi_max, c->B, 4, &top);
  size_t need = top + 256;
  if (arena_bytes < need) {
    set_error("init: arena too small: %zu bytes given, %zu needed", arena_bytes, need);
    delete c; return -2;
  }
  size_t mis = (size_t)((uintptr_t)d_arena & 255);
  c->arena.base = (char*)d_arena + (mis ? 256 - mis : 0);
  c->arena.size = arena_bytes;
  layout(c);
  // pinned host buffers
  if (cudaMallocHost((void**)&c->h_ints, (size_t)c->B * 4 * 4 + 16) != cudaSuccess ||
      cudaMallocHost((void**)&c->h_dbls, (size_t)c->B * 2 * 8 + 16) != cudaSuccess ||
      cudaMallocHost((void**)&c->h_chi_msg, (size_t)2 * c->n_bonds * 4 + 16) != cudaSuccess ||
      cudaMallocHost((void**)&c->h_scal, 64) != cudaSuccess ||
      cudaMallocHost((void**)&c->h_delta, 8 * BP_GROUP + 16) != cudaSuccess ||
      cudaMallocHost((void**)&c->h_bpints, 16) != cudaSuccess) {
    set_error("init: cudaMallocHost failed"); pepo_destroy(c); return -3;
  }
  {
    int lo = 0, hi = 0;
    cudaDeviceGetStreamPriorityRange(&lo, &hi);          // hi = numerically smallest = highest priority
    // priorities: Jacobi kernels highest (they need whole SMs as soon as some are free), then the
    // first piece stream, then the second: when both piece streams hold GEMM work the first one is
    // served first, which re-creates the half-period skew between them after every join
    bool ok = true;
    for (int i = 0; i < pepo_ctx::NSMAX && ok; i++) {
      const int pr = std::min(lo, hi + 1 + i);           // descending priority, all below the Jacobi streams
      ok = cudaStreamCreateWithPriority(&c->ps[i], cudaStreamNonBlocking, pr) == cudaSuccess &&
           cudaStreamCreateWithPriority(&c->hp[i], cudaStreamNonBlocking, hi) == cudaSuccess;
    }
    for (int i = 0; i < 5 * pepo_ctx::NSMAX + 1 && ok; i++) ok = cudaEventCreateWithFlags(&c->pev[i], cudaEventDisableTiming) == cudaSuccess;
    if (!ok) { set_error("init: stream / event creation failed"); pepo_destroy(c); return -3; }
  }
  {
    bool ok = cudaStreamCreateWithFlags(&c->copy_st, cudaStreamNonBlocking) == cudaSuccess &&
              cudaEventCreateWithFlags(&c->copy_ev, cudaEventDisableTiming) == cudaSuccess;
    c->site_ev.assign(c->n_sites, nullptr);
    for (int v = 0; v < c->n_sites && ok; v++) ok = cudaEventCreateWithFlags(&c->site_ev[v], cudaEventDisableTiming) == cudaSuccess;
    if (!ok) { set_error("init: stream / event creation failed"); pepo_destroy(c); return -3; }
    c->site_pending.assign(c->n_sites, 0);
    c->field_todo.assign(c->n_sites, 0);
  }
  c->cur_st = c->st;
  int rc = 0;
  for (size_t g : c->arena.guards)
    if (cudaMemsetAsync(c->arena.base + g, 0xA5, 64, c->st) != cudaSuccess) { set_error("init: guard fill failed"); pepo_destroy(c); return -3; }
  double one = 1.0;
  rc |= upload(c, c->ones, &one, 8);
  rc |= upload(c, c->dG1, c->G1, 128);
  for (int i = 0; i < 2; i++) {
    rc |= upload(c, c->dGamma[i], Gam[i].data(), Gam[i].size() * 8);
    rc |= upload(c, c->dAhat[i], Ahat[i].data(), Ahat[i].size() * 8);
  }
  rc |= upload(c, c->dSigma, sig.data(), 32);
  if (!rc) rc = reset_state(c);
  if (rc) { pepo_destroy(c); return -3; }
  memset(&c->stats, 0, sizeof(c->stats));
  c->stats.min_cut_gap = 1.0;
  c->launches = 0;
  *out = c;
  return 0;
}

extern "C" int pepo_init(pepo_ctx** out, int Lx, int Ly, int cx, int cy, double J, double h,
                         double dt, int chi_max, double bp_tol, double bp_damping, void* d_arena,
                         size_t arena_bytes, void* stream) {
  return pepo_init_ex(out, Lx, Ly, cx, cy, J, h, dt, chi_max, bp_tol, bp_damping, d_arena,
                      arena_bytes, stream, 0, 3, 1, 3);
}

extern "C" int pepo_destroy(pepo_ctx* c) {
  if (!c) return 0;
  cudaStreamSynchronize(c->st);
  for (auto& e : c->prof.ev) if (e) cudaEventDestroy(e);
  for (int i = 0; i < pepo_ctx::NSMAX; i++) {
    if (c->ps[i]) { cudaStreamSynchronize(c->ps[i]); cudaStreamDestroy(c->ps[i]); }
    if (c->hp[i]) { cudaStreamSynchronize(c->hp[i]); cudaStreamDestroy(c->hp[i]); }
  }
  for (int i = 0; i < 5 * pepo_ctx::NSMAX + 1; i++) if (c->pev[i]) cudaEventDestroy(c->pev[i]);
  for (auto e : c->done_ev) cudaEventDestroy(e);
  if (c->copy_st) { cudaStreamSynchronize(c->copy_st); cudaStreamDestroy(c->copy_st); }
  for (auto e : c->site_ev) if (e) cudaEventDestroy(e);
  if (c->copy_ev) cudaEventDestroy(c->copy_ev);
  cudaFreeHost(c->h_ints); cudaFreeHost(c->h_dbls); cudaFreeHost(c->h_chi_msg);
  cudaFreeHost(c->h_scal); cudaFreeHost(c->h_delta); cudaFreeHost(c->h_bpints);
  delete c;
  return 0;
}

extern "C" int pepo_set_option(pepo_ctx* c, const char* key, double v) {
  if (!c || !key) { set_error("set_option: NULL"); return -1; }
  std::string k(key);
  if (k == "eps_cut") c->eps_cut = v;
  else if (k == "bp_max_sweeps") c->bp_max_sweeps = (int)v;
  else if (k == "bp_max_sweeps_damped") c->bp_max_sweeps_damped = (int)v;
  else if (k == "chol_min_ratio") c->chol_ratio = v;
  else if (k == "chol_tau") c->chol_tau = v;
  else if (k == "force_householder") c->force_hh = (int)v;
  else if (k == "direct_gemm") c->direct = (int)v;
  else if (k == "jacobi_tol") c->jacobi_tol = v;
  else if (k == "jacobi_max_sweeps") c->jacobi_max_sweeps = (int)v;
  else if (k == "svd_precond_min") c->svd_precond_min = (int)v;
  else if (k == "jacobi_early") c->jacobi_early = v < 0.0 ? 0.0 : v;
  else if (k == "svd_deflate") c->svd_deflate = v < 0.0 ? 0.0 : v;
  else if (k == "svd_orient") c->svd_orient = v < 0.5 ? 0 : v < 1.5 ? 1 : 2;
  else if (k == "bp_group") c->bp_group = (int)v;
  else if (k == "bp_ladder") c->bp_ladder = (int)v;
  else if (k == "bp_init") c->bp_init = (int)v;
  else if (k == "env") c->env_mode = (int)v ? 1 : 0;
  else if (k == "psqrt_eps") c->psqrt_eps = v;
  else if (k == "observe_ref_C") c->obs_prev_C = v;            // reference of pepo_observe's drop test (e.g. after a restart)
  else if (k == "observe_ref_gate_err") c->obs_prev_gerr = v;
  else if (k == "bp_damping2") { if (!(v >= 0.0 && v < 1.0)) { set_error("set_option: bp_damping2 must be in [0,1)"); return -1; } c->bp_damping2 = v; }
  else if (k == "trotter_order") {
    if ((int)v != 1 && (int)v != 2) { set_error("set_option: trotter_order must be 1 or 2"); return -1; }
    c->trotter_order = (int)v;
  }
  else if (k == "pipeline") c->pipeline = (int)v;
  else if (k == "trace") c->prof.trace = (int)v;
  else if (k == "profile") {
    Prof& P = c->prof;
    if (v != 0.0 && P.ev.empty()) {
      P.ev.resize(2 * 4096); P.cat.assign(4096, 0); P.strm.assign(4096, 0);
      for (auto& e : P.ev) if (cudaEventCreate(&e) != cudaSuccess) { set_error("profile: cudaEventCreate failed"); return -3; }
    }
    cudaStreamSynchronize(c->st); prof_flush(c);
    P.on = (v != 0.0);
    if (v == 2.0) for (int i = 0; i < PC_COUNT; i++) { P.ms[i] = P.flops[i] = P.bytes[i] = 0; P.cnt[i] = 0; }
  }
  else if (k == "bp_tol") c->bp_tol = v;
  else if (k == "bp_damping") c->bp_damping = v;
  else { set_error("set_option: unknown key %s", key); return -1; }
  return 0;
}

// ============================================================================================
// state access
// ============================================================================================
static size_t site_live_size(const pepo_ctx* c, int v) {
  size_t n = 4;
  const SiteInfo& s = c->sites[v];
  for (int l = 0; l < s.nlegs; l++) n *= c->chi[s.leg_bond[l]];
  return n;
}
extern "C" int pepo_n_bonds(pepo_ctx* c) { return c ? c->n_bonds : -1; }
extern "C" int pepo_get_bond_dims(pepo_ctx* c, int* h_chi) {
  if (!c || !h_chi) { set_error("get_bond_dims: NULL"); return -1; }
  for (int e = 0; e < c->n_bonds; e++) h_chi[e] = c->chi[e];
  return 0;
}
extern "C" int pepo_set_bond_dims(pepo_ctx* c, const int* h_chi) {
  if (!c || !h_chi) { set_error("set_bond_dims: NULL"); return -1; }
  { int rcw = wait_pending_uploads(c, c->st); if (rcw) return rcw; }
  for (int e = 0; e < c->n_bonds; e++)
    if (h_chi[e] < 1 || h_chi[e] > c->chi_max) { set_error("set_bond_dims: chi[%d]=%d out of range", e, h_chi[e]); return -1; }
  for (int e = 0; e < c->n_bonds; e++) c->chi[e] = h_chi[e];
  c->msgs_valid = false; c->n_valid = false; c->n_sqrt_valid = false;
  return 0;
}
extern "C" size_t pepo_site_size(pepo_ctx* c, int x, int y) {
  if (!c || x < 0 || x >= c->Lx || y < 0 || y >= c->Ly) return 0;
  return site_live_size(c, y * c->Lx + x);
}
extern "C" double* pepo_site_ptr(pepo_ctx* c, int x, int y) {
  if (!c || x < 0 || x >= c->Lx || y < 0 || y >= c->Ly) return nullptr;
  return c->sites[y * c->Lx + x].psi;
}
extern "C" int pepo_get_site(pepo_ctx* c, int x, int y, double* h_dst, size_t n) {
  if (!c || !h_dst || x < 0 || x >= c->Lx || y < 0 || y >= c->Ly) { set_error("get_site: bad argument"); return -1; }
  { int rcw = wait_pending_uploads(c, c->st); if (rcw) return rcw; }
  int v = y * c->Lx + x;
  if (n != site_live_size(c, v)) { set_error("get_site: size %zu != live size %zu", n, site_live_size(c, v)); return -1; }
  PEPO_CUDA_OK(cudaMemcpyAsync(h_dst, c->sites[v].psi, n * 8, cudaMemcpyDeviceToHost, c->st));
  PEPO_CUDA_OK(cudaStreamSynchronize(c->st));
  return 0;
}
namespace {
// every pending asynchronous site upload becomes visible to `st` (and stops being pending)
int wait_pending_uploads(pepo_ctx* c, cudaStream_t st) {
  if (c->n_pending == 0) { c->copy_forked = false; return 0; }
  for (int v = 0; v < c->n_sites; v++) {
    if (!c->site_pending[v]) continue;
    PEPO_CUDA_OK(cudaStreamWaitEvent(st, c->site_ev[v], 0));
    c->site_pending[v] = 0;
  }
  c->n_pending = 0;
  c->copy_forked = false;
  return 0;
}
}  // namespace

// Asynchronous pepo_set_site: the copy is queued on an internal copy stream and the call returns;
// h_src (pinned memory for a truly asynchronous copy) must stay valid and unchanged until the next
// call that returns a host value (bp_converge, correlation, getters) or pepo_trotter_step has
// returned.  The next pepo_trotter_step starts on the sites already uploaded while the others are
// still in flight (the field gate and the first bond gate of a site wait for that site only).
extern "C" int pepo_set_site_async(pepo_ctx* c, int x, int y, const double* h_src, size_t n) {
  if (!c || !h_src || x < 0 || x >= c->Lx || y < 0 || y >= c->Ly) { set_error("set_site_async: bad argument"); return -1; }
  const int v = y * c->Lx + x;
  if (n != site_live_size(c, v)) { set_error("set_site_async: size %zu != live size %zu", n, site_live_size(c, v)); return -1; }
  if (!c->copy_forked) {
    // the slot may still be read by kernels queued on the context stream (BP of the previous step)
    PEPO_CUDA_OK(cudaEventRecord(c->copy_ev, c->st));
    PEPO_CUDA_OK(cudaStreamWaitEvent(c->copy_st, c->copy_ev, 0));
    c->copy_forked = true;
  }
  PEPO_CUDA_OK(cudaMemcpyAsync(c->sites[v].psi, h_src, n * 8, cudaMemcpyHostToDevice, c->copy_st));
  PEPO_CUDA_OK(cudaEventRecord(c->site_ev[v], c->copy_st));
  if (!c->site_pending[v]) { c->site_pending[v] = 1; c->n_pending++; }
  c->msgs_valid = false;
  return 0;
}

extern "C" int pepo_set_site(pepo_ctx* c, int x, int y, const double* h_src, size_t n) {
  if (!c || !h_src || x < 0 || x >= c->Lx || y < 0 || y >= c->Ly) { set_error("set_site: bad argument"); return -1; }
  { int rcw = wait_pending_uploads(c, c->st); if (rcw) return rcw; }
  int v = y * c->Lx + x;
  if (n != site_live_size(c, v)) { set_error("set_site: size %zu != live size %zu", n, site_live_size(c, v)); return -1; }
  c->msgs_valid = false;
  return upload(c, c->sites[v].psi, h_src, n * 8);
}
extern "C" int pepo_get_lambda(pepo_ctx* c, int bond, double* h_dst, int n) {
  if (!c || !h_dst || bond < 0 || bond >= c->n_bonds || n != c->chi[bond]) { set_error("get_lambda: bad argument"); return -1; }
  PEPO_CUDA_OK(cudaMemcpyAsync(h_dst, bond_vec(c->lambda, bond, c->chi_max), n * 8, cudaMemcpyDeviceToHost, c->st));
  PEPO_CUDA_OK(cudaStreamSynchronize(c->st));
  return 0;
}
extern "C" int pepo_set_lambda(pepo_ctx* c, int bond, const double* h_src, int n) {
  if (!c || !h_src || bond < 0 || bond >= c->n_bonds || n != c->chi[bond]) { set_error("set_lambda: bad argument"); return -1; }
  std::vector<double> sq(n), isq(n);
  for (int i = 0; i < n; i++) {
    if (!(h_src[i] > 0.0)) { set_error("set_lambda: non-positive entry"); return -1; }
    sq[i] = std::sqrt(h_src[i]); isq[i] = 1.0 / sq[i];
  }
  c->n_valid = false; c->n_sqrt_valid = false;
  int rc = upload(c, bond_vec(c->lambda, bond, c->chi_max), h_src, n * 8);
  rc |= upload(c, bond_vec(c->sqrt_l, bond, c->chi_max), sq.data(), n * 8);
  rc |= upload(c, bond_vec(c->isqrt_l, bond, c->chi_max), isq.data(), n * 8);
  return rc ? -3 : 0;
}

extern "C" int pepo_get_stats(pepo_ctx* c, pepo_stats* s) {
  if (!c || !s) { set_error("get_stats: NULL"); return -1; }
  c->stats.kernel_launches = c->launches;
  c->stats.arena_high_water = c->arena.top;
  c->stats.arena_model_bytes = c->model_bytes;
  c->stats.max_inflight_gates = c->B;
  int m = 1;
  for (int e = 0; e < c->n_bonds; e++) m = std::max(m, c->chi[e]);
  c->stats.chi_max_live = m;
  *s = c->stats;
  return 0;
}

// ============================================================================================
// Trotter step
// ============================================================================================
namespace {
int apply_field_impl(pepo_ctx* c, bool half);
}
extern "C" int pepo_apply_field(pepo_ctx* c) {
  if (!c) { set_error("apply_field: NULL"); return -1; }
  CtxScope scope(c);
  return apply_field_impl(c, false);
}
namespace {
int apply_field_impl(pepo_ctx* c, bool half) {
  { int rcw = wait_pending_uploads(c, c->st); if (rcw) return rcw; }
  if (c->f_row_mask == 0) return 0;
  for (int v0 = 0; v0 < c->n_sites; v0 += PEPO_BP_MAXS) {
    FieldBatch fb;
    fb.count = std::min(PEPO_BP_MAXS, c->n_sites - v0);
    for (int i = 0; i < fb.count; i++) {
      fb.psi[i] = c->sites[v0 + i].psi;
      fb.slab[i] = (long long)(site_live_size(c, v0 + i) / 4);
    }
    memcpy(fb.G, half ? c->G1h : c->G1, sizeof(fb.G));
    fb.row_mask = c->f_row_mask; fb.col_mask = c->f_col_mask;
    double fbytes = 0; for (int i = 0; i < fb.count; i++) fbytes += 8.0 * fb.slab[i] * 2 * __builtin_popcount(fb.row_mask);
    ProfScope ps(c, PC_FIELD, 0, fbytes);
    int rc = launch_field_gate(c->st, fb);
    if (rc) return rc;
  }
  c->msgs_valid = false;
  return 0;
}
}  // namespace

namespace {

struct TaskGeo {           // one site of one gate
  int v, lane, slot, site_idx;     // site_idx: 0 = v1 (first Schmidt factor), 1 = v2
  int nlegs, cut_leg;
  int dims[5];             // live dims incl. Pauli
  int env_legs[3], n_env;
  long long m, ld;
  int n, chi_c, N, k, r;   // k = min(m,n); r = rows of Rx
  bool chol;
  bool direct;             // Cholesky path: the reconstruction reads psi in place and writes the site slot
  bool direct_gram;        // ... and so does the Gram kernel (no explicit cv at all)
  SiteView view;
  bool skip1, skip2;       // Householder path: Q = I when m <= n (R = cv); Qx = I when 4k <= N (Rx = X)
  int chi_new;
};

struct BatchState {        // one batch of gates moving through the three phases of Algorithm 1
  std::vector<int> gate_bonds;
  std::vector<TaskGeo> T;
  int ng = 0, lane0 = 0;           // lanes [lane0, lane0 + ng) of the workspace
  cudaStream_t st = nullptr;       // stream of this batch
  cudaStream_t hp = nullptr;       // high-priority stream for the Jacobi kernel (nullptr: st)
  cudaEvent_t ev[2] = {nullptr, nullptr};
  bool piped = false;              // another batch is in flight: keep the profiling events until the class ends
  bool have_chol = false;
  SvdFinishBatch fb;
};

int msg_index(const pepo_ctx* c, int v, int dir, bool outgoing);
int leg_apply(pepo_ctx* c, cudaStream_t st, const double* src, const int* dims, int nlegs, int leg,
              const double* Mat, int d_new, double* Wbuf, double* dst);
inline bool matrix_env(const pepo_ctx* c) { return c->env_mode == 1 && c->n_valid && c->n_sqrt_valid; }

// a2-a4 fused: cv = permute(psi * sqrt(lambda_env)) into the lane's work matrix (explicit path).
// Matrix environment (NEXT-1, option "env" = 1): the absorb is a chi x chi GEMM per environment leg with
// the PSEUDO_SQRT of the incoming matrix message, then a plain permutation.
int enqueue_permute_in(pepo_ctx* c, cudaStream_t st, const TaskGeo& t) {
  const SiteInfo& s = c->sites[t.v];
  SiteWs& W = c->lanes[t.lane].s[t.slot];
  const double* psrc = s.psi;
  const bool menv = matrix_env(c);
  if (menv && t.n_env > 0) {
    const double* src = s.psi;
    for (int j = 0; j < t.n_env; j++) {
      const int l = t.env_legs[j];
      double* dst = ((t.n_env - 1 - j) % 2 == 0) ? W.out : W.cv;         // the last one lands in W.out
      const double* Smat = c->nS + (size_t)msg_index(c, t.v, s.leg_dir[l], false) * c->chi_max * c->chi_max;
      int rc = leg_apply(c, st, src, t.dims, s.nlegs, l, Smat, t.dims[l], W.W, dst); if (rc) return rc;
      src = dst;
    }
    psrc = src;
  }
  PermuteDesc pd;
  pd.rank = s.nlegs + 1; pd.power = 1.0;
  long long sstr = 1;
  for (int l = 0; l <= s.nlegs; l++) { pd.shape[l] = t.dims[l]; pd.src_stride[l] = sstr; sstr *= t.dims[l]; pd.scale[l] = nullptr; }
  long long dstr = 1;
  for (int j = 0; j < t.n_env; j++) {
    int l = t.env_legs[j];
    pd.perm[j] = l; pd.dst_stride[j] = dstr; dstr *= t.dims[l];
    pd.scale[l] = menv ? nullptr : bond_vec(c->sqrt_l, s.leg_bond[l], c->chi_max);
  }
  pd.perm[t.n_env] = t.cut_leg; pd.dst_stride[t.n_env] = t.ld;
  pd.perm[t.n_env + 1] = s.nlegs; pd.dst_stride[t.n_env + 1] = t.ld * t.chi_c;
  ProfScope ps(c, PC_PERMUTE, 0, 16.0 * t.m * t.n);
  return launch_permute(st, psrc, W.cv, pd);
}

// phase 1: absorb + permute, Gram, dressing, Cholesky (enqueue only; ends with the flag read-back)
int batch_p1(pepo_ctx* c, BatchState& S) {
  const int ng = S.ng;
  cudaStream_t st = S.st;
  std::vector<TaskGeo>& T = S.T;
  const std::vector<int>& gate_bonds = S.gate_bonds;
  const int NA = c->NA;
  GateTables gt;
  gt.Gamma[0] = c->dGamma[0]; gt.Gamma[1] = c->dGamma[1];
  gt.Ahat[0] = c->dAhat[0]; gt.Ahat[1] = c->dAhat[1];
  gt.sigma = c->dSigma;
  c->cur_st = st;
  (void)gate_bonds; (void)gt; (void)NA;
  T.assign(2 * ng, TaskGeo());
  // ---- A: geometry + absorb/permute ----------------------------------------------------------
  for (int g = 0; g < ng; g++) {
    const BondInfo& b = c->bonds[gate_bonds[g]];
    for (int i = 0; i < 2; i++) {
      TaskGeo& t = T[2 * g + i];
      t.v = i == 0 ? b.v1 : b.v2;
      const int dcut = i == 0 ? b.d1 : b.d2;
      t.lane = S.lane0 + g; t.slot = i; t.site_idx = i;
      const SiteInfo& s = c->sites[t.v];
      t.nlegs = s.nlegs; t.n_env = 0; t.m = 1; t.cut_leg = -1;
      for (int l = 0; l < s.nlegs; l++) {
        t.dims[l] = c->chi[s.leg_bond[l]];
        if (s.leg_dir[l] == dcut) t.cut_leg = l;
        else { t.env_legs[t.n_env++] = l; t.m *= t.dims[l]; }
      }
      t.dims[s.nlegs] = 4;
      t.chi_c = t.dims[t.cut_leg];
      t.n = 4 * t.chi_c; t.N = NA * t.chi_c;
      t.ld = (t.m + 1) & ~1ll;
      t.k = (int)std::min<long long>(t.m, t.n);
      t.chol = !c->force_hh && (double)t.m >= c->chol_ratio * t.n;
      t.r = t.chol ? t.N : std::min(4 * t.k, t.N);
      t.skip1 = t.m <= t.n; t.skip2 = 4 * t.k <= t.N;
      t.direct = t.chol && c->direct && !matrix_env(c);
      t.view.nlegs = s.nlegs; t.view.cut = t.cut_leg;
      for (int l = 0; l < 4; l++) t.view.dims[l] = l < s.nlegs ? t.dims[l] : 1;
      // The Gram kernel reads psi in place when the rows of cv are contiguous runs in psi (cut leg not
      // the fastest one).  With the cut leg fastest its rows are strided by chi_c and the gathered Gram
      // is slower than transpose + plain Gram (measured 0.92 against 0.17 + 0.55 ms at chi = 60), so
      // that case keeps the explicit cv for the Gram and only the reconstruction runs in place.
      long long run = 1;
      for (int l = 0; l < t.cut_leg; l++) run *= t.dims[l];
      t.direct_gram = t.direct && c->direct != 3 && (run >= 2 || c->direct == 2);
      if (t.direct_gram) continue;            // no explicit cv (a3-a5 fused)
      int rc = enqueue_permute_in(c, st, t);
      if (rc) return rc;
    }
  }
  // ---- B: Cholesky path ------------------------------------------------------------------------
  {
    MatBatch pb; pb.count = 0;
    DressBatch db; db.count = 0; db.NA = NA;
    int* infos[PEPO_MAXT];
    for (auto& t : T) {
      if (!t.chol) continue;
      SiteWs& W = c->lanes[t.lane].s[t.slot];
      int ks, kc;
      gram_plan(t.m, t.n, &ks, &kc);
      if (ks > 1 && (size_t)ks * t.n * t.n > c->part_cap) { set_error("gate: split-K workspace too small (%d x %d^2 > %zu)", ks, t.n, c->part_cap); return -3; }
      GemmProb gp;
      gp.A = W.cv; gp.B = W.cv; gp.C = W.C; gp.lda = t.ld; gp.ldb = t.ld; gp.ldc = t.n;
      gp.M = t.n; gp.N = t.n; gp.K = (int)t.m;
      ProfScope ps(c, PC_GRAM, (double)t.m * t.n * (t.n + 1), 8.0 * t.m * t.n);
      int rc;
      if (t.direct_gram) {
        // C = cv^T cv with cv = psi * sqrt(lambda_env): weights lambda on the rows, psi read in place
        const SiteInfo& sv = c->sites[t.v];
        const double* w2[4] = {nullptr, nullptr, nullptr, nullptr};
        for (int l = 0; l < sv.nlegs; l++) if (l != t.cut_leg) w2[l] = bond_vec(c->lambda, sv.leg_bond[l], c->chi_max);
        rc = launch_site_gram(st, sv.psi, t.view, w2, W.C, W.part);
        if (rc) return rc;
      } else {
      rc = launch_dgemm(st, 1, 0, gp, ks, kc, W.part, true);
      if (rc) return rc;
      if (ks > 1) rc = launch_gram_reduce(st, W.part, ks, t.n, W.C, t.n);
      else {
        // single split wrote the upper tiles straight into C: mirror through the same reducer
        rc = launch_gram_reduce(st, W.C, 1, t.n, W.C, t.n);
      }
      if (rc) return rc;
      }
      int q = db.count++;
      db.in[q] = W.C; db.out[q] = W.Rx; db.chi[q] = t.chi_c; db.k[q] = t.n; db.site[q] = t.site_idx;
      db.ld_in[q] = t.n; db.ld_out[q] = t.N;
      int p = pb.count++;
      pb.A[p] = W.Rx; pb.ld[p] = t.N; pb.m[p] = t.N; pb.n[p] = t.N; infos[p] = W.info;
    }
    // the latency-bound small kernels of the gate's critical chain (dressing, POTRF here; the whole
    // of p2; bridges and W in p3) go to the piece's high-priority stream, so that their few CTAs do
    // not queue behind the GEMM / permutation CTAs of the other pieces (seen: POTRF 1.05 ms instead
    // of 0.42, core GEMM 0.4 instead of 0.1)
    cudaStream_t sh = S.hp ? S.hp : st;
    if (sh != st) {
      PEPO_CUDA_OK(cudaEventRecord(S.ev[0], st));
      PEPO_CUDA_OK(cudaStreamWaitEvent(sh, S.ev[0], 0));
      c->cur_st = sh;
    }
    if (db.count) {
      int rc;
      { ProfScope ps(c, PC_DRESS, 0, 0); rc = launch_dress_gram(sh, db, gt); if (rc) return rc; }
      { ProfScope ps(c, PC_CHOL, 0, 0); rc = launch_potrf(sh, pb, infos, c->chol_tau); if (rc) return rc; }
      PEPO_CUDA_OK(cudaMemcpyAsync(c->h_ints + 4 * S.lane0, c->lane_ints + 4 * S.lane0, (size_t)ng * 16, cudaMemcpyDeviceToHost, sh));
      S.have_chol = true;
    }
    c->cur_st = st;
  }
  return 0;
}

// phase 2: Cholesky flags (host), Householder fallback, core, SVD, truncation (ends with the chi_new read-back)
int batch_p2(pepo_ctx* c, BatchState& S) {
  const int ng = S.ng;
  cudaStream_t st = S.hp ? S.hp : S.st;     // p2 is all small kernels + the Jacobi kernel: high-priority stream
  std::vector<TaskGeo>& T = S.T;
  const std::vector<int>& gate_bonds = S.gate_bonds;
  const int NA = c->NA;
  GateTables gt;
  gt.Gamma[0] = c->dGamma[0]; gt.Gamma[1] = c->dGamma[1];
  gt.Ahat[0] = c->dAhat[0]; gt.Ahat[1] = c->dAhat[1];
  gt.sigma = c->dSigma;
  c->cur_st = st;
  (void)gate_bonds; (void)gt; (void)NA;
  if (S.have_chol) {
    PEPO_CUDA_OK(cudaStreamSynchronize(st));
    if (!S.piped) prof_flush(c);
    for (auto& t : T) {
      if (!t.chol) continue;
      int info = c->h_ints[4 * t.lane + 2 + t.slot];
      if (info != 0) {
        t.chol = false; t.r = std::min(4 * t.k, t.N);
        c->stats.n_chol_failed++;
        if (t.direct_gram) {                   // the Householder fallback needs the explicit cv after all
          int rc = enqueue_permute_in(c, st, t);
          if (rc) return rc;
        }
        t.direct = t.direct_gram = false;
      }
    }
  }
  // ---- C: Householder path / finish Cholesky path ----------------------------------------------
  {
    HHBatch h1; h1.count = 0;
    HHBatch h2; h2.count = 0;
    DressBatch dr; dr.count = 0; dr.NA = NA;
    double* Rout1[PEPO_MAXT]; long long ldr1[PEPO_MAXT];
    double* Rout2[PEPO_MAXT]; long long ldr2[PEPO_MAXT];
    MatBatch zl; zl.count = 0;
    MatBatch ti; ti.count = 0;
    for (auto& t : T) {
      SiteWs& W = c->lanes[t.lane].s[t.slot];
      if (t.chol) {
        int q = zl.count++;
        zl.A[q] = W.Rx; zl.ld[q] = t.N; zl.m[q] = t.N; zl.n[q] = t.N;
        ti.A[q] = W.Rxinv; ti.ld[q] = t.N; ti.m[q] = t.N; ti.n[q] = t.N; ti.count = zl.count;
        c->stats.n_cholesky++;
      } else {
        // first factor: cv = Q R (k x n); for m <= n take Q = I, R = cv (any factor with orthonormal Q serves)
        const double* Rsrc = W.Rbuf; long long ldR = t.k;
        if (t.skip1) { Rsrc = W.cv; ldR = t.ld; }
        else {
          int q = h1.count++;
          h1.A[q] = W.cv; h1.lda[q] = t.ld; h1.m[q] = t.m; h1.n[q] = t.n; h1.beta[q] = W.beta1; h1.tau[q] = W.tau1;
          Rout1[q] = W.Rbuf; ldr1[q] = t.k;
        }
        // X = dress(R) (4k x N); when 4k <= N it is already the small factor Rx (Qx = I)
        int q = dr.count++;
        dr.in[q] = Rsrc; dr.chi[q] = t.chi_c; dr.k[q] = t.k; dr.site[q] = t.site_idx; dr.ld_in[q] = ldR;
        if (t.skip2) { dr.out[q] = W.Rx; dr.ld_out[q] = t.r; }
        else {
          dr.out[q] = W.X; dr.ld_out[q] = 4ll * t.k;
          int q2 = h2.count++;
          h2.A[q2] = W.X; h2.lda[q2] = 4ll * t.k; h2.m[q2] = 4ll * t.k; h2.n[q2] = t.N; h2.beta[q2] = W.beta2; h2.tau[q2] = W.tau2;
          Rout2[q2] = W.Rx; ldr2[q2] = t.r;
        }
        c->stats.n_householder++;
      }
    }
    int rc = 0;
    if (zl.count) { ProfScope ps(c, PC_CHOL, 0, 0); rc = launch_zero_lower(st, zl); if (rc) return rc; rc = launch_trtri(st, zl, ti); if (rc) return rc; }
    if (dr.count) {
      ProfScope ps(c, PC_HOUSEHOLDER, 0, 0);
      if (h1.count) {
        rc = launch_hh_factor(st, h1); if (rc) return rc;
        rc = launch_hh_extract_r(st, h1, Rout1, ldr1); if (rc) return rc;
      }
      rc = launch_dress_R(st, dr, gt); if (rc) return rc;
      if (h2.count) {
        rc = launch_hh_factor(st, h2); if (rc) return rc;
        rc = launch_hh_extract_r(st, h2, Rout2, ldr2); if (rc) return rc;
      }
    }
  }
  // ---- D: core, SVD, truncation ------------------------------------------------------------------
  {
    DressBatch sc; sc.count = ng; sc.NA = NA;
    SvdBatch sb; sb.count = ng;
    SvdFinishBatch& fb = S.fb; fb.count = ng; fb.with_v = 0; fb.precond_min = c->svd_precond_min;
    for (int g = 0; g < ng; g++) {
      TaskGeo& t1 = T[2 * g]; TaskGeo& t2 = T[2 * g + 1];
      LaneWs& L = c->lanes[S.lane0 + g];
      const int e = gate_bonds[g];
      sc.in[g] = L.s[0].Rx; sc.out[g] = L.Ks; sc.chi[g] = t1.chi_c; sc.k[g] = t1.r; sc.site[g] = 0;
      sc.ld_in[g] = t1.r; sc.ld_out[g] = t1.r;
      sb.K[g] = L.K; sb.ldk[g] = t1.r; sb.r1[g] = t1.r; sb.r2[g] = t2.r;
      sb.G[g] = L.G; sb.V[g] = L.V; sb.sv[g] = L.sv; sb.order[g] = L.order; sb.sweeps[g] = L.ints + 1;
      sb.orient[g] = L.orient; fb.orient[g] = L.orient;
      fb.K[g] = L.K; fb.ldk[g] = t1.r;
      fb.r1[g] = t1.r; fb.r2[g] = t2.r; fb.G[g] = L.G; fb.V[g] = L.V; fb.sv[g] = L.sv; fb.order[g] = L.order;
      fb.Us[g] = L.Us; fb.ldus[g] = t1.r; fb.Vs[g] = L.Vs; fb.ldvs[g] = t2.r;
      fb.lambda[g] = bond_vec(c->lambda, e, c->chi_max);
      fb.sqrt_l[g] = bond_vec(c->sqrt_l, e, c->chi_max);
      fb.isqrt_l[g] = bond_vec(c->isqrt_l, e, c->chi_max);
      fb.chi_new[g] = L.ints; fb.gate_stats[g] = L.dbls;
    }
    int rc = launch_scale_sigma(st, sc, gt); if (rc) return rc;
    for (int g = 0; g < ng; g++) {
      TaskGeo& t1 = T[2 * g]; TaskGeo& t2 = T[2 * g + 1];
      LaneWs& L = c->lanes[S.lane0 + g];
      GemmProb gp;
      gp.A = L.Ks; gp.lda = t1.r; gp.B = L.s[1].Rx; gp.ldb = t2.r; gp.C = L.K; gp.ldc = t1.r;
      gp.M = t1.r; gp.N = t2.r; gp.K = t1.N;
      ProfScope ps(c, PC_SMALL_GEMM, 2.0 * t1.r * t2.r * t1.N, 0);
      rc = launch_dgemm(st, 0, 1, gp, 1, 0, nullptr, false); if (rc) return rc;
    }
    {
      // the Jacobi kernel needs whole SMs (a cluster per core): on the pipelined schedule it goes to
      // a high-priority stream so that it is placed ahead of the other half-batch's GEMM CTAs
      {
        ProfScope ps(c, PC_SVD, 0, 0);
        rc = launch_svd_jacobi(st, sb, c->jacobi_tol, c->jacobi_max_sweeps, false, c->svd_precond_min, c->jacobi_early,
                               c->chi_max, c->svd_deflate, c->svd_orient);
        if (rc) return rc;
      }
      ProfScope ps(c, PC_SVD, 0, 0);
      rc = launch_svd_truncate(st, fb, c->chi_max, c->eps_cut); if (rc) return rc;
    }
    PEPO_CUDA_OK(cudaMemcpyAsync(c->h_ints + 4 * S.lane0, c->lane_ints + 4 * S.lane0, (size_t)ng * 16, cudaMemcpyDeviceToHost, st));
    PEPO_CUDA_OK(cudaMemcpyAsync(c->h_dbls + 2 * S.lane0, c->lane_dbls + 2 * S.lane0, (size_t)ng * 16, cudaMemcpyDeviceToHost, st));
  }
  return 0;
}

// phase 3: chi_new (host), bridges, reconstruction, inverse permute + de-absorb + write-back
int batch_p3(pepo_ctx* c, BatchState& S) {
  const int ng = S.ng;
  cudaStream_t st = S.st;
  cudaStream_t sh = S.hp ? S.hp : st;       // small kernels of the chain (see batch_p1)
  std::vector<TaskGeo>& T = S.T;
  const std::vector<int>& gate_bonds = S.gate_bonds;
  const int NA = c->NA;
  GateTables gt;
  gt.Gamma[0] = c->dGamma[0]; gt.Gamma[1] = c->dGamma[1];
  gt.Ahat[0] = c->dAhat[0]; gt.Ahat[1] = c->dAhat[1];
  gt.sigma = c->dSigma;
  c->cur_st = sh;
  (void)gate_bonds; (void)gt; (void)NA;
  {
    SvdFinishBatch& fb = S.fb;
    int rc = 0;
    PEPO_CUDA_OK(cudaStreamSynchronize(sh));
    if (!S.piped) prof_flush(c);
    int chi_cap = 1;
    for (int g = 0; g < ng; g++) {
      int cn = c->h_ints[4 * (S.lane0 + g)];
      if (cn < 1) {
        // diagnostics: leading entries of the core and of the computed spectrum
        double hk[4] = {0, 0, 0, 0}, hs[2] = {0, 0};
        const int r1 = T[2 * g].r, r2 = T[2 * g + 1].r;
        cudaMemcpy(hk, c->lanes[S.lane0 + g].K, sizeof(double) * std::min(4, r1 * r2), cudaMemcpyDeviceToHost);
        cudaMemcpy(hs, c->lanes[S.lane0 + g].sv, sizeof(double) * std::min(2, std::min(r1, r2)), cudaMemcpyDeviceToHost);
        set_error("gate on bond %d: s0 = 0 or NaN in the core SVD (core %d x %d, K[0..3] = %g %g %g %g, s[0..1] = %g %g, "
                  "sweeps %d)", gate_bonds[g], r1, r2, hk[0], hk[1], hk[2], hk[3], hs[0], hs[1], c->h_ints[4 * (S.lane0 + g) + 1]);
        return -4;
      }
      T[2 * g].chi_new = T[2 * g + 1].chi_new = cn;
      chi_cap = std::max(chi_cap, cn);
      c->stats.jacobi_sweeps += c->h_ints[4 * (S.lane0 + g) + 1];
      if (c->prof.trace) fprintf(stderr, "SWEEPS bond %d core %dx%d sweeps %d\n", gate_bonds[g], T[2 * g].r, T[2 * g + 1].r, c->h_ints[4 * (S.lane0 + g) + 1]);
      if (c->prof.on) {
        // algorithmic flops of the one-sided Jacobi iteration: per sweep Nc(Nc-1)/2 pairs, each
        // 3 inner products (6 L flop) + one plane rotation of two L-vectors (6 L flop)
        const double Nc = std::min(T[2 * g].r, T[2 * g + 1].r), Mx = std::max(T[2 * g].r, T[2 * g + 1].r);
        const double Lc = (c->svd_precond_min > 0 && Nc >= c->svd_precond_min) ? Nc : Mx;
        c->prof.flops[PC_SVD] += c->h_ints[4 * (S.lane0 + g) + 1] * 0.5 * Nc * (Nc - 1) * 12.0 * Lc;
      }
      c->stats.gate_err += c->h_dbls[2 * (S.lane0 + g)];
      c->stats.min_cut_gap = std::min(c->stats.min_cut_gap, c->h_dbls[2 * (S.lane0 + g) + 1]);
    }
    rc = launch_svd_bridge(sh, fb, chi_cap); if (rc) return rc;
  }
  // ---- E: bridge + reconstruction ------------------------------------------------------------------
  {
    DressBatch bw; bw.count = 0; bw.NA = NA;
    int* cn_w[PEPO_MAXT];
    HHApplyBatch a2; a2.count = 0;
    DressBatch rs; rs.count = 0; rs.NA = NA;
    int* cn_r[PEPO_MAXT]; long long mrows[PEPO_MAXT];
    HHApplyBatch a1; a1.count = 0;
    HHApplyBatch pad; pad.count = 0;
    MatBatch padsrc; padsrc.count = 0;
    int rc = 0;
    for (auto& t : T) {
      SiteWs& W = c->lanes[t.lane].s[t.slot];
      LaneWs& L = c->lanes[t.lane];
      const double* UV = t.slot == 0 ? L.Us : L.Vs;
      if (t.chol) {
        // T = Rx^-1 (U sqrt S)   (N x chi_new)
        GemmProb gp;
        gp.A = W.Rxinv; gp.lda = t.N; gp.B = UV; gp.ldb = t.r; gp.C = W.T; gp.ldc = t.N;
        gp.M = t.N; gp.N = t.chi_new; gp.K = t.N;
        { ProfScope ps(c, PC_SMALL_GEMM, 2.0 * t.N * t.N * t.chi_new, 0);
          rc = launch_dgemm(sh, 0, 0, gp, 1, 0, nullptr, false); if (rc) return rc; }
        int q = bw.count++;
        bw.in[q] = W.T; bw.out[q] = W.W; bw.chi[q] = t.chi_c; bw.k[q] = t.chi_new; bw.site[q] = t.site_idx;
        bw.ld_in[q] = t.N; bw.ld_out[q] = t.n; cn_w[q] = L.ints;
      } else {
        // Mx = Qx [U sqrt S ; 0] (4k x chi_new); Qx = I when 4k <= N (then r = 4k: plain copy)
        int qp = padsrc.count++;
        padsrc.A[qp] = const_cast<double*>(UV); padsrc.ld[qp] = t.r; padsrc.m[qp] = t.r; padsrc.n[qp] = t.chi_new;
        pad.Y[qp] = W.Mx; pad.ldy[qp] = 4ll * t.k; pad.m[qp] = 4ll * t.k; pad.ncols[qp] = t.chi_new; pad.count = padsrc.count;
        if (!t.skip2) {
          int q = a2.count++;
          a2.A[q] = W.X; a2.lda[q] = 4ll * t.k; a2.m[q] = 4ll * t.k; a2.k[q] = t.r;
          a2.beta[q] = W.beta2; a2.tau[q] = W.tau2; a2.Y[q] = W.Mx; a2.ldy[q] = 4ll * t.k; a2.ncols[q] = t.chi_new;
        }
        int qr = rs.count++;
        rs.in[qr] = W.Mx; rs.out[qr] = W.out; rs.chi[qr] = t.chi_new; rs.k[qr] = t.k; rs.site[qr] = t.site_idx;
        rs.ld_in[qr] = 4ll * t.k; rs.ld_out[qr] = t.ld;
        cn_r[qr] = L.ints; mrows[qr] = t.m;
        if (!t.skip1) {
          int q = a1.count++;
          a1.A[q] = W.cv; a1.lda[q] = t.ld; a1.m[q] = t.m; a1.k[q] = t.k; a1.beta[q] = W.beta1; a1.tau[q] = W.tau1;
          a1.Y[q] = W.out; a1.ldy[q] = t.ld; a1.ncols[q] = 4 * t.chi_new;
        }
      }
    }
    if (bw.count) {
      { ProfScope ps(c, PC_DRESS, 0, 0); rc = launch_build_W(sh, bw, gt, cn_w); if (rc) return rc; }
    }
    if (sh != st) {                                       // join: the heavy kernels run on the piece stream
      PEPO_CUDA_OK(cudaEventRecord(S.ev[1], sh));
      PEPO_CUDA_OK(cudaStreamWaitEvent(st, S.ev[1], 0));
    }
    c->cur_st = st;
    if (bw.count) {
      for (auto& t : T) {
        if (!t.chol) continue;
        SiteWs& W = c->lanes[t.lane].s[t.slot];
        GemmProb gp;
        gp.A = W.cv; gp.lda = t.ld; gp.B = W.W; gp.ldb = t.n; gp.C = W.out; gp.ldc = t.ld;
        gp.M = t.m; gp.N = 4 * t.chi_new; gp.K = t.n;
        ProfScope ps(c, PC_APPLY, 2.0 * t.m * t.n * 4 * t.chi_new, 8.0 * t.m * (t.n + 4 * t.chi_new));
        if (t.direct) {
          // psi_new = psi x_(cut,P) W written in the canonical layout into the lane's spare slot of this
          // site class (the absorb / de-absorb scalings cancel: cv W / sqrt(lambda_env) = psi W); the
          // site takes the spare, its old slot becomes the spare (a10-a13 fused, no permute pass)
          SiteInfo& sv = c->sites[t.v];
          double* dst = W.spare[sv.nlegs];
          rc = launch_site_apply(st, sv.psi, t.view, W.W, t.n, t.chi_new, dst); if (rc) return rc;
          W.spare[sv.nlegs] = sv.psi;
          if (W.out == dst) W.out = sv.psi;
          sv.psi = dst;
          continue;
        }
        rc = launch_dgemm(st, 0, 0, gp, 1, 0, nullptr, false); if (rc) return rc;
      }
    }
    if (rs.count) {
      ProfScope ps(c, PC_HOUSEHOLDER, 0, 0);
      rc = launch_copy_pad(st, padsrc, pad); if (rc) return rc;
      if (a2.count) { rc = launch_hh_apply_q(st, a2); if (rc) return rc; }
      rc = launch_reshuffle_M(st, rs, cn_r, mrows); if (rc) return rc;
      if (a1.count) { rc = launch_hh_apply_q(st, a1); if (rc) return rc; }
    }
  }
  // ---- F: inverse permute + deabsorb + write-back ----------------------------------------------------
  for (auto& t : T) {
    if (t.direct) continue;                    // already in place (reconstruction wrote the site slot)
    const SiteInfo& s = c->sites[t.v];
    SiteWs& W = c->lanes[t.lane].s[t.slot];
    PermuteDesc pd;
    pd.rank = s.nlegs + 1; pd.power = 1.0;
    // source dims in cv order: env legs, cut (chi_new), P
    int newdims[5];
    for (int l = 0; l < s.nlegs; l++) newdims[l] = (l == t.cut_leg) ? t.chi_new : t.dims[l];
    newdims[s.nlegs] = 4;
    long long dst_stride_of_leg[5];
    long long ds = 1;
    for (int l = 0; l <= s.nlegs; l++) { dst_stride_of_leg[l] = ds; ds *= newdims[l]; }
    long long sstr = 1;
    int src_leg[5];
    for (int j = 0; j < t.n_env; j++) {
      int l = t.env_legs[j];
      src_leg[j] = l; pd.shape[j] = t.dims[l]; pd.src_stride[j] = sstr; sstr *= t.dims[l];
      pd.scale[j] = matrix_env(c) ? nullptr : bond_vec(c->isqrt_l, s.leg_bond[l], c->chi_max);
    }
    src_leg[t.n_env] = t.cut_leg; pd.shape[t.n_env] = t.chi_new; pd.src_stride[t.n_env] = t.ld; pd.scale[t.n_env] = nullptr;
    src_leg[t.n_env + 1] = s.nlegs; pd.shape[t.n_env + 1] = 4; pd.src_stride[t.n_env + 1] = t.ld * t.chi_new; pd.scale[t.n_env + 1] = nullptr;
    // output dim j (canonical leg j) is source dim whose leg is j
    for (int j = 0; j <= s.nlegs; j++) {
      int sd = -1;
      for (int q = 0; q <= s.nlegs; q++) if (src_leg[q] == j) sd = q;
      pd.perm[j] = sd; pd.dst_stride[j] = dst_stride_of_leg[j];
    }
    ProfScope ps(c, PC_PERMUTE, 0, 16.0 * t.m * 4 * t.chi_new);
    if (matrix_env(c) && t.n_env > 0) {
      // de-absorb (a12) by chi x chi GEMMs with the pseudo-inverse square roots
      int rc = launch_permute(st, W.out, W.cv, pd); if (rc) return rc;
      const double* src = W.cv;
      for (int j = 0; j < t.n_env; j++) {
        const int l = t.env_legs[j];
        double* dst = (j == t.n_env - 1) ? s.psi : ((j % 2 == 0) ? W.out : W.cv);
        const double* Si = c->nSinv + (size_t)msg_index(c, t.v, s.leg_dir[l], false) * c->chi_max * c->chi_max;
        rc = leg_apply(c, st, src, newdims, s.nlegs, l, Si, newdims[l], W.W, dst); if (rc) return rc;
        src = dst;
      }
      continue;
    }
    int rc = launch_permute(st, W.out, s.psi, pd);
    if (rc) return rc;
  }
  if (matrix_env(c)) {
    // a13: mu <- diag(lambda) on the updated bond, both directions, in the new index basis
    const size_t x2 = (size_t)c->chi_max * c->chi_max;
    for (int g = 0; g < ng; g++) {
      const int e = gate_bonds[g], cn = T[2 * g].chi_new;
      const double* lam = bond_vec(c->lambda, e, c->chi_max);
      for (int k = 0; k < 2; k++) {
        int rc = launch_set_diag(st, lam, cn, 0, c->nM[c->n_cur] + (2 * e + k) * x2); if (rc) return rc;
        rc = launch_set_diag(st, lam, cn, 1, c->nS + (2 * e + k) * x2); if (rc) return rc;
        rc = launch_set_diag(st, lam, cn, 2, c->nSinv + (2 * e + k) * x2); if (rc) return rc;
      }
    }
  }
  for (int g = 0; g < ng; g++) c->chi[gate_bonds[g]] = T[2 * g].chi_new;
  c->msgs_valid = false;
  return 0;
}

int run_batch(pepo_ctx* c, const std::vector<int>& gate_bonds) {
  if (gate_bonds.empty()) return 0;
  BatchState S;
  S.gate_bonds = gate_bonds; S.ng = (int)gate_bonds.size(); S.lane0 = 0; S.st = c->st;
  int rc = batch_p1(c, S);
  if (!rc) rc = batch_p2(c, S);
  if (!rc) rc = batch_p3(c, S);
  return rc;
}

// ---------------------------------------------------------------------------------------------
// Pipelined Trotter step (option "pipeline", default on).  The Jacobi SVD of a batch is latency-
// bound on a few SMs (one cluster per core), so the gates of a step run as pieces of up to B / NS
// gates on NS piece streams: while one piece sits in its SVD the others run their Gram /
// reconstruction GEMMs.  The schedule is a list schedule over the gate dependency graph (a gate
// depends on the gate that touched each of its two sites before it, in class order): a stream that
// has enqueued the write-back of its piece takes READY gates - ready = the gates it depends on have
// their write-back enqueued, so the dependency becomes stream order or one cudaStreamWaitEvent.
// Classes therefore overlap wherever the lattice allows it (on a square grid a row runs through both
// horizontal classes without waiting for the other rows, and the outer columns start the vertical
// classes while the inner columns are still in the second horizontal one).  The host drives the
// streams by polling the read-back events of the phases (Cholesky flags, chi_new).  Gate results do
// not depend on the schedule or on which gates share a piece: no kernel takes its configuration
// from the batch composition (tested bit-identical to the serial schedule).
// ---------------------------------------------------------------------------------------------
struct Piece {
  BatchState S;
  int stream = 0, phase = 0;
  std::vector<int> sites;
};

// field gate (a1) of the sites of `sites` that have not had it in this step, on `st`, each after its
// own pending upload
int lazy_field_gate(pepo_ctx* c, const std::vector<int>& sites, cudaStream_t st) {
  FieldBatch fb; fb.count = 0;
  double fbytes = 0;
  for (int v : sites) {
    if (!c->field_todo[v]) continue;
    c->field_todo[v] = 0;
    if (c->site_pending[v]) {
      PEPO_CUDA_OK(cudaStreamWaitEvent(st, c->site_ev[v], 0));
      c->site_pending[v] = 0; c->n_pending--;
    }
    if (c->f_row_mask == 0) continue;
    fb.psi[fb.count] = c->sites[v].psi;
    fb.slab[fb.count] = (long long)(site_live_size(c, v) / 4);
    fbytes += 8.0 * fb.slab[fb.count] * 2 * __builtin_popcount(c->f_row_mask);
    if (++fb.count == PEPO_BP_MAXS) {
      memcpy(fb.G, c->lazy_half ? c->G1h : c->G1, sizeof(fb.G));
      fb.row_mask = c->f_row_mask; fb.col_mask = c->f_col_mask;
      int rc = launch_field_gate(st, fb); if (rc) return rc;
      fb.count = 0;
    }
  }
  if (fb.count) {
    memcpy(fb.G, c->lazy_half ? c->G1h : c->G1, sizeof(fb.G));
    fb.row_mask = c->f_row_mask; fb.col_mask = c->f_col_mask;
    cudaStream_t keep = c->cur_st; c->cur_st = st;
    ProfScope ps(c, PC_FIELD, 0, fbytes);
    int rc = launch_field_gate(st, fb);
    c->cur_st = keep;
    if (rc) return rc;
  }
  if (c->n_pending == 0) c->copy_forked = false;
  return 0;
}

int run_step_piped_impl(pepo_ctx* c) {
  const int NS = std::min(std::min(c->pipeline, pepo_ctx::NSMAX), c->B);
  const int hb = c->B / NS;                      // lanes per stream
  // the gates of the step in class order, each with the gates that last touched its two sites
  struct GateNode { int bond, dep[2], piece; };
  std::vector<GateNode> G;
  {
    std::vector<int> last(c->n_sites, -1);
    for (auto& cls : c->classes)
      for (int e : cls) {
        GateNode g;
        g.bond = e; g.piece = -1;
        g.dep[0] = last[c->bonds[e].v1]; g.dep[1] = last[c->bonds[e].v2];
        last[c->bonds[e].v1] = last[c->bonds[e].v2] = (int)G.size();
        G.push_back(g);
      }
  }
  const int ngates = (int)G.size();
  while ((int)c->done_ev.size() < ngates) {
    cudaEvent_t e;
    PEPO_CUDA_OK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    c->done_ev.push_back(e);
  }
  std::deque<Piece> P;                           // references stay valid while pieces are appended
  int cur[pepo_ctx::NSMAX];
  for (int s = 0; s < pepo_ctx::NSMAX; s++) cur[s] = -1;
  // the piece streams start after everything already queued on the caller's stream (the field gate)
  cudaEvent_t fork = c->pev[3 * pepo_ctx::NSMAX];
  PEPO_CUDA_OK(cudaEventRecord(fork, c->st));
  for (int s = 0; s < NS; s++) PEPO_CUDA_OK(cudaStreamWaitEvent(c->ps[s], fork, 0));
  int rc = 0, left = ngates, first_free = 0;
  double t_enq = 0.0; const auto t_all0 = std::chrono::steady_clock::now();
  // GEMM weight of a gate: the sizes of its two site tensors
  auto weight = [&](int g) {
    double w = 0;
    for (int v : {c->bonds[G[g].bond].v1, c->bonds[G[g].bond].v2}) {
      double m = 4;
      for (int l = 0; l < c->sites[v].nlegs; l++) m *= c->chi[c->sites[v].leg_bond[l]];
      w += m;
    }
    return w;
  };
  while (!rc && left > 0) {
    bool progressed = false;
    for (int s = 0; s < NS && !rc; s++) {
      cudaEvent_t rb = c->pev[3 * s + 2];
      if (cur[s] < 0 || P[cur[s]].phase == 3) {
        // idle stream: a new piece of up to hb READY gates.  Ready = every gate that touched one of its
        // sites before has its write-back enqueued (phase 3), so the dependency is a stream order or one
        // cudaStreamWaitEvent.  Two ready gates never share a site.
        while (first_free < ngates && G[first_free].piece >= 0) first_free++;
        std::vector<int> pick, rdy;
        for (int g = first_free; g < ngates; g++) {
          if (G[g].piece >= 0) continue;
          bool ready = true;
          for (int d : G[g].dep) ready &= (d < 0 || (G[d].piece >= 0 && P[G[d].piece].phase == 3));
          if (ready) rdy.push_back(g);
        }
        if (rdy.empty()) continue;
        if (c->lazy_field && c->n_pending > 0) {
          // asynchronous uploads in flight (pepo_set_site_async): only gates whose two sites have ARRIVED start
          // now; a piece that mixed an early and a late site would hold its stream until the late one is there
          std::vector<int> here;
          for (int g : rdy) {
            bool ok = true;
            for (int v : {c->bonds[G[g].bond].v1, c->bonds[G[g].bond].v2})
              ok &= (!c->site_pending[v] || cudaEventQuery(c->site_ev[v]) == cudaSuccess);
            if (ok) here.push_back(g);
          }
          if (here.empty()) continue;
          rdy.swap(here);
        }
        // the heaviest ready gate, then the lightest ones: every piece gets its share of the GEMM-heavy
        // gates (pieces taken in list order put the interior gates of a class on two of the four streams:
        // 38.7 against 36.6 ms per step on 4x4 chi = 60)
        std::stable_sort(rdy.begin(), rdy.end(), [&](int a, int b) { return weight(a) > weight(b); });
        pick.push_back(rdy[0]);
        for (int k = (int)rdy.size() - 1; k >= 1 && (int)pick.size() < hb; k--) pick.push_back(rdy[k]);
        std::sort(pick.begin(), pick.end());
        const int i = (int)P.size();
        P.emplace_back();
        Piece& u = P.back();
        u.stream = s;
        for (int g : pick) {
          G[g].piece = i;
          u.S.gate_bonds.push_back(G[g].bond);
          u.sites.push_back(c->bonds[G[g].bond].v1); u.sites.push_back(c->bonds[G[g].bond].v2);
        }
        u.S.ng = (int)pick.size();
        u.S.lane0 = s * hb;
        u.S.st = c->ps[s];
        u.S.hp = c->hp[s];
        u.S.ev[0] = c->pev[3 * s]; u.S.ev[1] = c->pev[3 * s + 1];
        u.S.piped = true;
        std::vector<int> waited;
        for (int g : pick)
          for (int d : G[g].dep) {
            if (d < 0) continue;
            const int pd = G[d].piece;
            if (P[pd].stream == s || std::find(waited.begin(), waited.end(), pd) != waited.end()) continue;
            PEPO_CUDA_OK(cudaStreamWaitEvent(u.S.st, c->done_ev[pd], 0));
            waited.push_back(pd);
          }
        const auto tq0 = std::chrono::steady_clock::now();
        if (c->lazy_field) { rc = lazy_field_gate(c, u.sites, u.S.st); if (rc) break; }
        rc = batch_p1(c, u.S);
        t_enq += std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - tq0).count();
        if (!rc) { PEPO_CUDA_OK(cudaEventRecord(rb, u.S.hp ? u.S.hp : u.S.st)); }
        u.phase = 1; cur[s] = i; progressed = true;
      } else if (cudaEventQuery(rb) == cudaSuccess) {
        const int i = cur[s];
        Piece& u = P[i];
        const auto tq0 = std::chrono::steady_clock::now();
        if (u.phase == 1) {
          rc = batch_p2(c, u.S);
          if (!rc) { PEPO_CUDA_OK(cudaEventRecord(rb, u.S.hp ? u.S.hp : u.S.st)); }
          u.phase = 2;
        } else {
          rc = batch_p3(c, u.S);
          if (!rc) { PEPO_CUDA_OK(cudaEventRecord(c->done_ev[i], u.S.st)); }
          u.phase = 3; left -= u.S.ng;
        }
        t_enq += std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - tq0).count();
        progressed = true;
      }
    }
    if (!progressed) std::this_thread::yield();
  }
  if (c->lazy_field && !rc) {                 // sites no gate touched (none on connected grids)
    std::vector<int> all(c->n_sites);
    for (int v = 0; v < c->n_sites; v++) all[v] = v;
    // ordered after the piece streams by the join below: do it on the first piece stream
    rc = lazy_field_gate(c, all, c->ps[0]);
    c->lazy_field = false;
  }
  if (c->prof.trace)
    fprintf(stderr, "HOST step %.3f ms, of which enqueueing phases %.3f ms\n",
            std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_all0).count(), t_enq);
  // join: the caller's stream continues after all piece streams
  for (int s = 0; s < NS; s++) {
    cudaEventRecord(c->pev[3 * pepo_ctx::NSMAX + 1 + s], c->ps[s]);
    cudaStreamWaitEvent(c->st, c->pev[3 * pepo_ctx::NSMAX + 1 + s], 0);
  }
  c->cur_st = c->st;
  if (rc || c->prof.on) {
    cudaStreamSynchronize(c->st);
    for (int s = 0; s < NS; s++) { cudaStreamSynchronize(c->ps[s]); cudaStreamSynchronize(c->hp[s]); }
    if (c->prof.on) prof_flush(c);
  }
  return rc;
}

// Every exit of the pipelined step - also an error return from the middle of the state machine -
// leaves the piece streams joined and idle and the lazy field-gate state cleared.
int run_step_piped(pepo_ctx* c) {
  const int rc = run_step_piped_impl(c);
  if (rc) {
    cudaStreamSynchronize(c->st);
    for (int s = 0; s < pepo_ctx::NSMAX; s++) { if (c->ps[s]) cudaStreamSynchronize(c->ps[s]); if (c->hp[s]) cudaStreamSynchronize(c->hp[s]); }
    if (c->copy_st) cudaStreamSynchronize(c->copy_st);
    c->lazy_field = false;
    std::fill(c->site_pending.begin(), c->site_pending.end(), 0);
    c->n_pending = 0; c->copy_forked = false;
    c->cur_st = c->st;
    c->prof.used = 0;
  }
  return rc;
}

}  // namespace

// Order in which a Trotter step first touches the sites (gate by gate, class by class): uploading the site tensors in this order (pepo_set_site_async) lets the step
// start earliest.  h_order: n_sites ints (site index = y * Lx + x).
extern "C" int pepo_site_order(pepo_ctx* c, int* h_order, int n) {
  if (!c || !h_order || n < c->n_sites) { set_error("site_order: bad argument"); return -1; }
  std::vector<char> seen(c->n_sites, 0);
  int k = 0;
  // the list schedule hands out the gates class by class
  for (auto& cls : c->classes)
    for (int e : cls)
      for (int v : {c->bonds[e].v1, c->bonds[e].v2})
        if (!seen[v]) { seen[v] = 1; h_order[k++] = v; }
  for (int v = 0; v < c->n_sites; v++) if (!seen[v]) h_order[k++] = v;
  return 0;
}

extern "C" int pepo_apply_bond(pepo_ctx* c, int bond) {
  if (!c || bond < 0 || bond >= c->n_bonds) { set_error("apply_bond: bad bond"); return -1; }
  CtxScope scope(c);
  { int rcw = wait_pending_uploads(c, c->st); if (rcw) return rcw; }
  std::vector<int> g(1, bond);
  return run_batch(c, g);
}

extern "C" int pepo_trotter_step(pepo_ctx* c) {
  if (!c) { set_error("trotter_step: NULL"); return -1; }
  CtxScope scope(c);
  c->stats.gate_err = 0.0; c->stats.min_cut_gap = 1.0; c->stats.jacobi_sweeps = 0;
  // order 1 (R2): field gate, bond sweep.  order 2 (PAPER eq. (6)):
  // half field gate, bond sweep, half field gate.
  const bool sym = c->trotter_order == 2;
  const bool piped = c->pipeline >= 2 && c->B >= 2;
  int rc = 0;
  // asynchronous uploads in flight: the field gate is applied piece by piece, each piece waiting
  // only for its own sites, so the step starts while the rest of the state is still arriving
  c->lazy_field = piped && c->n_pending > 0;
  if (c->lazy_field) { c->lazy_half = sym; std::fill(c->field_todo.begin(), c->field_todo.end(), 1); }
  else rc = apply_field_impl(c, sym);
  if (rc) return rc;
  if (piped) rc = run_step_piped(c);
  else {
    for (auto& cls : c->classes) {
      for (size_t i0 = 0; i0 < cls.size() && !rc; i0 += c->B) {
        std::vector<int> g(cls.begin() + i0, cls.begin() + std::min(cls.size(), i0 + (size_t)c->B));
        rc = run_batch(c, g);
      }
      if (rc) break;
    }
  }
  if (rc) return rc;
  if (sym) rc = apply_field_impl(c, true);
  return rc;
}

// ============================================================================================
// BP + Bethe
// ============================================================================================
namespace {

int msg_index(const pepo_ctx* c, int v, int dir, bool outgoing) {
  const SiteInfo& s = c->sites[v];
  int e = s.bond_of_dir[dir];
  const BondInfo& b = c->bonds[e];
  bool is_v1 = (b.v1 == v);
  // message 2e: v1 -> v2 ; 2e+1: v2 -> v1
  int out = is_v1 ? 2 * e : 2 * e + 1;
  return outgoing ? out : (out ^ 1);
}

void fill_bp_site(pepo_ctx* c, int v, int cur, BpSite& S) {
  const SiteInfo& s = c->sites[v];
  size_t slab = site_live_size(c, v) / 4;
  int pv = (v == c->center) ? c->obsP : 0;
  S.T = s.psi + slab * pv;
  // The sweep kernel sees a 4-index tensor T[u,d,l,r] and puts lanes on u and warps on d.  A missing leg
  // has dimension 1 and can sit anywhere in the index list without changing the memory layout, so the
  // legs that exist take the roles u, d, l, r in storage order and the missing ones the trailing roles
  // (a top-row site, stored [D,L,R], would otherwise run with one active lane per warp).
  S.first_slot = s.nlegs > 0 ? 0 : -1;
  for (int role = 0; role < 4; role++) {
    if (role < s.nlegs) {
      const int d = s.leg_dir[role];
      const int e = s.leg_bond[role];
      S.d[role] = c->chi[e]; S.present[role] = 1;
      S.in[role] = c->msgs[cur] + (size_t)msg_index(c, v, d, false) * c->chi_max;
      S.out_old[role] = c->msgs[cur] + (size_t)msg_index(c, v, d, true) * c->chi_max;
      S.out_new[role] = c->msgs[cur ^ 1] + (size_t)msg_index(c, v, d, true) * c->chi_max;
    } else {
      S.d[role] = 1; S.present[role] = 0;
      S.in[role] = c->ones; S.out_old[role] = c->ones; S.out_new[role] = nullptr;
    }
  }
  S.partU = c->partU[v]; S.partD = c->partD[v]; S.partS = c->partS[v];
  S.vs = c->vs + v;
}

// one sweep from message set `cur`; delta goes to slot `slot` of delta_bits; if prev_slot >= 0 the
// sweep is skipped on the device when the delta in that slot is already below the tolerance
int bp_sweep(pepo_ctx* c, double damping, int update, int cur = -1, int slot = 0, int prev_slot = -1) {
  if (cur < 0) cur = c->cur_msg;
  for (int v0 = 0; v0 < c->n_sites; v0 += PEPO_BP_MAXS) {
    BpBatch bb;
    bb.count = std::min(PEPO_BP_MAXS, c->n_sites - v0);
    if (prev_slot >= 0) { bb.skip_if = c->delta_bits + prev_slot; bb.skip_tol = c->bp_tol; }
    for (int i = 0; i < bb.count; i++) fill_bp_site(c, v0 + i, cur, bb.s[i]);
    double bbytes = 0; for (int i = 0; i < bb.count; i++) bbytes += 8.0 * bb.s[i].d[0] * bb.s[i].d[1] * bb.s[i].d[2] * bb.s[i].d[3];
    // chunking: ~8 CTAs per SM over the batch, each CTA a contiguous run of (l,r) slices
    const double per_cta = std::max(bbytes / (148.0 * 8.0), 32768.0);
    for (int i = 0; i < bb.count; i++) {
      BpSite& S = bb.s[i];
      const double slice = 8.0 * S.d[0] * S.d[1];
      const int nlr = S.d[2] * S.d[3];
      int ch = (int)std::min<double>(std::max(per_cta / slice, 1.0), (double)PEPO_BP_MAXCHUNK);
      S.chunk = std::min(ch, nlr);
      S.nchunks = (nlr + S.chunk - 1) / S.chunk;
    }
    ProfScope ps(c, PC_BP, 0, bbytes);
    int rc = launch_bp_partial(c->st, bb); if (rc) return rc;
    rc = launch_bp_finalize(c->st, bb, damping, update, c->delta_bits + slot, c->bp_ints); if (rc) return rc;
  }
  return 0;
}

int bp_init_messages(pepo_ctx* c) {
  for (int e = 0; e < c->n_bonds; e++) { c->h_chi_msg[2 * e] = c->chi[e]; c->h_chi_msg[2 * e + 1] = c->chi[e]; }
  if (c->n_bonds) {
    PEPO_CUDA_OK(cudaMemcpyAsync(c->chi_of_msg, c->h_chi_msg, (size_t)2 * c->n_bonds * 4, cudaMemcpyHostToDevice, c->st));
    int rc = launch_bp_init(c->st, c->msgs[c->cur_msg], c->chi_of_msg, 2 * c->n_bonds, c->chi_max, c->bp_init);
    if (rc) return rc;
  }
  PEPO_CUDA_OK(cudaMemsetAsync(c->bp_ints, 0, 16, c->st));
  return 0;
}

}  // namespace

namespace {
// One stage of BP: restart from the deterministic init (R7) and sweep with `damping` until delta < tol
// or `budget` sweeps.  Returns 0 converged, 1 budget exhausted, < 0 error.  Sweeps go out in groups of
// up to BP_GROUP with one read-back of their deltas per group (one host round trip instead of
// BP_GROUP); inside a group the stop test of eq. (14) is taken on the device: the kernels of a sweep
// return at once when the previous sweep's delta is below tol.
int bp_run_stage(pepo_ctx* c, double damping, int budget, int& sweeps, double& delta, int& flags) {
  int rc = bp_init_messages(c); if (rc) return rc;
  int status = 1;
  for (int it = 0; it < budget && status;) {
    const int ngr = std::min(c->bp_group < 1 ? 1 : std::min(c->bp_group, BP_GROUP), budget - it);
    PEPO_CUDA_OK(cudaMemsetAsync(c->delta_bits, 0, 8 * ngr, c->st));
    for (int g = 0; g < ngr; g++) {
      rc = bp_sweep(c, damping, 1, c->cur_msg ^ (g & 1), g, g - 1); if (rc) return rc;
    }
    PEPO_CUDA_OK(cudaMemcpyAsync(c->h_delta, c->delta_bits, 8 * ngr, cudaMemcpyDeviceToHost, c->st));
    PEPO_CUDA_OK(cudaMemcpyAsync(c->h_bpints, c->bp_ints, 8, cudaMemcpyDeviceToHost, c->st));
    PEPO_CUDA_OK(cudaStreamSynchronize(c->st));
    prof_flush(c);
    flags |= c->h_bpints[0];
    if (flags & 2) break;                               // non-finite norm: no point in spending the budget
    int done = ngr;                                     // sweeps of the group that actually ran
    for (int g = 0; g < ngr; g++) {
      double dg;
      memcpy(&dg, c->h_delta + g, 8);
      if (c->n_bonds == 0) dg = 0.0;
      delta = dg;
      if (dg < c->bp_tol) { status = 0; done = g + 1; break; }
    }
    if (done & 1) c->cur_msg ^= 1;
    sweeps += done;
    it += done;
  }
  return status;
}

// Stages of bp_converge (R7 + the alpha-retry ladder of PAPER.md L451-L457): 0 = undamped (alpha = 1),
// 1 = the configured damping d (alpha = 1 - d), 2 = option "bp_damping2" (default 0.2, i.e. alpha = 0.8;
// only with option "bp_ladder").  Runs stages first..last until one converges.
int bp_run_stages(pepo_ctx* c, int first, int& sweeps, double& delta, int& flags, int& stage_out, int& stage_sweeps) {
  int status = 1;
  const int last = c->bp_ladder ? 2 : 1;
  for (int stage = first; stage <= last && status == 1 && !(flags & 2); stage++) {
    const double damping = stage == 0 ? 0.0 : (stage == 1 ? c->bp_damping : c->bp_damping2);
    const int budget = stage == 0 ? c->bp_max_sweeps : c->bp_max_sweeps_damped;
    if (stage >= 1 && !(damping > 0.0)) continue;
    if (stage == 2 && damping == c->bp_damping) continue;
    const int before = sweeps;
    status = bp_run_stage(c, damping, budget, sweeps, delta, flags);
    if (status < 0) return status;
    stage_out = stage; stage_sweeps = sweeps - before;
  }
  return status;
}

int bp_finish(pepo_ctx* c, int status, int sweeps, double delta, int flags, int stage, int stage_sweeps) {
  c->msgs_valid = true;
  c->stats.last_bp_sweeps = sweeps; c->stats.last_bp_status = status; c->stats.last_bp_delta = delta;
  // trap candidate of PAPER.md L451-L457: converged, but only after >= 30 sweeps
  c->stats.last_bp_trap = (status == 0 && sweeps >= 30) ? 1 : 0;
  (void)stage_sweeps;
  c->stats.last_bp_flags = flags;
  c->stats.last_bp_stage = stage;
  if (flags & 2) { set_error("bp_converge: a message update had a non-finite norm (NaN / Inf in the site tensors or messages)"); return -4; }
  return status;
}
}  // namespace

extern "C" int pepo_bp_converge(pepo_ctx* c, int* h_sweeps, double* h_delta) {
  if (!c) { set_error("bp_converge: NULL"); return -1; }
  CtxScope scope(c);
  { int rcw = wait_pending_uploads(c, c->st); if (rcw) return rcw; }
  int sweeps = 0, flags = 0, stage = 0, stage_sweeps = 0;
  double delta = INFINITY;
  int status = bp_run_stages(c, 0, sweeps, delta, flags, stage, stage_sweeps);
  if (status < 0) return status;
  if (h_sweeps) *h_sweeps = sweeps;
  if (h_delta) *h_delta = delta;
  return bp_finish(c, status, sweeps, delta, flags, stage, stage_sweeps);
}

// BP + Bethe with the trap remediation procedure of PAPER.md L451-L457:
//  1. run the stages (undamped, then the alpha ladder) until one converges;
//  2. a converged run that needed >= 30 sweeps in all is a trap candidate; it is taken for a trap when
//     |C| dropped by more than 50 % against the last accepted C(t) while gate_err did not grow by more
//     than a factor 2 ("no corresponding increase in gate_err");
//  3. then the next stages (another alpha) are tried, each from the init; the first converged one
//     that is not a trap by the same test is accepted;
//  4. if every alpha fails, status 2: the bond dimension is the bottleneck (raise chi).
// Status: 0 accepted, 1 no stage converged, 2 every converged stage looks trapped (C of the last one).
extern "C" int pepo_observe(pepo_ctx* c, double* h_C, int* h_sweeps, int* h_stage) {
  if (!c || !h_C) { set_error("observe: NULL"); return -1; }
  CtxScope scope(c);
  { int rcw = wait_pending_uploads(c, c->st); if (rcw) return rcw; }
  int sweeps = 0, flags = 0, stage = 0, stage_sweeps = 0, first = 0;
  double delta = INFINITY, C = 0.0;
  bool have = false, trapped_any = false;
  const int last = c->bp_ladder ? 2 : 1;
  const double gerr = c->stats.gate_err;
  int status = 1;
  while (first <= last) {
    status = bp_run_stages(c, first, sweeps, delta, flags, stage, stage_sweeps);
    if (status < 0) return status;
    int rcf = bp_finish(c, status, sweeps, delta, flags, stage, stage_sweeps);
    if (rcf < 0) return rcf;
    if (status != 0) break;                                     // nothing (more) converges
    int rc = pepo_correlation(c, &C); if (rc) return rc;
    have = true;
    const bool candidate = sweeps >= 30;
    const bool dropped = std::fabs(C) < 0.5 * std::fabs(c->obs_prev_C);
    // "no corresponding increase in gate_err" (L454) needs a reference: none yet -> not a trap
    const bool gerr_quiet = c->obs_prev_gerr > 0.0 && !(gerr > 2.0 * c->obs_prev_gerr);
    if (!(candidate && dropped && gerr_quiet)) { trapped_any = false; break; }
    trapped_any = true;
    first = stage + 1;                                          // retry with the next alpha
  }
  if (h_sweeps) *h_sweeps = sweeps;
  if (h_stage) *h_stage = stage;
  int out = status;
  if (status == 0 && trapped_any) out = 2;
  if (status != 0 && have && trapped_any) out = 2;              // the only converged stages were traps
  if (out == 0) { c->obs_prev_C = C; c->obs_prev_gerr = gerr; }
  *h_C = have ? C : 0.0;
  c->stats.last_bp_status = out;
  return out;
}

extern "C" int pepo_correlation(pepo_ctx* c, double* h_C) {
  if (!c || !h_C) { set_error("correlation: NULL"); return -1; }
  CtxScope scope(c);
  { int rcw = wait_pending_uploads(c, c->st); if (rcw) return rcw; }
  if (!c->msgs_valid) { set_error("correlation: no converged messages (call pepo_bp_converge after the last state change)"); return -1; }
  int rc = bp_sweep(c, 0.0, 0); if (rc) return rc;
  rc = launch_bethe(c->st, c->vs, c->n_sites, c->msgs[c->cur_msg], c->chi_of_msg, c->n_bonds, c->chi_max,
                    c->bp_scalars, c->bp_ints + 1);
  if (rc) return rc;
  PEPO_CUDA_OK(cudaMemcpyAsync(c->h_scal, c->bp_scalars, 8, cudaMemcpyDeviceToHost, c->st));
  PEPO_CUDA_OK(cudaMemcpyAsync(c->h_bpints, c->bp_ints, 8, cudaMemcpyDeviceToHost, c->st));
  PEPO_CUDA_OK(cudaStreamSynchronize(c->st));
  *h_C = c->h_scal[0];
  if (c->h_bpints[1] != 0) { set_error("correlation: zero or non-finite Z_e / vs_v"); return -4; }
  return 0;
}

// Current BP message over `bond` (from_v1 != 0: v1 -> v2, else v2 -> v1), for parity tests.
extern "C" int pepo_get_message(pepo_ctx* c, int bond, int from_v1, double* h_dst, int n) {
  if (!c || !h_dst || bond < 0 || bond >= c->n_bonds || n != c->chi[bond]) { set_error("get_message: bad argument"); return -1; }
  if (!c->msgs_valid) { set_error("get_message: no messages (call pepo_bp_converge after the last state change)"); return -1; }
  const size_t idx = (size_t)(2 * bond + (from_v1 ? 0 : 1));
  PEPO_CUDA_OK(cudaMemcpyAsync(h_dst, c->msgs[c->cur_msg] + idx * c->chi_max, (size_t)n * 8, cudaMemcpyDeviceToHost, c->st));
  PEPO_CUDA_OK(cudaStreamSynchronize(c->st));
  return 0;
}

// Diagnostics of PAPER.md Table 1 (L373-L380): bond entanglement entropies.
// Uses the message-partial scratch of the BP sweep (free between sweeps) as the output buffer.
extern "C" int pepo_bond_entropy(pepo_ctx* c, double* h_S, int n) {
  if (!c || !h_S || n < c->n_bonds) { set_error("bond_entropy: bad argument (need n >= n_bonds)"); return -1; }
  CtxScope scope(c);
  if (c->n_bonds == 0) return 0;
  for (int e = 0; e < c->n_bonds; e++) { c->h_chi_msg[2 * e] = c->chi[e]; c->h_chi_msg[2 * e + 1] = c->chi[e]; }
  PEPO_CUDA_OK(cudaMemcpyAsync(c->chi_of_msg, c->h_chi_msg, (size_t)2 * c->n_bonds * 4, cudaMemcpyHostToDevice, c->st));
  double* d_out = c->msgs[c->cur_msg ^ 1];             // spare message buffer: >= n_bonds doubles, rewritten by the next sweep
  int rc = launch_bond_entropy(c->st, c->lambda, c->chi_of_msg, c->n_bonds, c->chi_max, d_out);
  if (rc) return rc;
  PEPO_CUDA_OK(cudaMemcpyAsync(h_S, d_out, (size_t)c->n_bonds * 8, cudaMemcpyDeviceToHost, c->st));
  PEPO_CUDA_OK(cudaStreamSynchronize(c->st));
  return 0;
}

// Arena canaries: every sub-buffer of the arena is followed by 64 guard bytes filled at init.  Returns 0
// when all are intact, else -4 with the index of the first damaged one in the error text (a kernel wrote
// past the end of the buffer in front of it).  Synchronises every stream of the context.
extern "C" int pepo_check_guards(pepo_ctx* c) {
  if (!c) { set_error("check_guards: NULL"); return -1; }
  PEPO_CUDA_OK(cudaStreamSynchronize(c->st));
  for (int i = 0; i < pepo_ctx::NSMAX; i++) { if (c->ps[i]) cudaStreamSynchronize(c->ps[i]); if (c->hp[i]) cudaStreamSynchronize(c->hp[i]); }
  std::vector<unsigned char> h(64);
  for (size_t k = 0; k < c->arena.guards.size(); k++) {
    PEPO_CUDA_OK(cudaMemcpy(h.data(), c->arena.base + c->arena.guards[k], 64, cudaMemcpyDeviceToHost));
    for (int b = 0; b < 64; b++)
      if (h[b] != 0xA5) {
        set_error("check_guards: guard %zu of %zu (arena offset %zu, after buffer %s) overwritten", k, c->arena.guards.size(), c->arena.guards[k], c->arena.names[k]); return -4; }
  }
  return (int)0;
}

// n(r, t) and the spreading measures of PAPER.md section 6.4 / appendix A.3 (reading R19).
extern "C" int pepo_site_weights(pepo_ctx* c, double* h_n, int n, double* h_spread) {
  if (!c || !h_n || n < c->n_sites) { set_error("site_weights: bad argument (need n >= n_sites)"); return -1; }
  CtxScope scope(c);
  { int rcw = wait_pending_uploads(c, c->st); if (rcw) return rcw; }
  for (int v0 = 0; v0 < c->n_sites; v0 += PEPO_BP_MAXS) {
    SiteWeightBatch b;
    b.count = std::min(PEPO_BP_MAXS, c->n_sites - v0);
    for (int i = 0; i < b.count; i++) {
      const SiteInfo& s = c->sites[v0 + i];
      b.psi[i] = s.psi;
      for (int l = 0; l < 4; l++) {
        if (l < s.nlegs) { b.d[i][l] = c->chi[s.leg_bond[l]]; b.lam[i][l] = bond_vec(c->lambda, s.leg_bond[l], c->chi_max); }
        else { b.d[i][l] = 1; b.lam[i][l] = c->ones; }
      }
      b.part[i] = c->sw_part + (size_t)(v0 + i) * PEPO_SW_CHUNKS * 4;
      b.out[i] = c->sw_out + (size_t)(v0 + i) * 4;
    }
    int rc = launch_site_weights(c->st, b); if (rc) return rc;
  }
  std::vector<double> w((size_t)c->n_sites * 4);
  PEPO_CUDA_OK(cudaMemcpyAsync(w.data(), c->sw_out, w.size() * 8, cudaMemcpyDeviceToHost, c->st));
  PEPO_CUDA_OK(cudaStreamSynchronize(c->st));
  double tot = 0.0;
  for (int v = 0; v < c->n_sites; v++) {
    const double sum = w[4 * v] + w[4 * v + 1] + w[4 * v + 2] + w[4 * v + 3];
    if (!(sum > 0.0) || !std::isfinite(sum)) { set_error("site_weights: site %d has zero or non-finite norm", v); return -4; }
    h_n[v] = 1.0 - w[4 * v] / sum;
    tot += h_n[v];
  }
  if (h_spread) {
    double r1 = 0.0, r2 = 0.0, ent = 0.0;
    for (int v = 0; v < c->n_sites && tot > 0.0; v++) {
      const double p = h_n[v] / tot;
      const int dx = std::abs(c->sites[v].x - c->cx), dy = std::abs(c->sites[v].y - c->cy);
      r1 += p * (dx + dy); r2 += p * (dx * dx + dy * dy);
      if (p > 0.0) ent -= p * std::log(p);
    }
    h_spread[0] = r1; h_spread[1] = std::sqrt(r2);
    h_spread[2] = c->n_sites > 1 ? ent / std::log((double)c->n_sites) : 0.0;
  }
  return 0;
}

// ============================================================================================
// NEXT-1: norm-network BP with chi x chi matrix messages (PAPER.md:L72, L146-L150,
// L315-L317, L336, Table 1).  Built from the site-level DMMA contractions: "one leg times a matrix" is
// launch_site_apply with W = I_4 (x) M, the double-layer contraction over all legs but one is the cross
// Gram of (psi with the incoming messages applied) and psi.  Written for parity at test sizes, not tuned.
// ============================================================================================
namespace {

inline double* nmsg(pepo_ctx* c, double* base, int idx) { return base + (size_t)idx * c->chi_max * c->chi_max; }

// dst = src with leg `leg` contracted with Mat (d_leg x d_new, ld d_leg): dims[] = live dims of src
int leg_apply(pepo_ctx* c, cudaStream_t st, const double* src, const int* dims, int nlegs, int leg,
              const double* Mat, int d_new, double* Wbuf, double* dst) {
  int rc = launch_kron_i4(st, Mat, dims[leg], d_new, dims[leg], Wbuf); if (rc) return rc;
  SiteView v; v.nlegs = nlegs; v.cut = leg;
  for (int l = 0; l < 4; l++) v.dims[l] = l < nlegs ? dims[l] : 1;
  return launch_site_apply(st, src, v, Wbuf, 4ll * dims[leg], d_new, dst);
}

int nbp_init(pepo_ctx* c) {
  for (int e = 0; e < c->n_bonds; e++)
    for (int k = 0; k < 2; k++) {
      int rc = launch_set_diag(c->st, bond_vec(c->lambda, e, c->chi_max), c->chi[e], 0, nmsg(c, c->nM[c->n_cur], 2 * e + k));
      if (rc) return rc;
    }
  c->n_valid = true; c->n_sqrt_valid = false;
  return 0;
}

// psi_v with the incoming messages applied on every leg except `skip` (-1: none skipped): result pointer
// in *out (psi itself when there is nothing to apply); scratch = the explicit-cv buffers of lane 0
int nbp_dress_site(pepo_ctx* c, int v, int skip, const double** out) {
  const SiteInfo& s = c->sites[v];
  int dims[4];
  for (int l = 0; l < s.nlegs; l++) dims[l] = c->chi[s.leg_bond[l]];
  double* buf[2] = {c->lanes[0].s[0].cv, c->lanes[0].s[1].cv};
  const double* src = s.psi;
  int k = 0;
  for (int l = 0; l < s.nlegs; l++) {
    if (l == skip) continue;
    const double* Min = nmsg(c, c->nM[c->n_cur], msg_index(c, v, s.leg_dir[l], false));
    int rc = leg_apply(c, c->st, src, dims, s.nlegs, l, Min, dims[l], c->lanes[0].s[0].W, buf[k]); if (rc) return rc;
    src = buf[k]; k ^= 1;
  }
  *out = src;
  return 0;
}

// unnormalised, symmetrised message leaving v through its leg lw into c->nraw; with update: also the new
// damped message into the other set
int nbp_site_leg(pepo_ctx* c, int v, int lw, double damping, bool update) {
  const SiteInfo& s = c->sites[v];
  const double* B = nullptr;
  int rc = nbp_dress_site(c, v, lw, &B); if (rc) return rc;
  SiteView sv; sv.nlegs = s.nlegs; sv.cut = lw;
  for (int l = 0; l < 4; l++) sv.dims[l] = l < s.nlegs ? c->chi[s.leg_bond[l]] : 1;
  rc = launch_site_gram(c->st, B, sv, nullptr, c->nG, c->lanes[0].s[0].part, s.psi); if (rc) return rc;
  const int oi = msg_index(c, v, s.leg_dir[lw], true);
  double* old = nmsg(c, c->nM[c->n_cur], oi);
  double* out = update ? nmsg(c, c->nM[c->n_cur ^ 1], oi) : c->nEw;      // no update: scratch
  return launch_norm_msg(c->st, c->nG, sv.dims[lw], old, damping, out, c->nraw, c->delta_bits, c->bp_ints);
}

int nbp_sqrt_all(pepo_ctx* c) {
  for (int e = 0; e < c->n_bonds; e++)
    for (int k = 0; k < 2; k++) {
      const int chi = c->chi[e], idx = 2 * e + k;
      SvdBatch sb; sb.count = 1;
      sb.K[0] = nmsg(c, c->nM[c->n_cur], idx); sb.ldk[0] = chi; sb.r1[0] = chi; sb.r2[0] = chi;
      sb.G[0] = c->nEg; sb.V[0] = c->nEv; sb.sv[0] = c->nEs; sb.order[0] = c->nEo; sb.sweeps[0] = c->nEo + c->chi_max;
      int rc = launch_svd_jacobi(c->st, sb, 1e-15, 60, true, 0, 0.0); if (rc) return rc;
      rc = launch_svd_vectors(c->st, c->nEg, c->nEv, c->nEs, c->nEo, chi, chi, c->nEu, c->nEw); if (rc) return rc;
      rc = launch_psqrt_build(c->st, c->nEu, c->nEw, c->nEs, chi, c->psqrt_eps, nmsg(c, c->nS, idx), nmsg(c, c->nSinv, idx));
      if (rc) return rc;
    }
  c->n_sqrt_valid = true;
  return 0;
}

}  // namespace

// Sweeps of the matrix-message BP from the CURRENT messages (diag(lambda) if there are none) until
// delta < tol or max_sweeps; afterwards the PSEUDO_SQRTs of all messages are refreshed.
extern "C" int pepo_norm_bp_converge(pepo_ctx* c, double tol, double damping, int max_sweeps, int* h_sweeps, double* h_delta) {
  if (!c || !(tol > 0.0) || damping < 0.0 || damping >= 1.0 || max_sweeps < 1) { set_error("norm_bp_converge: bad argument"); return -1; }
  CtxScope scope(c);
  { int rcw = wait_pending_uploads(c, c->st); if (rcw) return rcw; }
  int rc = 0;
  if (!c->n_valid) { rc = nbp_init(c); if (rc) return rc; }
  int sweeps = 0, status = 1;
  double delta = INFINITY;
  PEPO_CUDA_OK(cudaMemsetAsync(c->bp_ints, 0, 16, c->st));
  for (int it = 0; it < max_sweeps && status; it++) {
    PEPO_CUDA_OK(cudaMemsetAsync(c->delta_bits, 0, 8, c->st));
    for (int v = 0; v < c->n_sites; v++)
      for (int l = 0; l < c->sites[v].nlegs; l++) { rc = nbp_site_leg(c, v, l, damping, true); if (rc) return rc; }
    c->n_cur ^= 1;
    PEPO_CUDA_OK(cudaMemcpyAsync(c->h_delta, c->delta_bits, 8, cudaMemcpyDeviceToHost, c->st));
    PEPO_CUDA_OK(cudaMemcpyAsync(c->h_bpints, c->bp_ints, 8, cudaMemcpyDeviceToHost, c->st));
    PEPO_CUDA_OK(cudaStreamSynchronize(c->st));
    memcpy(&delta, c->h_delta, 8);
    if (c->n_bonds == 0) delta = 0.0;
    sweeps++;
    if (c->h_bpints[0] & 2) { set_error("norm_bp_converge: non-finite message norm"); return -4; }
    if (delta < tol) status = 0;
  }
  c->n_sqrt_valid = false;
  rc = nbp_sqrt_all(c); if (rc) return rc;
  if (h_sweeps) *h_sweeps = sweeps;
  if (h_delta) *h_delta = delta;
  return status;
}

// Bethe norm of PAPER.md Table 1 (L373-L380, L550): exp(sum_v log f_v - sum_e log Z_e) of the double-layer
// network with the current matrix messages (1 on a tree).
extern "C" int pepo_bethe_norm(pepo_ctx* c, double* h_norm) {
  if (!c || !h_norm) { set_error("bethe_norm: NULL"); return -1; }
  CtxScope scope(c);
  if (!c->n_valid) { int rc = nbp_init(c); if (rc) return rc; }
  for (int v = 0; v < c->n_sites; v++) {
    const SiteInfo& s = c->sites[v];
    if (s.nlegs == 0) { set_error("bethe_norm: single-site lattice"); return -1; }
    int rc = nbp_site_leg(c, v, 0, 0.0, false); if (rc) return rc;
    const int chi = c->chi[s.leg_bond[0]];
    rc = launch_frob_dot(c->st, c->nraw, nmsg(c, c->nM[c->n_cur], msg_index(c, v, s.leg_dir[0], false)), chi * chi, c->nscal + v);
    if (rc) return rc;
  }
  for (int e = 0; e < c->n_bonds; e++) {
    int rc = launch_frob_dot(c->st, nmsg(c, c->nM[c->n_cur], 2 * e), nmsg(c, c->nM[c->n_cur], 2 * e + 1), c->chi[e] * c->chi[e],
                             c->nscal + c->n_sites + e);
    if (rc) return rc;
  }
  std::vector<double> h((size_t)c->n_sites + c->n_bonds);
  PEPO_CUDA_OK(cudaMemcpyAsync(h.data(), c->nscal, h.size() * 8, cudaMemcpyDeviceToHost, c->st));
  PEPO_CUDA_OK(cudaStreamSynchronize(c->st));
  double lg = 0.0;
  for (int v = 0; v < c->n_sites; v++) { if (!(h[v] > 0.0)) { set_error("bethe_norm: f_v <= 0 at site %d", v); return -4; } lg += std::log(h[v]); }
  for (int e = 0; e < c->n_bonds; e++) { const double z = h[c->n_sites + e]; if (!(z > 0.0)) { set_error("bethe_norm: Z_e <= 0 at bond %d", e); return -4; } lg -= std::log(z); }
  *h_norm = std::exp(lg);
  return 0;
}

// Matrix message over `bond` (from_v1 != 0: sent by v1), chi x chi column-major, n = chi^2.
extern "C" int pepo_get_norm_message(pepo_ctx* c, int bond, int from_v1, double* h_dst, int n) {
  if (!c || !h_dst || bond < 0 || bond >= c->n_bonds || n != c->chi[bond] * c->chi[bond]) { set_error("get_norm_message: bad argument"); return -1; }
  if (!c->n_valid) { set_error("get_norm_message: no matrix messages (call pepo_norm_bp_converge)"); return -1; }
  PEPO_CUDA_OK(cudaMemcpyAsync(h_dst, nmsg(c, c->nM[c->n_cur], 2 * bond + (from_v1 ? 0 : 1)), (size_t)n * 8, cudaMemcpyDeviceToHost, c->st));
  PEPO_CUDA_OK(cudaStreamSynchronize(c->st));
  return 0;
}

extern "C" int pepo_get_profile(pepo_ctx* c, int n, double* h_ms, double* h_flops, double* h_bytes,
                                long long* h_count) {
  if (!c || n < 0) { set_error("get_profile: bad argument"); return -1; }
  cudaStreamSynchronize(c->st);
  prof_flush(c);
  for (int i = 0; i < n && i < PC_COUNT; i++) {
    if (h_ms) h_ms[i] = c->prof.ms[i];
    if (h_flops) h_flops[i] = c->prof.flops[i];
    if (h_bytes) h_bytes[i] = c->prof.bytes[i];
    if (h_count) h_count[i] = c->prof.cnt[i];
  }
  return PC_COUNT;
}
