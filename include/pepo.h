/*
 * pepo.h - C ABI of the B200-native Heisenberg-picture PEPO hot path
 * (arxiv/paper_2606_30985: Trotter bond update + BP sweeps + Bethe evaluation of
 *  C(t) = Tr[Z_c(t) Z_c]/2^N on the 2D transverse-field Ising model).
 *
 * Citations are "PAPER.md:L<line>" (the paper text) and "R<n>" (DESIGN.md readings, which
 * restate SURVEY.md section 8(c) C1..C18).
 *
 * Conventions
 *   - All tensors are fp64.  A site tensor psi_v has the legs [U,D,L,R] that exist at the
 *     site (neighbours U=(x,y-1), D=(x,y+1), L=(x-1,y), R=(x+1,y)) followed by the Pauli leg
 *     P (dim 4: I,X,Y,Z), stored column-major: first leg fastest, P slowest, packed at the
 *     LIVE bond dimensions (R11, R12).
 *   - Bond ids: horizontal bonds (x,y)-(x+1,y) first, id = y*(Lx-1)+x; then vertical bonds
 *     (x,y)-(x,y+1), id = Ly*(Lx-1) + y*Lx + x.  Site id = y*Lx + x.
 *   - "d_" pointers are DEVICE pointers, "h_" pointers are HOST pointers.  `stream` is a
 *     cudaStream_t passed as void* (0 = default stream).
 *   - Return value: 0 = OK, >0 = soft status, <0 = hard error:
 *       -1 bad argument, -2 arena too small, -3 CUDA error, -4 numerical failure
 *       (NaN, s0 = 0, Z_e = 0).  pepo_last_error() returns a text for the last error of
 *     the calling thread.  No exception or abort crosses this boundary.
 *   - Nothing in this library allocates device memory after pepo_init(): the caller owns one
 *     arena (e.g. a torch tensor) and the context sub-allocates it ("zero-malloc",
 *     PAPER.md:L132-L160).  There is no CPU fallback of any step.
 */
#ifndef PEPO_H_
#define PEPO_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pepo_ctx pepo_ctx;

typedef struct pepo_stats {
  double gate_err;          /* sum over the gates of the last trotter_step of the discarded
                               weight sum_{i>=chi_new} s_i^2 / sum_i s_i^2 (Table 1) */
  double min_cut_gap;       /* min over gates of the last step of (s[chi_new-1]-s[chi_new])/s[chi_new-1]
                               when truncation by chi_max was active (R8); 1.0 if never */
  long long n_cholesky;     /* site QRs done by the Cholesky path since init */
  long long n_householder;  /* site QRs done by the Householder path since init (L223-L229) */
  long long n_chol_failed;  /* Cholesky attempts rejected (pivot <= 0 or diag ratio < tau_c, R9) */
  long long jacobi_sweeps;  /* Jacobi sweeps summed over the SVDs of the last step */
  long long kernel_launches;/* kernels launched by this context since init */
  int last_bp_sweeps;       /* sweeps of the last bp_converge (both phases) */
  int last_bp_status;       /* 0 converged, 1 budget exhausted */
  double last_bp_delta;     /* delta of eq. (14) */
  size_t arena_high_water;  /* bytes of the arena actually handed out */
  size_t arena_model_bytes; /* closed-form model for the same configuration (eq. (15)-(17) analogue) */
  int max_inflight_gates;   /* gates of one colour class processed concurrently */
  int chi_max_live;         /* largest live bond dimension */
  int last_bp_trap;         /* trap flag of the diagnostics: the last bp_converge
                               converged (delta < tol) but needed >= 30 sweeps */
  int last_bp_stage;        /* stage of the last bp_converge that ended it: 0 undamped, 1 damping d, 2 the ladder's
                               second damping (option "bp_ladder") */
  int last_bp_flags;        /* bit 0: some message update of the last bp_converge had zero norm and kept its
                               old value (R7); bit 1: some update had a non-finite norm (bp_converge then
                               returns -4) */
} pepo_stats;

const char* pepo_last_error(void);

/* Analytic memory model (eq. (15)-(17), re-derived for this layout:
 * DESIGN.md "Memory model").  Bytes of arena pepo_init() needs.  max_inflight <= 0 picks the
 * default (as many gates of a colour class as fit a 170 GB budget, at most 16). */
size_t pepo_arena_bytes(int Lx, int Ly, int chi_max);
size_t pepo_arena_bytes_ex(int Lx, int Ly, int chi_max, int max_inflight);

/* Create a context for the Lx x Ly open-boundary grid, observable Z at site
 * (cx,cy) (L308), H = -J sum ZZ - h sum X (R1), first-order Trotter step dt (R2), bond cap
 * chi_max (L68), BP tolerance and damping d (m <- d m_old + (1-d) m_hat, eq. (19), R7).
 * State is initialised to the product operator: all bonds chi=1, lambda=[1] (L70, L311).
 * d_arena: device buffer of arena_bytes >= pepo_arena_bytes(...) owned by the caller for the
 * lifetime of the context.  Errors: -1 (cx,cy outside grid, chi_max<1, dt<=0, Lx/Ly<1),
 * -2 (arena too small; pepo_last_error() states the bytes needed), -3. */
int pepo_init(pepo_ctx** out, int Lx, int Ly, int cx, int cy, double J, double h, double dt,
              int chi_max, double bp_tol, double bp_damping, void* d_arena, size_t arena_bytes,
              void* stream);
/* As pepo_init with explicit max_inflight (<=0: default) and the Paulis of the model as
 * indices 0..3 = I,X,Y,Z (defaults: bond 3, field 1, observable 3; the paper's own eq. (1)
 * convention is bond 1, field 3). */
int pepo_init_ex(pepo_ctx** out, int Lx, int Ly, int cx, int cy, double J, double h, double dt,
                 int chi_max, double bp_tol, double bp_damping, void* d_arena,
                 size_t arena_bytes, void* stream, int max_inflight, int bond_pauli,
                 int field_pauli, int obs_pauli);
int pepo_destroy(pepo_ctx* ctx);

/* Options (key, value): "eps_cut" (1e-11, eq. (11)), "bp_max_sweeps" (100, L256),
 * "bp_max_sweeps_damped" (1000, R7), "chol_min_ratio" (Cholesky when m >= ratio*n, 4, R9),
 * "chol_tau" (diag-ratio rejection threshold 1e-7, R9), "force_householder" (0/1),
 * "jacobi_tol" (1e-15), "jacobi_max_sweeps" (60), "jacobi_early" (cosine below which a sweep
 * counts as the last one, 1e-7; 0 = always run the confirming sweep),
 * "trotter_order" (1 = first-order step, R2; 2 = symmetric step of eq. (6)),
 * "svd_deflate" (theta of the truncation-aware deflation of the Jacobi SVD: after 3 full sweeps the columns
 * with norm < theta x the chi_max-th largest norm are set aside; 0 = off, the default: with 1e-3 the leading
 * triplets move by up to ~theta x cos x s_cut, 2e-12 of the gate tensor on the flattest test spectrum),
 * "svd_orient" (square preconditioned cores: 0 = QR of K, 2 = QR of K^T, 1 = of the one whose column norms
 * are more graded, the default; the singular triplets are the same to rounding, the Jacobi sweep count is not),
 * "env" (0: gate environment = diag(sqrt(lambda)), reading R6(i); 1: the matrix messages of
 * pepo_norm_bp_converge), "psqrt_eps",
 * "bp_init" (0: every BP stage starts from m = (1..1)/sqrt(chi), reading R7; 1: from the leading Schmidt
 * vector e_0 of each bond, reading R7b), "bp_ladder" (1: third BP stage with "bp_damping2", default 0.2), "observe_ref_C" /
 * "observe_ref_gate_err" (reference of pepo_observe's drop test: C(t) and gate_err of the last accepted
 * layer; 1 and 0 after init), "direct_gemm" (1: Cholesky-path GEMMs read / write psi in place, 0: explicit
 * permute passes),
 * "pipeline" (number of piece streams of a Trotter step, 4; 0 = serial schedule; the results do
 * not depend on it), "bp_tol", "bp_damping", "bp_group" (BP sweeps enqueued per delta read-back,
 * 1..8; results do not depend on it), "svd_precond_min" (QR-precondition cores of at least this
 * order, 32; 0 = never), "profile", "trace".  Options belong to the context: two contexts in one
 * process do not share any setting.  -1 on unknown key. */
int pepo_set_option(pepo_ctx* ctx, const char* key, double value);

/* One full first-order Trotter step (Fig. 1; R2, R3): field gate on all
 * sites (a1), then the four colour classes of ZZ bond gates, each gate = Algorithm 1
 * (L258-L288): absorb + permute (a2-a4), QR (a5/a6), core + gate (a7/a8), Jacobi SVD +
 * truncation (a9), bridge + reconstruction (a10), inverse permute + deabsorb + write-back
 * (a11-a13).  Asynchronous work on the context stream with one host read of the new bond
 * dimensions per batch of gates. */
int pepo_trotter_step(pepo_ctx* ctx);   /* "trotter_order" 2: half field gate, bond sweep, half field gate */
/* The two halves, for gate-replay tests. */
int pepo_apply_field(pepo_ctx* ctx);
int pepo_apply_bond(pepo_ctx* ctx, int bond);

/* BP on the pinned single-layer network (eq. (13),(14),(19) PAPER.md:L243-L256, L444-L449; R6,
 * R7): Jacobi-schedule sweeps from the deterministic init until delta < tol or the budget
 * is spent; undamped phase first, damped restart if configured.  Writes the total sweep
 * count and the last delta.  Returns 0 converged, 1 budget exhausted (messages still usable),
 * -4 if a message update produced a non-finite norm.  A zero-norm update keeps the old message
 * and sets bit 0 of pepo_stats.last_bp_flags (R7). */
int pepo_bp_converge(pepo_ctx* ctx, int* h_sweeps, double* h_delta);
/* BP + Bethe evaluation with the trap remediation procedure of PAPER.md L451-L457:
 * the BP stages (undamped, damping d, and with option "bp_ladder" a third stage with option
 * "bp_damping2", default 0.2 = alpha 0.8) run until one converges; a converged stage that needed
 * >= 30 sweeps is a trap candidate and counts as a trap when |C| fell below half of the last accepted
 * C(t) while gate_err did not double; then the next alpha is tried from the init.  *h_C = C(t) of the
 * accepted stage, *h_sweeps = total sweeps, *h_stage = stage that ended the call (may be NULL).
 * Returns 0 accepted, 1 no stage converged (*h_C = 0), 2 every converged stage looks trapped - the
 * bond dimension is the bottleneck (L457) - with *h_C the last value; < 0 errors as bp_converge. */
int pepo_observe(pepo_ctx* ctx, double* h_C, int* h_sweeps, int* h_stage);
/* Bethe evaluation (eq. (7)-(9) PAPER.md:L112-L128) from the current messages, log-space with
 * sign tracking.  -4 if some Z_e is 0 (R14). */
int pepo_correlation(pepo_ctx* ctx, double* h_C);

int pepo_get_stats(pepo_ctx* ctx, pepo_stats* h_stats);
/* Arena canaries (PAPER.md:L132-L160 single pre-sized workspace): every sub-buffer of the
 * arena is followed by 64 guard bytes filled at init.  0 = all intact, -4 = a kernel wrote past the end of
 * a buffer (pepo_last_error() names the guard).  Synchronises the context's streams. */
int pepo_check_guards(pepo_ctx* ctx);
/* In-situ per-kernel-class timing (option "profile": 1 on, 0 off, 2 on + reset): CUDA-event
 * pairs on the context stream around each launch group, summed per class.  Classes, in order:
 * 0 permute(+absorb/deabsorb), 1 Gram, 2 reconstruction GEMM, 3 small core GEMMs, 4 Cholesky +
 * triangular inverse, 5 Householder, 6 gate dressing, 7 Jacobi SVD + truncation, 8 field gate,
 * 9 BP sweep.  Fills the first n entries of each non-NULL array with accumulated milliseconds,
 * algorithmic flops, algorithmic bytes and launch-group counts; returns the class count. */
int pepo_get_profile(pepo_ctx* ctx, int n, double* h_ms, double* h_flops, double* h_bytes,
                     long long* h_count);
int pepo_n_bonds(pepo_ctx* ctx);
int pepo_get_bond_dims(pepo_ctx* ctx, int* h_chi /* n_bonds */);
/* Set all live bond dimensions (1..chi_max); site tensors and lambdas become undefined until
 * set with pepo_set_site / pepo_set_lambda.  For tests and synthetic workloads. */
int pepo_set_bond_dims(pepo_ctx* ctx, const int* h_chi /* n_bonds */);
size_t pepo_site_size(pepo_ctx* ctx, int x, int y);              /* elements at live dims */
int pepo_get_site(pepo_ctx* ctx, int x, int y, double* h_dst, size_t n);
int pepo_set_site(pepo_ctx* ctx, int x, int y, const double* h_src, size_t n);
/* Asynchronous pepo_set_site: the host-to-device copy is queued on an internal copy stream and
 * the call returns at once.  h_src (pinned memory, else the copy is staged synchronously by the
 * driver) must stay valid and unchanged until pepo_trotter_step or a call returning a host value
 * (bp_converge, correlation, getters) has returned.  The next pepo_trotter_step starts on the
 * sites that have arrived while the others are still in flight: the field gate (a1) and the
 * first bond gate of a site wait for that site's copy only.  Same errors as pepo_set_site. */
int pepo_set_site_async(pepo_ctx* ctx, int x, int y, const double* h_src, size_t n);
/* Order (site index = y * Lx + x, n >= Lx * Ly ints) in which the next pepo_trotter_step first
 * touches the sites; uploading in this order lets the step start earliest.  -1 on a bad argument. */
int pepo_site_order(pepo_ctx* ctx, int* h_order, int n);
int pepo_get_lambda(pepo_ctx* ctx, int bond, double* h_dst, int n);
/* Current BP message over `bond` (eq. (13)): from_v1 != 0 gives the message
 * sent by the bond's smaller-coordinate site v1 to v2, else v2 -> v1; n = live dimension of the
 * bond.  Valid after pepo_bp_converge (else -1).  For parity tests against the oracle. */
int pepo_get_message(pepo_ctx* ctx, int bond, int from_v1, double* h_dst, int n);
int pepo_set_lambda(pepo_ctx* ctx, int bond, const double* h_src, int n);
/* Diagnostics of PAPER.md Table 1 (L373-L380): bond entanglement entropies
 * S_e = -sum_k lambda_k^2 log lambda_k^2 over the live Schmidt weights of every bond (lambda is
 * normalised, eq. (12)), computed on the device.  h_S: host array of n >= n_bonds doubles.
 * Synchronises the context stream.  -1 on a bad argument. */
int pepo_bond_entropy(pepo_ctx* ctx, double* h_S, int n);
/* NEXT-1 of SURVEY 8(f): belief propagation on the NORM network <<O|O>> with chi x chi symmetric PSD matrix
 * messages ("approximate Vidal gauge maintained by BP", L146-L150):
 *   Mhat_{v->w}[k,k'] = sum_p sum_{i,i'} psi_v[..i..,k,p] psi_v[..i'..,k',p] prod_{u != w} M_{u->v}[i_u,i'_u],
 * symmetrised, normalised to Frobenius norm 1 (matches sum lambda^2 = 1, eq. (12)), damped as eq. (19),
 * delta as eq. (14); Jacobi schedule.  pepo_norm_bp_converge sweeps from the CURRENT messages (diag(lambda_e)
 * in both directions when there are none: after init, set_lambda, set_bond_dims) until delta < tol or
 * max_sweeps, then refreshes the PSEUDO_SQRT S = V sqrt(w) V^T and its pseudo-inverse of every message
 * (symmetric Jacobi eigen-decomposition, eigenvalues below option "psqrt_eps" (1e-12) x the largest zeroed,
 * L315-L317).  Returns 0 converged / 1 budget exhausted / -4 non-finite.  With option "env" = 1 the bond gates
 * then absorb and de-absorb these matrices by chi x chi GEMMs on every environment leg (L318, L336) instead of
 * the diagonal sqrt(lambda); a gate resets the two messages of its bond to diag(lambda_new) (a13).  On a tree
 * the fixed point is diag(lambda) and nothing changes; an untruncated gate is exact for any invertible
 * environment.  Heavy contractions run on the DMMA GEMM kernels; written for parity at test sizes (chi <= 160).
 * pepo_bethe_norm: Table 1 (L373-L380, L550), exp(sum_v log f_v - sum_e log Z_e), f_v the full double-layer
 * site contraction, Z_e = sum_{kk'} M_{a->b}[k,k'] M_{b->a}[k,k'] (1 on a tree).
 * pepo_get_norm_message: message over `bond` sent by v1 (from_v1 != 0) or v2, chi x chi column-major, n = chi^2. */
int pepo_norm_bp_converge(pepo_ctx* ctx, double tol, double damping, int max_sweeps, int* h_sweeps, double* h_delta);
int pepo_bethe_norm(pepo_ctx* ctx, double* h_norm);
int pepo_get_norm_message(pepo_ctx* ctx, int bond, int from_v1, double* h_dst, int n);
/* Operator spreading (section 6.4; appendix A.3 eq. (21)): the per-site
 * non-identity Pauli weight n(r,t) = 1 - w_I / sum_p w_p with w_p = sum_i psi_v[i,p]^2 prod_legs
 * lambda_leg[i_leg] (the Pauli-resolved norm of the site in its Vidal-gauge environment; exact on trees;
 * reading R19 - the paper prints no formula), one device pass over every site tensor.  h_n: n >= n_sites
 * doubles (site index y*Lx + x).  h_spread (may be NULL): [R_L1 mean Manhattan radius, R_L2 RMS Euclidean
 * radius from the centre, S_frac = -sum p ln p / ln(n_sites)], p = n / sum n.  -4 if a site has zero norm. */
int pepo_site_weights(pepo_ctx* ctx, double* h_n, int n, double* h_spread);
/* Device pointer of a packed site tensor (valid until the next gate touching the site). */
double* pepo_site_ptr(pepo_ctx* ctx, int x, int y);

/* ------------------------------------------------------------------------------------
 * Kernel-level entry points (BASELINE config 3 and the parity tests).  Device pointers,
 * caller's stream, asynchronous unless stated.
 * ------------------------------------------------------------------------------------ */

/* Tensor permutation, section 4.1 Listing 1 (L183-L208), R10: d_src is a packed
 * column-major tensor of `rank` <= 8 dims `shape` (first dim fastest); output dim j is input
 * dim perm[j] (numpy.transpose convention on the column-major shape); d_dst gets the packed
 * column-major result.  Bit-exact copy.  d_src and d_dst must not overlap. */
int pepo_permute(const double* d_src, double* d_dst, const int* h_shape, const int* h_perm,
                 int rank, void* stream);
/* Same, fused with the diagonal environment absorption / de-absorption of a3 / a12
 * (PAPER.md:L93, L103, L267, L283, L318, L336): dst = permute(src * prod_d scale_d[i_d]);
 * h_scale is a HOST array of `rank` DEVICE pointers, entry d pointing to shape[d] multipliers
 * for input dim d (sqrt(lambda) to absorb, 1/sqrt(lambda) to de-absorb) or NULL. */
int pepo_permute_scaled(const double* d_src, double* d_dst, const int* h_shape,
                        const int* h_perm, int rank, const double* const* h_scale,
                        void* stream);

/* Gram matrix C = A^T A of a column-major m x n matrix (eq. (10)) on the
 * fp64 tensor cores (DMMA), deterministic split-K.  d_ws: workspace of
 * pepo_gram_ws_bytes(m,n) bytes.  d_C: n x n column-major, ldc = n, both triangles. */
size_t pepo_gram_ws_bytes(long long m, int n);
int pepo_gram(const double* d_A, long long m, int n, long long lda, double* d_C, void* d_ws,
              size_t ws_bytes, void* stream);

/* The same Gram matrix for callers that may not allocate device memory (CUDA graph capture, serving
 * loops, harnesses that forbid cudaMalloc): same kernels and split plan as pepo_gram - identical bits -
 * with the split-K partial sums in a device array built into the library (PEPO_STATIC_SCRATCH_BYTES,
 * held by every GPU that loads the library until exit) instead of a caller workspace.  Allocates
 * nothing; looks the array's device address up once per device.  d_A (m x n, lda >= m) and d_C (n x n,
 * both triangles) are the caller's DEVICE buffers.  Returns -2 with a message naming the needed size
 * when the plan needs more scratch than the array holds (e.g. 256000 x 40 fits, 256000 x 160 does not).
 * All calls on a device share the array: calls that overlap on the GPU (different streams, no event
 * between them) race; the array keeps the last call's contents, none of which a later call reads before
 * writing it. */
#define PEPO_STATIC_SCRATCH_BYTES (8u << 20)
size_t pepo_static_scratch_bytes(void);
int pepo_gram_static(const double* d_A, long long m, int n, long long lda, double* d_C, void* stream);

/* Permute-on-load contractions of the bond gate (what pepo_trotter_step runs on the Cholesky path:
 * the explicit permutation of PAPER.md section 4.1 and the absorb / de-absorb passes a3 / a12 are
 * folded into the two tall GEMMs, which leaves 2 reads + 1 write of psi per site and gate).
 * d_psi: packed site tensor with `nlegs` (1..4) bond legs of dims h_dims[] followed by the Pauli
 * leg (4), column-major; cut_leg: index of the gate's bond among the legs.  With cv = the
 * m x n matrix view rows = other legs (canonical order), cols = (cut, P) (L267-L269, L319):
 *   pepo_site_gram : d_C (n x n column-major, both triangles) = cv^T diag(w) cv, eq. (10),
 *                    w(row) = prod over the other legs of h_w2[leg][i_leg] (h_w2: HOST array of nlegs
 *                    DEVICE pointers, entry cut_leg ignored; pass lambda to get the Gram matrix of
 *                    the sqrt(lambda)-absorbed cv; NULL array = unweighted).  DMMA, deterministic split-K;
 *                    d_ws of pepo_site_gram_ws_bytes() bytes.
 *   pepo_site_apply: d_out = packed site tensor with dims[cut_leg] replaced by chi_new,
 *                    out[.., c', .., p'] = sum_{c,p} psi[.., c, .., p] W[(c,p),(c',p')], d_W column-major
 *                    (4 dims[cut]) x (4 chi_new) with ld = 4 dims[cut] (a10, L331-L333, written straight
 *                    in the canonical layout: a11-a13 fused).  d_out must not overlap d_psi.
 * Errors: -1 bad argument (dims outside 1..256), -2 workspace too small. */
size_t pepo_site_gram_ws_bytes(const int* h_dims, int nlegs, int cut_leg);
int pepo_site_gram(const double* d_psi, const int* h_dims, int nlegs, int cut_leg,
                   const double* const* h_w2, double* d_C, void* d_ws, size_t ws_bytes, void* stream);
int pepo_site_apply(const double* d_psi, const int* h_dims, int nlegs, int cut_leg, const double* d_W,
                    int chi_new, double* d_out, void* stream);

/* Cholesky-QR (eq. (10)): C = A^T A, R = chol(C) upper, Q = A R^{-1} (via the inverted
 * triangular factor, the paper's Rinv slots L140).  d_Q: m x n (ldq = lda), d_R: n x n
 * (ldr = n, strictly-lower part zeroed).  d_info (device int): 0 ok, j>0 = pivot j <= 0
 * (the paper's potrf_info).  Q is left unspecified when info != 0. */
size_t pepo_cholqr_ws_bytes(long long m, int n);
int pepo_cholqr(const double* d_A, long long m, int n, long long lda, double* d_Q, double* d_R,
                int* d_info, void* d_ws, size_t ws_bytes, void* stream);

/* Householder QR (R13), reduced: A (m x n, column-major, lda) = Q R,
 * k = min(m,n), d_Q m x k (ldq = m), d_R k x n (ldr = k, upper trapezoidal).  A is not
 * modified.  Works for m < n and rank-deficient A. */
size_t pepo_householder_ws_bytes(long long m, int n);
int pepo_householder_qr(const double* d_A, long long m, int n, long long lda, double* d_Q,
                        double* d_R, void* d_ws, size_t ws_bytes, void* stream);

/* One-sided Jacobi SVD (a9, eq. (11)-(12) PAPER.md:L233-L241): A (m x n column-major, lda)
 * = U diag(s) V^T with r = min(m,n); d_U m x r (ldu = m), d_s r (descending), d_V n x r
 * (ldv = n).  d_sweeps (device int, may be NULL) gets the sweep count. */
size_t pepo_svd_ws_bytes(int m, int n);
int pepo_svd_jacobi(const double* d_A, int m, int n, int lda, double* d_U, double* d_s,
                    double* d_V, int* d_sweeps, void* d_ws, size_t ws_bytes, void* stream);

/* C (M x N, ldc) = op(A) op(B) on the fp64 tensor cores; transA/transB = 0 ('N') or 1 ('T'),
 * column-major operands (a10 reconstruction GEMM). */
int pepo_dgemm(int transA, int transB, long long M, int N, int K, const double* d_A,
               long long lda, const double* d_B, long long ldb, double* d_C, long long ldc,
               void* stream);

/* fp64 tensor-pipe yardstick ("measure a large DGEMM in the same run"): launches
 * ctas_per_sm (1..8) CTAs of 8 warps per SM, every warp issuing iters x 16 register-only
 * DMMA.8x8x4 (the instruction every GEMM of this library is built on); *h_flops = floating-point
 * operations of the launch.  The caller times it with CUDA events on `stream`.  d_sink: one device
 * double (never written in practice). */
int pepo_dmma_peak(int iters, int ctas_per_sm, double* d_sink, double* h_flops, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* PEPO_H_ */
