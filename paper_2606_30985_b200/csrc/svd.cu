// svd.cu - hand-written one-sided (Hestenes) Jacobi SVD of the small bond core, the
// truncation rule eq. (11) and the Vidal normalisation eq. (12) (PAPER.md:L233-L241,
// L277-L279, L329-L330; a9), all on the device (the paper does the threshold on the host,
// L344).  K (r1 x r2) = U diag(s) V^T.
//
// One CTA per problem.  Columns of G (= K or K^T, tall) are orthogonalised pairwise in the
// round-robin ("circle") order, one warp per pair; V accumulates the rotations.  Columns whose
// squared norm is below 1e-30 ||K||_F^2 are numerically zero (the rank threshold of eq. (11)
// is 1e-11 s_0, i.e. 1e-22 in squared norm) and are not rotated, so exactly rank-deficient
// cores (the norm at early layers) converge.
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

// 64-bit butterfly exchange through the two 32-bit halves (keeps the compiler from swapping the
// halves around a register-pair shuffle) and the reductions built on it.  warp_sum3 interleaves
// three independent reductions so their shuffle latencies overlap.
__device__ __forceinline__ double shfl_xor_f64(double v, int o) {
  int lo = __double2loint(v), hi = __double2hiint(v);
  lo = __shfl_xor_sync(0xffffffffu, lo, o);
  hi = __shfl_xor_sync(0xffffffffu, hi, o);
  return __hiloint2double(hi, lo);
}
__device__ __forceinline__ double warp_sum1(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += shfl_xor_f64(v, o);
  return v;
}
__device__ __forceinline__ void warp_sum3(double& a, double& b, double& c) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const double a2 = shfl_xor_f64(a, o), b2 = shfl_xor_f64(b, o), c2 = shfl_xor_f64(c, o);
    a += a2; b += b2; c += c2;
  }
}

// Short-latency fp64 reciprocal square root / reciprocal for the rotation parameters: hardware
// approximation (MUFU.RSQ64H / RCP64H, ~2^-22) + two Newton steps (-> a few ulp).  The library
// sqrt()/division are long dependent instruction sequences with special-case branches and sit on
// the critical path of every pair rotation.  Arguments here are positive, finite and normal
// (guarded by the noise test); a rotation stays orthogonal to rounding for any c, s = c t.
__device__ __forceinline__ double fast_rsqrt(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double hx = 0.5 * x;
#pragma unroll
  for (int it = 0; it < 2; it++) {
    const double e = fma(-hx * y, y, 0.5);
    y = fma(y, e, y);
  }
  return y;
}
__device__ __forceinline__ double fast_rcp(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
#pragma unroll
  for (int it = 0; it < 2; it++) {
    const double e = fma(-x, y, 1.0);
    y = fma(y, e, y);
  }
  return y;
}
// (c, s) of the Jacobi rotation that orthogonalises two columns with squared norms al, be and
// inner product ga: t = sgn(zeta)/(|zeta| + sqrt(1 + zeta^2)), zeta = (be - al)/(2 ga).
__device__ __forceinline__ void jacobi_cst(double al, double be, double ga, double& cs, double& sn, double& tt) {
  const double d = be - al, g2 = 2.0 * ga;
  const double h = fma(d, d, g2 * g2);
  const double r = h * fast_rsqrt(h);                      // sqrt(d^2 + g2^2) > 0
  tt = g2 * fast_rcp(d + copysign(r, d));
  cs = fast_rsqrt(fma(tt, tt, 1.0));
  sn = cs * tt;
}
__device__ __forceinline__ void jacobi_cs(double al, double be, double ga, double& cs, double& sn) {
  double tt;
  jacobi_cst(al, be, ga, cs, sn, tt);
}

__global__ void __launch_bounds__(1024) jacobi_svd_kernel(SvdBatch b, double tol, int max_sweeps) {
  extern __shared__ double snorm[];     // Nc doubles
  __shared__ double s_red[32];
  __shared__ int s_rot;
  __shared__ double s_ref;
  const int t = blockIdx.x;
  const int r1 = b.r1[t], r2 = b.r2[t];
  const bool tr = r1 < r2;
  const int M = tr ? r2 : r1, Nc = tr ? r1 : r2;
  const double* K = b.K[t];
  const int ldk = b.ldk[t];
  double* G = b.G[t];
  double* V = b.V[t];
  if (b.orient[t] != nullptr && threadIdx.x == 0) *b.orient[t] = 0;   // this kernel never flips a square core
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nw = blockDim.x >> 5;
  // load
  double fro = 0.0;
  for (int e = tid; e < M * Nc; e += blockDim.x) {
    int i = e % M, j = e / M;
    double v = tr ? K[j + (long long)i * ldk] : K[i + (long long)j * ldk];
    G[e] = v;
    fro += v * v;
  }
  for (int e = tid; e < Nc * Nc; e += blockDim.x) V[e] = ((e % Nc) == (e / Nc)) ? 1.0 : 0.0;
  fro = warp_sum(fro);
  if (lane == 0) s_red[warp] = fro;
  __syncthreads();
  if (tid == 0) {
    double s = 0.0;
    for (int w = 0; w < nw; w++) s += s_red[w];
    s_ref = s;
  }
  __syncthreads();
  const double noise2 = 1e-30 * s_ref;
  const int npos = (Nc & 1) ? Nc + 1 : Nc;
  int sweeps = 0;
  if (Nc >= 2 && s_ref > 0.0 && isfinite(s_ref)) {
    for (int sw = 0; sw < max_sweeps; sw++) {
      if (tid == 0) s_rot = 0;
      __syncthreads();
      for (int r = 0; r < npos - 1; r++) {
        for (int i = warp; i < npos / 2; i += nw) {
          int a, c;
          if (i == 0) { a = npos - 1; c = r; }
          else { a = (r + i) % (npos - 1); c = (r - i + npos - 1) % (npos - 1); }
          int p = min(a, c), q = max(a, c);
          if (q >= Nc) continue;
          double* gp = G + (long long)p * M;
          double* gq = G + (long long)q * M;
          double al = 0.0, be = 0.0, ga = 0.0;
          for (int k = lane; k < M; k += 32) {
            double x = gp[k], y = gq[k];
            al += x * x; be += y * y; ga += x * y;
          }
          al = warp_sum(al); be = warp_sum(be); ga = warp_sum(ga);
          if (al < noise2 || be < noise2 || !(al > 0.0) || !(be > 0.0)) continue;
          if (fabs(ga) <= tol * sqrt(al) * sqrt(be)) continue;
          double zeta = (be - al) / (2.0 * ga);
          double tt = ((zeta >= 0.0) ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
          double cs = 1.0 / sqrt(1.0 + tt * tt), sn = cs * tt;
          for (int k = lane; k < M; k += 32) {
            double x = gp[k], y = gq[k];
            gp[k] = cs * x - sn * y;
            gq[k] = sn * x + cs * y;
          }
          double* vp = V + (long long)p * Nc;
          double* vq = V + (long long)q * Nc;
          for (int k = lane; k < Nc; k += 32) {
            double x = vp[k], y = vq[k];
            vp[k] = cs * x - sn * y;
            vq[k] = sn * x + cs * y;
          }
          if (lane == 0) s_rot = 1;
        }
        __syncthreads();
      }
      sweeps = sw + 1;
      int rot = s_rot;
      __syncthreads();
      if (!rot) break;
    }
  }
  // singular values = column norms; sort descending (rank by counting, ties by index)
  for (int j = warp; j < Nc; j += nw) {
    double s = 0.0;
    for (int k = lane; k < M; k += 32) { double x = G[(long long)j * M + k]; s += x * x; }
    s = warp_sum(s);
    if (lane == 0) snorm[j] = sqrt(s);
  }
  __syncthreads();
  for (int j = tid; j < Nc; j += blockDim.x) {
    double sj = snorm[j];
    int rank = 0;
    for (int l = 0; l < Nc; l++) {
      double sl = snorm[l];
      rank += (sl > sj || (sl == sj && l < j)) ? 1 : 0;
    }
    b.order[t][rank] = j;
    b.sv[t][rank] = sj;
  }
  if (tid == 0 && b.sweeps[t]) *b.sweeps[t] = sweeps;
}


// ---------------------------------------------------------------------------------------------
// Cluster version: the columns of [G; V] (length LEN = M + Nc) live in the shared memory of a
// thread-block cluster of CS CTAs, two blocks of `bs` columns per CTA (2 CS blocks in all).
// One sweep = all pairs inside every block, then 2 CS - 1 super-rounds in which every CTA
// orthogonalises its two resident blocks against each other (bs local rounds of bs disjoint
// pairs, one warp per pair, __syncthreads only) and the blocks then move one position along
// the round-robin circle through distributed shared memory (staged in registers between two
// cluster barriers).  No global-memory traffic inside the iteration.
// ---------------------------------------------------------------------------------------------
constexpr int JC_THREADS = 1024;
constexpr int JC_STAGE = 26;            // doubles staged per thread during a block exchange
constexpr size_t JC_SMEM_CAP = 200 * 1024;

// cp, cq: 16-byte aligned columns; MP2 = (padded) number of double2 of the G part that enter the
// inner products, LEN2 = double2 per column (G part + optional V part); pad entries are zero.
__device__ __forceinline__ bool rotate_pair(double* cp, double* cq, int MP2, int LEN2, double tol2,
                                            double noise2, int lane) {
  double2* p2 = reinterpret_cast<double2*>(cp);
  double2* q2 = reinterpret_cast<double2*>(cq);
  double al = 0.0, be = 0.0, ga = 0.0;
  for (int k = lane; k < MP2; k += 32) {
    double2 x = p2[k], y = q2[k];
    al += x.x * x.x; be += y.x * y.x; ga += x.x * y.x;
    al += x.y * x.y; be += y.y * y.y; ga += x.y * y.y;
  }
  warp_sum3(al, be, ga);
  if (al < noise2 || be < noise2 || !(al > 0.0) || !(be > 0.0)) return false;
  if (ga * ga <= tol2 * al * be) return false;          // |ga| <= tol ||p|| ||q||
  // tan of the rotation angle, smaller root: t = sgn(zeta)/(|zeta| + sqrt(1 + zeta^2)), zeta =
  // (be - al)/(2 ga), written with one sqrt and one division
  double cs, sn;
  jacobi_cs(al, be, ga, cs, sn);
  for (int k = lane; k < LEN2; k += 32) {
    double2 x = p2[k], y = q2[k];
    double2 xn, yn;
    xn.x = cs * x.x - sn * y.x; yn.x = sn * x.x + cs * y.x;
    xn.y = cs * x.y - sn * y.y; yn.y = sn * x.y + cs * y.y;
    p2[k] = xn; q2[k] = yn;
  }
  return true;
}

template <int STAGE, int NREG>
__global__ void __launch_bounds__(JC_THREADS, 1)
jacobi_cluster_kernel(SvdBatch b, double tol, int max_sweeps, int bs, int CS, int with_v, int LEN,
                      int precond_min, int pw) {
  extern __shared__ __align__(16) double jsm[];
  cg::cluster_group cluster = cg::this_cluster();
  const int crank = (int)cluster.block_rank();
  const int t = blockIdx.x / CS;
  const int r1 = b.r1[t], r2 = b.r2[t];
  const bool tr = r1 < r2;
  const int M = tr ? r2 : r1, Nc = tr ? r1 : r2;
  if (b.orient[t] != nullptr && crank == 0 && threadIdx.x == 0) *b.orient[t] = 0;   // never flips a square core
  // column layout: [G part: M, zero-padded to MP (even)] [V part: Nc, zero-padded, only with_v];
  // LEN (even, same for the whole launch) >= MP + (with_v ? Nc : 0)
  const int MP = (M + 1) & ~1;
  int Mj = M;                             // rows of the matrix the Jacobi iteration works on
  int MP2 = MP >> 1;
  const int LEN2 = LEN >> 1;
  const double tol2 = tol * tol;
  const double* K = b.K[t];
  const int ldk = b.ldk[t];
  // shared layout: cols[2][bs][LEN], ids[2][bs] (as double-aligned ints), scal[4]
  double* cols = jsm;
  int* ids = (int*)(cols + (size_t)2 * bs * LEN);
  double* scal = (double*)(ids + ((2 * bs + 3) & ~3));        // [0] partial fro, [1] rotated flag
  double* vbuf = scal + 4;                                    // pw x (MP + 2): Householder panel
  const int PW = (2 * bs + 3) & ~3;                           // pitch of the small matrices W, J
  double* Wm = vbuf + (size_t)pw * (MP + 2);                  // block form: Gram of the resident columns
  double* Jm = Wm + (size_t)2 * bs * PW;                      //             accumulated rotations
  double* rc = Jm + (size_t)2 * bs * PW;
  double* rs = rc + bs;
  double* nrm = rs + bs;                                      // squared norms of the resident columns [2 bs]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nw = JC_THREADS / 32;
  const int blk_of_slot[2] = {crank, 2 * CS - 1 - crank};
  // ---- load ---------------------------------------------------------------------------------
  double fro = 0.0;
  for (int e = tid; e < 2 * bs * LEN; e += JC_THREADS) {
    int k = e % LEN, ci = e / LEN;               // ci = slot*bs + i
    int j = blk_of_slot[ci / bs] * bs + (ci % bs);
    double v = 0.0;
    if (j < Nc) {
      if (k < M) { v = tr ? K[j + (long long)k * ldk] : K[k + (long long)j * ldk]; fro += v * v; }
      else if (with_v && k >= MP) v = (k - MP == j) ? 1.0 : 0.0;
    }
    cols[e] = v;
  }
  for (int e = tid; e < 2 * bs; e += JC_THREADS) ids[e] = blk_of_slot[e / bs] * bs + (e % bs);
  __shared__ double s_red[32];
  fro = warp_sum(fro);
  if (lane == 0) s_red[warp] = fro;
  __syncthreads();
  if (tid == 0) {
    double s = 0.0;
    for (int w = 0; w < nw; w++) s += s_red[w];
    scal[0] = s; scal[1] = 0.0;
  }
  cluster.sync();
  double ref = 0.0;
  for (int c = 0; c < CS; c++) ref += cluster.map_shared_rank(scal, c)[0];
  const double noise2 = 1e-30 * ref;
  // ---- QR preconditioning (Drmac-Veselic): A = Q R by Householder reflections on the columns
  // resident in the cluster, then iterate on L = R^T (Nc x Nc).  R R^T is one LR step closer to
  // diagonal than R^T R, which roughly halves the number of sweeps; Q is never needed because
  // the bridges are rebuilt from the untouched core K (svd_bridge_nov_kernel).
  const bool precond = !with_v && precond_min > 0 && Nc >= precond_min && ref > 0.0 && isfinite(ref);
  if (precond) {
    // panels of <= pw consecutive columns (inside one block, i.e. inside one CTA): the owner
    // factors the panel locally, broadcasts its reflectors once, every CTA applies them to its
    // later columns: two cluster barriers per panel instead of per column.
    const int VS = MP + 2;                               // stride of one reflector in vbuf
    const int nblk = (Nc + bs - 1) / bs;
    for (int blk = 0; blk < nblk; blk++) {
      const int owner = blk < CS ? blk : 2 * CS - 1 - blk;
      for (int p0 = 0; p0 < bs; p0 += pw) {
        const int j0 = blk * bs + p0;
        if (j0 >= Nc) break;
        const int j1 = min(min(j0 + pw, (blk + 1) * bs), Nc);
        if (crank == owner) {
          double* pcols = cols + ((size_t)(blk < CS ? 0 : 1) * bs + p0) * LEN;   // panel columns
          for (int j = j0; j < j1; j++) {
            double* col = pcols + (size_t)(j - j0) * LEN;
            double* vl = vbuf + (size_t)(j - j0) * VS;
            if (warp == 0) {
              double ss = 0.0;
              for (int k = j + lane; k < M; k += 32) { double x = col[k]; ss += x * x; }
              ss = warp_sum(ss);
              const double ajj = col[j];
              const double nrm = sqrt(ss);
              const double alpha = (ajj > 0.0) ? -nrm : nrm;
              const double vj = ajj - alpha;
              const double vtv = ss - ajj * ajj + vj * vj;
              for (int k = j + lane; k < M; k += 32) {
                vl[k] = (k == j) ? vj : col[k];
                col[k] = (k == j) ? alpha : 0.0;               // column j of R
              }
              if (lane == 0) vl[MP] = (vtv > 1e-290) ? 2.0 / vtv : 0.0;     // identity for underflow-level columns
            }
            __syncthreads();
            const double tau = vl[MP];
            if (tau != 0.0) {
              for (int jj = j + 1 + warp; jj < j1; jj += nw) {
                double* c2 = pcols + (size_t)(jj - j0) * LEN;
                double w = 0.0;
                for (int k = j + lane; k < M; k += 32) w += vl[k] * c2[k];
                w = warp_sum(w) * tau;
                for (int k = j + lane; k < M; k += 32) c2[k] -= w * vl[k];
              }
            }
            __syncthreads();
          }
          const int tot = (j1 - j0) * VS;
          for (int c = 0; c < CS; c++) {
            if (c == crank) continue;
            double* rv = cluster.map_shared_rank(vbuf, c);
            for (int e = tid; e < tot; e += JC_THREADS) rv[e] = vbuf[e];
          }
        }
        cluster.sync();
        for (int ci = warp; ci < 2 * bs; ci += nw) {
          const int id = ids[ci];
          if (id < j1 || id >= Nc) continue;
          double* col = cols + (size_t)ci * LEN;
          for (int j = j0; j < j1; j++) {
            const double* vl = vbuf + (size_t)(j - j0) * VS;
            const double tau = vl[MP];
            if (tau == 0.0) continue;
            double w = 0.0;
            for (int k = j + lane; k < M; k += 32) w += vl[k] * col[k];
            w = warp_sum(w) * tau;
            for (int k = j + lane; k < M; k += 32) col[k] -= w * vl[k];
          }
        }
        cluster.sync();
      }
    }
    // transpose R through the global scratch G (ld M): new column i = row i of R
    double* Gs = b.G[t];
    for (int ci = warp; ci < 2 * bs; ci += nw) {
      const int id = ids[ci];
      if (id >= Nc) continue;
      const double* col = cols + (size_t)ci * LEN;
      for (int k = lane; k < Nc; k += 32) Gs[k + (size_t)id * M] = (k <= id) ? col[k] : 0.0;
    }
    __threadfence();
    cluster.sync();
    for (int ci = warp; ci < 2 * bs; ci += nw) {
      const int id = ids[ci];
      double* col = cols + (size_t)ci * LEN;
      for (int k = lane; k < LEN; k += 32)
        col[k] = (id < Nc && k < Nc && k >= id) ? Gs[id + (size_t)k * M] : 0.0;
    }
    __syncthreads();
    cluster.sync();
    Mj = Nc;
    MP2 = ((Nc + 1) & ~1) >> 1;
  }
  int sweeps = 0;
  const bool active = (Nc >= 2) && (ref > 0.0) && isfinite(ref);
  double* top = cols;
  double* bot = cols + (size_t)bs * LEN;
  const int nb2 = (bs & 1) ? bs + 1 : bs;        // circle size for the intra-block pairs
  for (int sw = 0; active && sw < max_sweeps; sw++) {
    bool rot = false;
    // intra-block pairs (both blocks at once)
    for (int r = 0; r < nb2 - 1; r++) {
      for (int w = warp; w < nb2; w += nw) {
        int slot = w / (nb2 / 2), i = w % (nb2 / 2);
        int a, c;
        if (i == 0) { a = nb2 - 1; c = r; }
        else { a = (r + i) % (nb2 - 1); c = (r - i + nb2 - 1) % (nb2 - 1); }
        if (a >= bs || c >= bs) continue;
        double* base = slot ? bot : top;
        rot |= rotate_pair(base + (size_t)min(a, c) * LEN, base + (size_t)max(a, c) * LEN, MP2, LEN2, tol2, noise2, lane);
      }
      __syncthreads();
    }
    // squared norms of the resident columns, fresh once per sweep (carried through the super-rounds)
    for (int ci = warp; ci < 2 * bs; ci += nw) {
      const double2* c2 = reinterpret_cast<const double2*>(cols + (size_t)ci * LEN);
      double a0 = 0.0;
      for (int k = lane; k < MP2; k += 32) { const double2 x = c2[k]; a0 = fma(x.x, x.x, a0); a0 = fma(x.y, x.y, a0); }
      a0 = warp_sum1(a0);
      if (lane == 0) nrm[ci] = a0;
    }
    __syncthreads();
    // super-rounds
    for (int sr = 0; sr < 2 * CS - 1; sr++) {
      if (NREG > 0) {
        // The pair rotations are shared-memory-bandwidth and latency bound.  Warp i keeps top column
        // i in registers for the bs rounds of the super-round, so only the bottom column of each pair
        // moves through shared memory; the squared norms of the columns are carried along (al in a
        // register, the bottom norms in nrm[]) and updated by ||p'||^2 = al - t ga, ||q'||^2 = be +
        // t ga, so that a rotation costs ONE warp reduction (the inner product) instead of three.
        // The carried norms are refreshed from the columns once per sweep (above) and whenever an
        // update cancels more than two digits.
        double2 tp[NREG > 0 ? NREG : 1];
        const bool own = warp < bs;
        double2* tcol = reinterpret_cast<double2*>(top + (size_t)(own ? warp : 0) * LEN);
        double al = 0.0;
        if (own) {
#pragma unroll
          for (int q = 0; q < NREG; q++) {
            const int k = lane + 32 * q;
            tp[q] = (k < LEN2) ? tcol[k] : make_double2(0.0, 0.0);
          }
          al = nrm[warp];
        }
        for (int r = 0; r < bs; r++) {
          if (own) {
            int j = warp + r; if (j >= bs) j -= bs;
            double2* cq = reinterpret_cast<double2*>(bot + (size_t)j * LEN);
            double2 y[NREG > 0 ? NREG : 1];
            double ga0 = 0.0, ga1 = 0.0;
#pragma unroll
            for (int q = 0; q < NREG; q++) {
              const int k = lane + 32 * q;
              y[q] = (k < LEN2) ? cq[k] : make_double2(0.0, 0.0);
              if (k < MP2) { ga0 = fma(tp[q].x, y[q].x, ga0); ga1 = fma(tp[q].y, y[q].y, ga1); }
            }
            const double be = nrm[bs + j];
            const double ga = warp_sum1(ga0 + ga1);
            if (al >= noise2 && be >= noise2 && ga * ga > tol2 * al * be) {
              double cs, sn, tt;
              jacobi_cst(al, be, ga, cs, sn, tt);
#pragma unroll
              for (int q = 0; q < NREG; q++) {
                const int k = lane + 32 * q;
                const double2 x = tp[q];
                tp[q].x = cs * x.x - sn * y[q].x; tp[q].y = cs * x.y - sn * y[q].y;
                y[q].x = sn * x.x + cs * y[q].x; y[q].y = sn * x.y + cs * y[q].y;
                if (k < LEN2) cq[k] = y[q];
              }
              const double tg = tt * ga;
              double aln = al - tg, ben = be + tg;
              if (aln < 0.01 * al || ben < 0.01 * be) {         // heavy cancellation (rare): fresh norms
                double a0 = 0.0, b0 = 0.0, z0 = 0.0;
#pragma unroll
                for (int q = 0; q < NREG; q++) {
                  if (lane + 32 * q < MP2) {
                    a0 = fma(tp[q].x, tp[q].x, a0); a0 = fma(tp[q].y, tp[q].y, a0);
                    b0 = fma(y[q].x, y[q].x, b0); b0 = fma(y[q].y, y[q].y, b0);
                  }
                }
                warp_sum3(a0, b0, z0);
                aln = a0; ben = b0;
              }
              al = aln;
              if (lane == 0) nrm[bs + j] = ben;
              rot = true;
            }
          }
          __syncthreads();
        }
        if (own) {
#pragma unroll
          for (int q = 0; q < NREG; q++) {
            const int k = lane + 32 * q;
            if (k < LEN2) tcol[k] = tp[q];
          }
          if (lane == 0) nrm[warp] = al;
        }
        __syncthreads();
      } else {
        for (int r = 0; r < bs; r++) {
          for (int i = warp; i < bs; i += nw) {
            int j = i + r; if (j >= bs) j -= bs;
            rot |= rotate_pair(top + (size_t)i * LEN, bot + (size_t)j * LEN, MP2, LEN2, tol2, noise2, lane);
          }
          __syncthreads();
        }
      }
      if (CS > 1) {
        cluster.sync();                           // A: every CTA finished computing
        const int per = bs * LEN;                 // doubles per block
        // sources of the new top / bottom blocks
        const double* src_top; const int* src_top_id;
        if (crank == 0) { src_top = nullptr; src_top_id = nullptr; }
        else if (crank == 1) { src_top = cluster.map_shared_rank(bot, 0); src_top_id = cluster.map_shared_rank(ids + bs, 0); }
        else { src_top = cluster.map_shared_rank(top, crank - 1); src_top_id = cluster.map_shared_rank(ids, crank - 1); }
        const double* src_bot; const int* src_bot_id;
        if (crank == CS - 1) { src_bot = top; src_bot_id = ids; }
        else { src_bot = cluster.map_shared_rank(bot, crank + 1); src_bot_id = cluster.map_shared_rank(ids + bs, crank + 1); }
        double stage[STAGE];
        int id_stage = -1;
        double nrm_stage = 0.0;
        const double* src_top_nrm = src_top ? (const double*)cluster.map_shared_rank(nrm, crank == 1 ? 0 : crank - 1) + (crank == 1 ? bs : 0) : nullptr;
        const double* src_bot_nrm = (crank == CS - 1) ? nrm : (const double*)cluster.map_shared_rank(nrm, crank + 1) + bs;
#pragma unroll
        for (int q = 0; q < STAGE; q++) {
          int e = tid + q * JC_THREADS;
          double v = 0.0;
          if (e < per) { if (src_top) v = src_top[e]; }
          else if (e < 2 * per) v = src_bot[e - per];
          stage[q] = v;
        }
        if (tid < bs) { if (src_top_id) { id_stage = src_top_id[tid]; nrm_stage = src_top_nrm[tid]; } }
        else if (tid < 2 * bs) { id_stage = src_bot_id[tid - bs]; nrm_stage = src_bot_nrm[tid - bs]; }
        cluster.sync();                           // B: every CTA finished reading
#pragma unroll
        for (int q = 0; q < STAGE; q++) {
          int e = tid + q * JC_THREADS;
          if (e < per) { if (src_top) top[e] = stage[q]; }
          else if (e < 2 * per) bot[e - per] = stage[q];
        }
        if (tid < bs) { if (src_top_id) { ids[tid] = id_stage; nrm[tid] = nrm_stage; } }
        else if (tid < 2 * bs) { ids[tid] = id_stage; nrm[tid] = nrm_stage; }
        __syncthreads();
      }
    }
    sweeps = sw + 1;
    // cluster-wide "any rotation" (uniform decision)
    int anyrot = __syncthreads_or(rot ? 1 : 0);
    if (tid == 0) scal[1] = anyrot ? 1.0 : 0.0;
    cluster.sync();
    double tot = 0.0;
    for (int c = 0; c < CS; c++) tot += cluster.map_shared_rank(scal, c)[1];
    cluster.sync();                               // flags read before anyone overwrites them
    if (tot == 0.0) break;
  }
  // ---- write back: column id -> global column id of G / V, norm -> sv scratch (unsorted) -------
  double* G = b.G[t];
  double* V = b.V[t];
  double* svu = b.V[t] + (size_t)Nc * Nc;         // unsorted norms: Nc doubles after V (caller sizes V as Nc*(Nc+1))
  for (int ci = warp; ci < 2 * bs; ci += nw) {
    int id = ids[ci];
    if (id >= Nc) continue;
    const double* col = cols + (size_t)ci * LEN;
    double s = 0.0;
    for (int k = lane; k < Mj; k += 32) { double x = col[k]; s += x * x; G[(size_t)id * M + k] = x; }
    if (with_v) for (int k = lane; k < Nc; k += 32) V[(size_t)id * Nc + k] = col[MP + k];
    s = warp_sum(s);
    if (lane == 0) svu[id] = sqrt(s);
  }
  __threadfence();
  cluster.sync();
  if (crank == 0) {
    for (int j = tid; j < Nc; j += JC_THREADS) {
      double sj = svu[j];
      int rank = 0;
      for (int l = 0; l < Nc; l++) {
        double sl = svu[l];
        rank += (sl > sj || (sl == sj && l < j)) ? 1 : 0;
      }
      b.order[t][rank] = j;
      b.sv[t][rank] = sj;
    }
    if (tid == 0 && b.sweeps[t]) *b.sweeps[t] = sweeps;
  }
}

// ---------------------------------------------------------------------------------------------
// Hot-path cluster kernel (no V, 2 <= CS, LEN = 32 NREG doubles per column, bs <= 16).
// Differences from jacobi_cluster_kernel, each measured on the 4x4 chi = 60 cores (N = 240):
//  * 16 lanes per column pair, two pairs per warp: the scalar part of a rotation (reduction,
//    convergence test, rotation parameters) is issued once for two pairs, and 8 warps instead of
//    15 compete for the issue slots and the fp64 pipe of the SM;
//  * carried squared norms (||p'||^2 = al - t ga, ||q'||^2 = be + t ga, refreshed from the columns
//    once per sweep and after heavy cancellation): one reduction per rotation instead of three;
//  * ping-pong column buffers: in the last round of a super-round the rotated columns are stored
//    straight into the neighbour's spare buffer through DSMEM (the top column from registers), so
//    the block exchange costs ONE cluster barrier and no extra pass over the columns;
//  * the cluster-wide "any rotation" flag rides on the last barrier of the sweep.
// ---------------------------------------------------------------------------------------------
constexpr int J16_THREADS = 512;       // NREG <= 8 (columns of <= 256 doubles); 256 threads above (255 registers)

__device__ __forceinline__ double half_sum1(double v) {
#pragma unroll
  for (int o = 8; o > 0; o >>= 1) v += shfl_xor_f64(v, o);
  return v;
}
__device__ __forceinline__ void half_sum3(double& a, double& b, double& c) {
#pragma unroll
  for (int o = 8; o > 0; o >>= 1) {
    const double a2 = shfl_xor_f64(a, o), b2 = shfl_xor_f64(b, o), c2 = shfl_xor_f64(c, o);
    a += a2; b += b2; c += c2;
  }
}
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

template <int NREG, int NTHR>
__global__ void __launch_bounds__(NTHR, 1)
jacobi_c16_kernel(SvdBatch b, double tol, int max_sweeps, int bs, int CS, int precond_min, int pw,
                  double early2, int keep_hint, int nfull, double theta, int orient_mode) {
  constexpr int LEN = 32 * NREG, LEN2 = 16 * NREG;
  extern __shared__ __align__(16) double jsm[];
  cg::cluster_group cluster = cg::this_cluster();
  const int crank = (int)cluster.block_rank();
  const int t = blockIdx.x / CS;
  const int r1 = b.r1[t], r2 = b.r2[t];
  bool tr = r1 < r2;                      // a square core may still be flipped below (orient_mode)
  const int M = tr ? r2 : r1, Nc = tr ? r1 : r2;
  const int MP = (M + 1) & ~1;
  int Mj = M;
  const double tol2 = tol * tol;
  const double* K = b.K[t];
  const int ldk = b.ldk[t];
  // shared layout: colbuf[2][2 bs][LEN], nrmbuf[2][2 bs], idbuf[2][2 bs], flags[16], scal[4], vbuf
  const int per = 2 * bs * LEN;
  double* colbuf = jsm;
  double* nrmbuf = colbuf + (size_t)2 * per;
  int* idbuf = (int*)(nrmbuf + 4 * bs);
  double* flags = (double*)(idbuf + ((4 * bs + 3) & ~3));
  double* scal = flags + 16;
  double* vbuf = scal + 4;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nw = NTHR / 32;
  int cur = 0;
  double* cols = colbuf;
  int* ids = idbuf;
  // ---- load ---------------------------------------------------------------------------------
  double fro = 0.0;
  for (int e = tid; e < per; e += NTHR) {
    const int k = e % LEN, ci = e / LEN;
    const int j = ((ci / bs) ? 2 * CS - 1 - crank : crank) * bs + (ci % bs);
    double v = 0.0;
    if (j < Nc && k < M) { v = tr ? K[j + (long long)k * ldk] : K[k + (long long)j * ldk]; fro += v * v; }
    cols[e] = v;
  }
  for (int e = tid; e < 2 * bs; e += NTHR) ids[e] = ((e / bs) ? 2 * CS - 1 - crank : crank) * bs + (e % bs);
  __shared__ double s_red[32];
  __shared__ int s_flag;                  // a pair with cos^2 > early2 was rotated in this sweep
  fro = warp_sum1(fro);
  if (lane == 0) s_red[warp] = fro;
  __syncthreads();
  if (tid == 0) {
    double s = 0.0;
    for (int w = 0; w < nw; w++) s += s_red[w];
    scal[0] = s;
    s_flag = 0;
  }
  cluster.sync();
  double ref = 0.0;
  for (int c = 0; c < CS; c++) ref += cluster.map_shared_rank(scal, c)[0];
  const double noise2 = 1e-30 * ref;
  // ---- QR preconditioning (as in jacobi_cluster_kernel): iterate on L = R^T ------------------
  const bool precond = precond_min > 0 && Nc >= precond_min && ref > 0.0 && isfinite(ref);
  // ---- which of K, K^T gets the QR (square cores; dense.cuh, launch_svd_jacobi `orient`) -------
  // An unpivoted QR preconditions well when the COLUMNS it sweeps are strongly graded; which side of a
  // Schmidt-dressed core is the graded one depends on the bond (measured: 9 sweeps vs 19-21).  The
  // grading is measured as the variance of ln ||.||^2 over the columns and over the rows; every CTA of
  // the cluster forms the same sums in the same order, so the decision is uniform and a function of K.
  int* orient_out = b.orient[t];
  bool flip = false;
  if (precond && r1 == r2 && orient_out != nullptr && orient_mode > 0) {
    flip = orient_mode == 2;
    if (orient_mode == 1) {
      for (int k = tid; k < M; k += NTHR) {             // row sums over my columns
        double a = 0.0;
        for (int ci = 0; ci < 2 * bs; ci++) { const double x = cols[(size_t)ci * LEN + k]; a = fma(x, x, a); }
        vbuf[k] = a;
      }
      double c1 = 0.0, c2 = 0.0;                        // my columns: sum ln, sum ln^2
      for (int ci = warp; ci < 2 * bs; ci += nw) {
        if (ids[ci] >= Nc) continue;
        double a = 0.0;
        for (int k = lane; k < M; k += 32) { const double x = cols[(size_t)ci * LEN + k]; a = fma(x, x, a); }
        a = warp_sum1(a);
        const double l = log(fmax(a, noise2));
        c1 += l; c2 += l * l;
      }
      __syncthreads();                                  // s_red was read by thread 0 above
      if (lane == 0) { s_red[warp] = c1; s_red[16 + warp] = c2; }
      __syncthreads();
      if (tid == 0) {
        double a1 = 0.0, a2 = 0.0;
        for (int w = 0; w < nw; w++) { a1 += s_red[w]; a2 += s_red[16 + w]; }
        scal[1] = a1; scal[2] = a2;
      }
      cluster.sync();
      double C1 = 0.0, C2 = 0.0;
      for (int c = 0; c < CS; c++) { const double* sc = cluster.map_shared_rank(scal, c); C1 += sc[1]; C2 += sc[2]; }
      double q1 = 0.0, q2 = 0.0;                        // rows: full sums through DSMEM
      for (int k = tid; k < M; k += NTHR) {
        double a = 0.0;
        for (int c = 0; c < CS; c++) a += cluster.map_shared_rank(vbuf, c)[k];
        const double l = log(fmax(a, noise2));
        q1 += l; q2 += l * l;
      }
      q1 = warp_sum1(q1); q2 = warp_sum1(q2);
      if (lane == 0) { s_red[warp] = q1; s_red[16 + warp] = q2; }
      __syncthreads();
      double R1 = 0.0, R2 = 0.0;
      for (int w = 0; w < nw; w++) { R1 += s_red[w]; R2 += s_red[16 + w]; }
      const double varC = C2 - C1 * C1 / (double)Nc, varR = R2 - R1 * R1 / (double)M;
      flip = varR > varC;
      cluster.sync();                                   // vbuf and scal are free again (panel broadcast below)
    }
    if (flip) {
      tr = true;
      for (int e = tid; e < per; e += NTHR) {
        const int k = e % LEN, ci = e / LEN;
        const int j = ((ci / bs) ? 2 * CS - 1 - crank : crank) * bs + (ci % bs);
        cols[e] = (j < Nc && k < M) ? K[j + (long long)k * ldk] : 0.0;
      }
      __syncthreads();
    }
  }
  if (orient_out != nullptr && crank == 0 && tid == 0) *orient_out = flip ? 1 : 0;
  if (precond) {
    const int VS = MP + 2;
    const int nblk = (Nc + bs - 1) / bs;
    for (int blk = 0; blk < nblk; blk++) {
      const int owner = blk < CS ? blk : 2 * CS - 1 - blk;
      for (int p0 = 0; p0 < bs; p0 += pw) {
        const int j0 = blk * bs + p0;
        if (j0 >= Nc) break;
        const int j1 = min(min(j0 + pw, (blk + 1) * bs), Nc);
        if (crank == owner) {
          double* pcols = cols + ((size_t)(blk < CS ? 0 : 1) * bs + p0) * LEN;
          for (int j = j0; j < j1; j++) {
            double* col = pcols + (size_t)(j - j0) * LEN;
            double* vl = vbuf + (size_t)(j - j0) * VS;
            if (warp == 0) {
              double ss = 0.0;
              for (int k = j + lane; k < M; k += 32) { double x = col[k]; ss += x * x; }
              ss = warp_sum1(ss);
              const double ajj = col[j];
              const double nrm = sqrt(ss);
              const double alpha = (ajj > 0.0) ? -nrm : nrm;
              const double vj = ajj - alpha;
              const double vtv = ss - ajj * ajj + vj * vj;
              for (int k = j + lane; k < M; k += 32) {
                vl[k] = (k == j) ? vj : col[k];
                col[k] = (k == j) ? alpha : 0.0;
              }
              if (lane == 0) vl[MP] = (vtv > 1e-290) ? 2.0 / vtv : 0.0;
            }
            __syncthreads();
            const double tau = vl[MP];
            if (tau != 0.0) {
              for (int jj = j + 1 + warp; jj < j1; jj += nw) {
                double* c2 = pcols + (size_t)(jj - j0) * LEN;
                double w = 0.0;
                for (int k = j + lane; k < M; k += 32) w += vl[k] * c2[k];
                w = warp_sum1(w) * tau;
                for (int k = j + lane; k < M; k += 32) c2[k] -= w * vl[k];
              }
            }
            __syncthreads();
          }
          const int tot = (j1 - j0) * VS;
          for (int c = 0; c < CS; c++) {
            if (c == crank) continue;
            double* rv = cluster.map_shared_rank(vbuf, c);
            for (int e = tid; e < tot; e += NTHR) rv[e] = vbuf[e];
          }
        }
        cluster.sync();
        for (int ci = warp; ci < 2 * bs; ci += nw) {
          const int id = ids[ci];
          if (id < j1 || id >= Nc) continue;
          double* col = cols + (size_t)ci * LEN;
          for (int j = j0; j < j1; j++) {
            const double* vl = vbuf + (size_t)(j - j0) * VS;
            const double tau = vl[MP];
            if (tau == 0.0) continue;
            double w = 0.0;
            for (int k = j + lane; k < M; k += 32) w += vl[k] * col[k];
            w = warp_sum1(w) * tau;
            for (int k = j + lane; k < M; k += 32) col[k] -= w * vl[k];
          }
        }
        cluster.sync();
      }
    }
    double* Gs = b.G[t];
    for (int ci = warp; ci < 2 * bs; ci += nw) {
      const int id = ids[ci];
      if (id >= Nc) continue;
      const double* col = cols + (size_t)ci * LEN;
      for (int k = lane; k < Nc; k += 32) Gs[k + (size_t)id * M] = (k <= id) ? col[k] : 0.0;
    }
    __threadfence();
    cluster.sync();
    for (int ci = warp; ci < 2 * bs; ci += nw) {
      const int id = ids[ci];
      double* col = cols + (size_t)ci * LEN;
      for (int k = lane; k < LEN; k += 32)
        col[k] = (id < Nc && k < Nc && k >= id) ? Gs[id + (size_t)k * M] : 0.0;
    }
    __syncthreads();
    cluster.sync();
    Mj = Nc;
  }
  // ---- iteration ------------------------------------------------------------------------------
  int sweeps = 0;
  const bool active = (Nc >= 2) && (ref > 0.0) && isfinite(ref);
  // bl = LIVE columns per block (bs = layout stride of the shared buffers): after the deflation below
  // the top block lives in slots [0, bl) and the bottom block in slots [bs, bs + bl)
  int bl = bs;
  int nb2 = (bl & 1) ? bl + 1 : bl;
  const int half = lane >> 4, l16 = lane & 15;
  const int hw = 2 * warp + half;                        // half-warp index
  int nrw = (bl + 1) / 2;                                // warps that rotate pairs in the super-rounds
  // destinations of the block exchange (see header): my top block and my bottom block
  const int top_dst_rank = (crank == 0 || crank == CS - 1) ? crank : crank + 1;
  const int top_dst_slot = (crank == CS - 1) ? 1 : 0;
  const int bot_dst_rank = (crank == 0) ? 1 : crank - 1;
  const int bot_dst_slot = (crank == 0) ? 0 : 1;
  int nrt = nrw * 32;
  for (int sw = 0; active && sw < max_sweeps; sw++) {
    double* nrm = nrmbuf + cur * 2 * bs;
    bool big = false;                                    // this thread rotated a pair with cos^2 > early2 in this sweep
    // intra-block pairs of both resident blocks: nb2 half-warps per round
    for (int r = 0; r < nb2 - 1; r++) {
      if (hw < nb2) {
        const int slot = hw / (nb2 / 2), i = hw % (nb2 / 2);
        int a, c;
        if (i == 0) { a = nb2 - 1; c = r; }
        else { a = (r + i) % (nb2 - 1); c = (r - i + nb2 - 1) % (nb2 - 1); }
        const bool valid = (a < bl && c < bl);
        const int p = valid ? min(a, c) : 0, q = valid ? max(a, c) : 0;
        double2* p2 = reinterpret_cast<double2*>(cols + ((size_t)slot * bs + p) * LEN);
        double2* q2 = reinterpret_cast<double2*>(cols + ((size_t)slot * bs + q) * LEN);
        double2 x[NREG], y[NREG];
        double al = 0.0, be = 0.0, ga = 0.0;
#pragma unroll
        for (int u = 0; u < NREG; u++) {
          x[u] = p2[l16 + 16 * u]; y[u] = q2[l16 + 16 * u];
          al = fma(x[u].x, x[u].x, al); be = fma(y[u].x, y[u].x, be); ga = fma(x[u].x, y[u].x, ga);
          al = fma(x[u].y, x[u].y, al); be = fma(y[u].y, y[u].y, be); ga = fma(x[u].y, y[u].y, ga);
        }
        half_sum3(al, be, ga);
        const bool dorot = valid && al >= noise2 && be >= noise2 && ga * ga > tol2 * al * be;
        if (dorot) {
          double cs, sn;
          jacobi_cs(al, be, ga, cs, sn);
#pragma unroll
          for (int u = 0; u < NREG; u++) {
            double2 xn, yn;
            xn.x = cs * x[u].x - sn * y[u].x; yn.x = sn * x[u].x + cs * y[u].x;
            xn.y = cs * x[u].y - sn * y[u].y; yn.y = sn * x[u].y + cs * y[u].y;
            p2[l16 + 16 * u] = xn; q2[l16 + 16 * u] = yn;
          }
          big |= (ga * ga > early2 * al * be);
        }
      }
      __syncthreads();
    }
    // squared norms of the resident columns, fresh once per sweep
    for (int c0 = 0; c0 < 2 * bs; c0 += 2 * nw) {          // 2 bs is even: whole warps stay together
      const int cc = c0 + hw;
      const double2* c2 = reinterpret_cast<const double2*>(cols + (size_t)min(cc, 2 * bs - 1) * LEN);
      double a0 = 0.0, a1 = 0.0;
#pragma unroll
      for (int u = 0; u < NREG; u++) { const double2 x = c2[l16 + 16 * u]; a0 = fma(x.x, x.x, a0); a1 = fma(x.y, x.y, a1); }
      a0 = half_sum1(a0 + a1);
      if (l16 == 0 && cc < 2 * bs) nrm[cc] = a0;
    }
    __syncthreads();
    // super-rounds
    for (int sr = 0; sr < 2 * CS - 1; sr++) {
      const int nxt = cur ^ 1;
      if (warp < nrw) {
        const bool own = hw < bl;
        const int pi = own ? hw : 0;
        double* top = cols;
        double* bot = cols + (size_t)bs * LEN;
        double* nrmc = nrmbuf + cur * 2 * bs;
        double2 tp[NREG];
        const double2* tcol = reinterpret_cast<const double2*>(top + (size_t)pi * LEN);
#pragma unroll
        for (int u = 0; u < NREG; u++) tp[u] = tcol[l16 + 16 * u];
        double al = nrmc[pi];
        for (int r = 0; r < bl; r++) {
          int j = pi + r; if (j >= bl) j -= bl;
          double2* cq = reinterpret_cast<double2*>(bot + (size_t)j * LEN);
          double2 y[NREG];
          double ga0 = 0.0, ga1 = 0.0;
#pragma unroll
          for (int u = 0; u < NREG; u++) {
            y[u] = cq[l16 + 16 * u];
            ga0 = fma(tp[u].x, y[u].x, ga0); ga1 = fma(tp[u].y, y[u].y, ga1);
          }
          double be = nrmc[bs + j];
          const double ga = half_sum1(ga0 + ga1);
          const bool dorot = own && al >= noise2 && be >= noise2 && ga * ga > tol2 * al * be;
          const bool last = (r == bl - 1);
          if (__any_sync(0xffffffffu, dorot)) {
            double cs, sn, tt;
            jacobi_cst(dorot ? al : 1.0, dorot ? be : 2.0, dorot ? ga : 0.5, cs, sn, tt);
            double ics = fma(tt, tt, 1.0) * cs;                // 1 / cs
            if (!dorot) { cs = 1.0; sn = 0.0; tt = 0.0; ics = 1.0; }
            // in place, no temporaries: p' = cs p - sn q, then q' = sn p + cs q = t p' + q / cs
#pragma unroll
            for (int u = 0; u < NREG; u++) {
              tp[u].x = fma(cs, tp[u].x, -(sn * y[u].x)); tp[u].y = fma(cs, tp[u].y, -(sn * y[u].y));
              y[u].x = fma(tt, tp[u].x, y[u].x * ics); y[u].y = fma(tt, tp[u].y, y[u].y * ics);
            }
            const double tg = tt * ga;
            double aln = al - tg, ben = be + tg;
            const bool bad = dorot && (aln < 0.01 * al || ben < 0.01 * be);
            if (__any_sync(0xffffffffu, bad)) {               // heavy cancellation (rare): fresh norms
              double a0 = 0.0, b0 = 0.0, z0 = 0.0;
#pragma unroll
              for (int u = 0; u < NREG; u++) {
                a0 = fma(tp[u].x, tp[u].x, a0); a0 = fma(tp[u].y, tp[u].y, a0);
                b0 = fma(y[u].x, y[u].x, b0); b0 = fma(y[u].y, y[u].y, b0);
              }
              half_sum3(a0, b0, z0);
              if (bad) { aln = a0; ben = b0; }
            }
            if (dorot) {
              big |= (ga * ga > early2 * al * be);
              al = aln; be = ben;
              if (!last) {
#pragma unroll
                for (int u = 0; u < NREG; u++) cq[l16 + 16 * u] = y[u];
                if (l16 == 0) nrmc[bs + j] = ben;
              }
            }
          }
          if (last && own) {
            // exchange fused into the last round: bottom column j and top column pi go to the spare
            // buffers of their next owners
            double* const rcol_top = cluster.map_shared_rank(colbuf, top_dst_rank);
            double* const rcol_bot = cluster.map_shared_rank(colbuf, bot_dst_rank);
            double2* dq = reinterpret_cast<double2*>(rcol_bot + (size_t)nxt * per + ((size_t)bot_dst_slot * bs + j) * LEN);
            double2* dp = reinterpret_cast<double2*>(rcol_top + (size_t)nxt * per + ((size_t)top_dst_slot * bs + pi) * LEN);
#pragma unroll
            for (int u = 0; u < NREG; u++) { dq[l16 + 16 * u] = y[u]; dp[l16 + 16 * u] = tp[u]; }
            if (l16 == 0) {
              double* const rnrm_top = cluster.map_shared_rank(nrmbuf, top_dst_rank);
              double* const rnrm_bot = cluster.map_shared_rank(nrmbuf, bot_dst_rank);
              int* const rid_top = cluster.map_shared_rank(idbuf, top_dst_rank);
              int* const rid_bot = cluster.map_shared_rank(idbuf, bot_dst_rank);
              rnrm_bot[nxt * 2 * bs + bot_dst_slot * bs + j] = be;
              rnrm_top[nxt * 2 * bs + top_dst_slot * bs + pi] = al;
              rid_bot[nxt * 2 * bs + bot_dst_slot * bs + j] = ids[bs + j];
              rid_top[nxt * 2 * bs + top_dst_slot * bs + pi] = ids[pi];
            }
          }
          if (!last) named_bar_sync(1, nrt);
        }
      }
      if (sr == 2 * CS - 2) {
        // last barrier of the sweep carries the largest rotated cos^2 of every CTA
        if (big) s_flag = 1;
        __syncthreads();
        if (tid < CS) cluster.map_shared_rank(flags, tid)[crank] = s_flag ? 1.0 : 0.0;
      }
      cluster.sync();
      cur = nxt;
      cols = colbuf + (size_t)cur * per;
      ids = idbuf + cur * 2 * bs;
    }
    sweeps = sw + 1;
    // Was any pair with |cos| > max(tol, early) rotated in this sweep, cluster-wide?  If not the
    // iteration has converged: either nothing was rotated, or only pairs with tiny cosines were,
    // and the cyclic Jacobi iteration converges quadratically (a sweep whose largest cosine is c
    // leaves cosines of order c^2), so the sweep that would only confirm |cos| <= tol is not run
    // (option "jacobi_early" = cosine threshold, default 1e-7; 0 = always run the confirming sweep).
    double anybig = 0.0;
    for (int c = 0; c < CS; c++) anybig += flags[c];
    if (tid == 0) s_flag = 0;                         // every thread passed the flag push (cluster barrier)
    __syncthreads();
    if (anybig == 0.0) break;
    // ---- deflation of the discarded tail (truncation-aware; eq. (11): only chi_max triplets
    // survive).  After `nfull` sweeps the columns whose norm is below theta x the norm of the keep_hint-th
    // largest column can no longer matter for the leading keep_hint triplets: rotating a column p of norm
    // alpha against one of norm beta <= theta alpha changes p by an angle <= (beta / alpha) cos(p, q) and
    // its norm by the square of that.  They are written out as they are (their norms stand in for their
    // singular values, which lie below the cut) and the iteration goes on with the remaining columns,
    // re-dealt over the cluster: a sweep of n' columns is n' - 1 rounds instead of Nc - 1.
    if (keep_hint > 0 && sw + 1 == nfull && bl == bs && Nc > 2 * keep_hint) {
      double* G = b.G[t];
      double* svu = b.V[t] + (size_t)Nc * Nc;
      for (int ci = warp; ci < 2 * bs; ci += nw) {
        const int id = ids[ci];
        if (id >= Nc) continue;
        const double* col = cols + (size_t)ci * LEN;
        double s2 = 0.0;
        for (int kk = lane; kk < Mj; kk += 32) { double x = col[kk]; s2 += x * x; G[(size_t)id * M + kk] = x; }
        s2 = warp_sum1(s2);
        if (lane == 0) svu[id] = sqrt(s2);
      }
      __threadfence();
      cluster.sync();
      int* kl = reinterpret_cast<int*>(vbuf);             // kl[rank] = column id (>= 2 (MP + 2) ints available)
      __shared__ int s_np;
      if (tid == 0) s_np = 0;
      for (int j = tid; j < Nc; j += NTHR) {
        const double sj = svu[j];
        int rank = 0;
        for (int l = 0; l < Nc; l++) { const double sl = svu[l]; rank += (sl > sj || (sl == sj && l < j)) ? 1 : 0; }
        kl[rank] = j;
      }
      __syncthreads();
      const double scut = svu[kl[keep_hint - 1]];
      for (int r = tid; r < Nc; r += NTHR) if (svu[kl[r]] >= theta * scut) atomicAdd(&s_np, 1);
      __syncthreads();
      const int np = s_np;
      const int bl2 = (np + 2 * CS - 1) / (2 * CS);
      if (bl2 < bl && np >= keep_hint) {                  // the same decision in every CTA (same data)
        const int np2 = min(Nc, 2 * CS * bl2);
        for (int e = tid; e < per; e += NTHR) {
          const int kk = e % LEN, ci = e / LEN, slot = ci / bs, i = ci % bs;
          int id = Nc;
          if (i < bl2) { const int rank = (slot ? 2 * CS - 1 - crank : crank) * bl2 + i; if (rank < np2) id = kl[rank]; }
          cols[e] = (id < Nc && kk < Mj) ? G[(size_t)id * M + kk] : 0.0;
        }
        for (int e = tid; e < 2 * bs; e += NTHR) {
          const int slot = e / bs, i = e % bs;
          int id = Nc;
          if (i < bl2) { const int rank = (slot ? 2 * CS - 1 - crank : crank) * bl2 + i; if (rank < np2) id = kl[rank]; }
          ids[e] = id;
          idbuf[(cur ^ 1) * 2 * bs + e] = Nc;             // stale ids of the other buffer's dead slots
        }
        bl = bl2; nb2 = (bl & 1) ? bl + 1 : bl; nrw = (bl + 1) / 2; nrt = nrw * 32;
      }
      __syncthreads();
      cluster.sync();
    }
  }
  // ---- write back ------------------------------------------------------------------------------
  double* G = b.G[t];
  double* svu = b.V[t] + (size_t)Nc * Nc;
  for (int ci = warp; ci < 2 * bs; ci += nw) {
    const int id = ids[ci];
    if (id >= Nc) continue;
    const double* col = cols + (size_t)ci * LEN;
    double s = 0.0;
    for (int k = lane; k < Mj; k += 32) { double x = col[k]; s += x * x; G[(size_t)id * M + k] = x; }
    s = warp_sum1(s);
    if (lane == 0) svu[id] = sqrt(s);
  }
  __threadfence();
  cluster.sync();
  if (crank == 0) {
    for (int j = tid; j < Nc; j += NTHR) {
      const double sj = svu[j];
      int rank = 0;
      for (int l = 0; l < Nc; l++) {
        const double sl = svu[l];
        rank += (sl > sj || (sl == sj && l < j)) ? 1 : 0;
      }
      b.order[t][rank] = j;
      b.sv[t][rank] = sj;
    }
    if (tid == 0 && b.sweeps[t]) *b.sweeps[t] = sweeps;
  }
}

__global__ void svd_truncate_kernel(SvdFinishBatch b, int chi_max, double eps_cut) {
  const int t = blockIdx.x;
  if (threadIdx.x != 0) return;
  const int Nc = min(b.r1[t], b.r2[t]);
  const double* s = b.sv[t];
  const double s0 = (Nc > 0) ? s[0] : 0.0;
  int chin = 0;
  double tot = 0.0, kept = 0.0, gap = 1.0;
  if (s0 > 0.0 && isfinite(s0)) {
    int count = 0;
    for (int i = 0; i < Nc; i++) {
      tot += s[i] * s[i];
      if (s[i] >= eps_cut * s0) count++;
    }
    chin = min(count, chi_max);
    for (int i = 0; i < chin; i++) kept += s[i] * s[i];
    const double nrm = sqrt(kept);
    for (int i = 0; i < chin; i++) {
      double l = s[i] / nrm;
      b.lambda[t][i] = l;
      double sq = sqrt(l);
      b.sqrt_l[t][i] = sq;
      b.isqrt_l[t][i] = 1.0 / sq;
    }
    if (count > chi_max && chin < Nc) gap = (s[chin - 1] - s[chin]) / s[chin - 1];
    double disc = 0.0;
    for (int i = chin; i < Nc; i++) disc += s[i] * s[i];
    b.gate_stats[t][0] = disc / tot;
    b.gate_stats[t][1] = gap;
  } else {
    b.gate_stats[t][0] = 0.0;
    b.gate_stats[t][1] = 1.0;
  }
  *b.chi_new[t] = chin;
}

// Us = U sqrt(S), Vs = V sqrt(S) restricted to the kept chi_new triplets
__global__ void svd_bridge_kernel(SvdFinishBatch b) {
  const int t = blockIdx.y;
  const int r1 = b.r1[t], r2 = b.r2[t];
  const bool tr = r1 < r2;
  const int M = tr ? r2 : r1, Nc = tr ? r1 : r2;
  const int chin = *b.chi_new[t];
  const double* G = b.G[t];
  const double* V = b.V[t];
  const long long tot = (long long)(r1 + r2) * chin;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < tot;
       e += (long long)gridDim.x * blockDim.x) {
    int row = (int)(e % (r1 + r2)), c = (int)(e / (r1 + r2));
    int j = b.order[t][c];
    double rs = sqrt(b.sv[t][c]);
    // G columns are (left vectors of the tall problem) * s ; V columns the right vectors
    if (row < r1) {
      double v = tr ? V[row + (long long)j * Nc] * rs : G[row + (long long)j * M] / rs;
      b.Us[t][row + (long long)c * b.ldus[t]] = v;
    } else {
      int rr = row - r1;
      double v = tr ? G[rr + (long long)j * M] / rs : V[rr + (long long)j * Nc] * rs;
      b.Vs[t][rr + (long long)c * b.ldvs[t]] = v;
    }
  }
}

// Bridges without an accumulated V (hot path): the Jacobi kernel leaves G = A V = (left vectors
// of A) * s for the tall problem A (= K, or K^T when r1 < r2).  The other side follows from
// b_j = A^T a_j / s_j, i.e. Z = A^T G[:, kept] computed here from the untouched core K.
//   !tr: Us = G/sqrt(s),   Vs = (K^T G)/s^1.5        tr: Vs = G/sqrt(s),   Us = (K G)/s^1.5
// Error of b_j is u ||K|| / s_j, so s_j b_j (what enters the tensors) is accurate to u ||K||.
__global__ void __launch_bounds__(256) svd_bridge_nov_kernel(SvdFinishBatch b) {
  const int t = blockIdx.y;
  const int r1 = b.r1[t], r2 = b.r2[t];
  // a square core may have been iterated as K^T (launch_svd_jacobi `orient`)
  const bool tr = r1 < r2 || (r1 == r2 && b.orient[t] != nullptr && *b.orient[t] != 0);
  const int M = tr ? r2 : r1, Nc = tr ? r1 : r2;
  const bool precond = b.precond_min > 0 && Nc >= b.precond_min;
  // columns of G (ld M): left vectors of the tall problem A (= K, or K^T if tr) times s; with the
  // QR preconditioner instead its right vectors times s (length Nc).  Either way they are
  // singular vectors of K on one side, and the other side is op(K) G / s.
  const bool g_is_v = (tr != precond);                 // G holds right vectors of K
  const int gr = g_is_v ? r2 : r1, zr = g_is_v ? r1 : r2;
  const int chin = *b.chi_new[t];
  const double* G = b.G[t];
  const double* K = b.K[t];
  const int ldk = b.ldk[t];
  const int* order = b.order[t];
  const double* sv = b.sv[t];
  double* Gside = g_is_v ? b.Vs[t] : b.Us[t];
  const int ldg = g_is_v ? b.ldvs[t] : b.ldus[t];
  double* Zside = g_is_v ? b.Us[t] : b.Vs[t];
  const int ldz = g_is_v ? b.ldus[t] : b.ldvs[t];
  const long long gtid = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  const long long gthreads = (long long)gridDim.x * blockDim.x;
  for (long long e = gtid; e < (long long)gr * chin; e += gthreads) {
    int row = (int)(e % gr), c = (int)(e / gr);
    Gside[row + (long long)c * ldg] = G[row + (long long)order[c] * M] / sqrt(sv[c]);
  }
  if (!g_is_v) {
    // Z = K^T G: Z[i,c] = sum_{k<r1} K[k + i ldk] G[k + j M]: one warp per output, lanes along k
    const int lane = threadIdx.x & 31;
    const long long gw = gtid >> 5, nwarps = gthreads >> 5;
    for (long long e = gw; e < (long long)zr * chin; e += nwarps) {
      int i = (int)(e % zr), c = (int)(e / zr);
      const double* kc = K + (long long)i * ldk;
      const double* gc = G + (long long)order[c] * M;
      double z = 0.0;
      for (int k = lane; k < gr; k += 32) z += kc[k] * gc[k];
      z = warp_sum(z);
      if (lane == 0) { double sc = sv[c]; Zside[i + (long long)c * ldz] = z / (sc * sqrt(sc)); }
    }
  } else {
    // Z = K G: Z[i,c] = sum_{k<r2} K[i + k ldk] G[k + j M]: one thread per output, coalesced along i
    for (long long e = gtid; e < (long long)zr * chin; e += gthreads) {
      int i = (int)(e % zr), c = (int)(e / zr);
      const double* gc = G + (long long)order[c] * M;
      double z = 0.0;
      for (int k = 0; k < gr; k++) z += K[i + (long long)k * ldk] * gc[k];
      double sc = sv[c];
      Zside[i + (long long)c * ldz] = z / (sc * sqrt(sc));
    }
  }
}

__global__ void svd_vectors_kernel(const double* G, const double* V, const double* s,
                                   const int* order, int m, int n, double* U, double* Vout) {
  const bool tr = m < n;
  const int M = tr ? n : m, Nc = tr ? m : n;
  const long long tot = (long long)(m + n) * Nc;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < tot;
       e += (long long)gridDim.x * blockDim.x) {
    int row = (int)(e % (m + n)), c = (int)(e / (m + n));
    int j = order[c];
    double sv = s[c];
    double inv = sv > 0.0 ? 1.0 / sv : 0.0;
    if (row < m) U[row + (long long)c * m] = tr ? V[row + (long long)j * Nc] : G[row + (long long)j * M] * inv;
    else { int rr = row - m; Vout[rr + (long long)c * n] = tr ? G[rr + (long long)j * M] * inv : V[rr + (long long)j * Nc]; }
  }
}

__global__ void set_identity_kernel(double* Q, long long m, int k) {
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < m * k;
       e += (long long)gridDim.x * blockDim.x) {
    long long i = e % m; int j = (int)(e / m);
    Q[e] = (i == j) ? 1.0 : 0.0;
  }
}

}  // namespace


int launch_svd_vectors(cudaStream_t st, const double* G, const double* V, const double* s,
                       const int* order, int m, int n, double* U, double* Vout) {
  long long w = (long long)(m + n) * std::min(m, n);
  long long g = std::min<long long>(std::max<long long>((w + 255) / 256, 1), 148 * 4);
  svd_vectors_kernel<<<(unsigned)g, 256, 0, st>>>(G, V, s, order, m, n, U, Vout);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

int launch_set_identity(cudaStream_t st, double* Q, long long m, int k) {
  long long w = m * k;
  long long g = std::min<long long>(std::max<long long>((w + 255) / 256, 1), 148 * 8);
  set_identity_kernel<<<(unsigned)g, 256, 0, st>>>(Q, m, k);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

static int launch_svd_group(cudaStream_t st, const SvdBatch& b, double tol, int max_sweeps, bool with_v,
                            int precond_min, double early, int keep_hint, double theta, int orient);

// The launch configuration (cluster size, columns per CTA, register tile) fixes the order of the
// pair rotations, i.e. the rounding of the result.  It is therefore chosen per problem SIZE, never
// from the composition of the batch: problems of equal (min, max) dimension share a launch, and a
// gate gives bit-identical results whichever other gates run beside it (serial or pipelined class).
int launch_svd_jacobi(cudaStream_t st, const SvdBatch& b, double tol, int max_sweeps, bool with_v,
                      int precond_min, double early, int keep_hint, double theta, int orient) {
  if (b.count == 0) return 0;
  bool done[PEPO_MAXT] = {false};
  for (int t0 = 0; t0 < b.count; t0++) {
    if (done[t0]) continue;
    const int nc0 = std::min(b.r1[t0], b.r2[t0]), mm0 = std::max(b.r1[t0], b.r2[t0]);
    SvdBatch g; g.count = 0;
    for (int t = t0; t < b.count; t++) {
      if (done[t] || std::min(b.r1[t], b.r2[t]) != nc0 || std::max(b.r1[t], b.r2[t]) != mm0) continue;
      const int q = g.count++;
      g.K[q] = b.K[t]; g.ldk[q] = b.ldk[t]; g.r1[q] = b.r1[t]; g.r2[q] = b.r2[t];
      g.G[q] = b.G[t]; g.V[q] = b.V[t]; g.sv[q] = b.sv[t]; g.order[q] = b.order[t]; g.sweeps[q] = b.sweeps[t];
      g.orient[q] = b.orient[t];
      done[t] = true;
    }
    int rc = launch_svd_group(st, g, tol, max_sweeps, with_v, precond_min, early, keep_hint, theta, orient);
    if (rc) return rc;
  }
  return 0;
}

static int launch_svd_group(cudaStream_t st, const SvdBatch& b, double tol, int max_sweeps, bool with_v,
                            int precond_min, double early, int keep_hint, double theta, int orient) {
  if (b.count == 0) return 0;
  int ncmax = 1, lenmax = 2;
  for (int t = 0; t < b.count; t++) {
    int nc = std::min(b.r1[t], b.r2[t]), mm = std::max(b.r1[t], b.r2[t]);
    ncmax = std::max(ncmax, nc); lenmax = std::max(lenmax, ((mm + 1) & ~1) + (with_v ? ((nc + 1) & ~1) : 0));
  }
  // smallest cluster whose per-CTA share of the columns fits shared memory and the staging regs
  if (((lenmax >> 1) & 1) == 0) lenmax += 2;          // LEN/2 odd: columns start in distinct 16-byte bank groups
  // a CTA keeps at most ~16 column pairs busy per round (the pair rotations are LSU / issue bound
  // beyond that, measured), so prefer the cluster size with bs <= 16, up to the portable 8
  int cs0 = 1;
  while (cs0 < 8 && (ncmax + 2 * cs0 - 1) / (2 * cs0) > 16) cs0 *= 2;
  // hot path: 16-lane kernel (no V, cluster >= 2, columns of <= 256 doubles, <= 16 pairs per CTA)
  if (!with_v) {
    const int CS = std::max(cs0, 2);
    const int bs = (ncmax + 2 * CS - 1) / (2 * CS);
    int mmax = 2;
    for (int t = 0; t < b.count; t++) mmax = std::max(mmax, std::max(b.r1[t], b.r2[t]));
    int nreg = (mmax + 31) / 32 <= 2 ? 2 : (mmax + 31) / 32 <= 4 ? 4 : (mmax + 31) / 32 <= 6 ? 6 : 8;
    int CSx = CS, bsx = bs, nthr = J16_THREADS;
    if (mmax > 256 && mmax <= 416) {
      // chi in 65..104: cluster of 16 (non-portable size), <= 13 pairs per CTA, columns of <= 416
      // doubles in registers of a 256-thread CTA; the two column buffers fill shared memory
      CSx = 16; bsx = (ncmax + 31) / 32; nthr = 256;
      nreg = (mmax + 31) / 32 <= 10 ? 10 : 13;
    }
    if (CSx <= 16 && bsx <= 16 && mmax <= 416 && (mmax <= 256 || bsx <= 13)) {
      const int CS = CSx, bs = bsx;
      const int LENc = 32 * nreg;
      const size_t cap = (nthr == 256) ? (size_t)225 * 1024 : JC_SMEM_CAP;
      const size_t base = ((size_t)4 * bs * LENc + 4 * bs) * 8 + (size_t)((4 * bs + 3) & ~3) * 4 + (16 + 4) * 8;
      const size_t vs8 = (size_t)(((mmax + 1) & ~1) + 2) * 8;
      int pw = 1;
      if (precond_min > 0 && cap > base + vs8) pw = (int)std::max<size_t>(1, std::min<size_t>((size_t)bs, (cap - base) / vs8));
      const size_t smem = base + (size_t)pw * vs8;
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3((unsigned)(b.count * CS));
      cfg.blockDim = dim3(nthr);
      cfg.dynamicSmemBytes = smem;
      cfg.stream = st;
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeClusterDimension;
      at[0].val.clusterDim.x = CS; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
      cfg.attrs = at; cfg.numAttrs = 1;
      static char attr_done[PEPO_MAX_DEVICES] = {0};
      if (first_use_on_device(attr_done)) {
        const int mx = 226 * 1024;                 // 227 KB per CTA less the static shared memory
        PEPO_CUDA_OK(cudaFuncSetAttribute(jacobi_c16_kernel<2, 512>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx));
        PEPO_CUDA_OK(cudaFuncSetAttribute(jacobi_c16_kernel<4, 512>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx));
        PEPO_CUDA_OK(cudaFuncSetAttribute(jacobi_c16_kernel<6, 512>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx));
        PEPO_CUDA_OK(cudaFuncSetAttribute(jacobi_c16_kernel<8, 512>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx));
        PEPO_CUDA_OK(cudaFuncSetAttribute(jacobi_c16_kernel<10, 256>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx));
        PEPO_CUDA_OK(cudaFuncSetAttribute(jacobi_c16_kernel<13, 256>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx));
        PEPO_CUDA_OK(cudaFuncSetAttribute(jacobi_c16_kernel<2, 512>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
        PEPO_CUDA_OK(cudaFuncSetAttribute(jacobi_c16_kernel<4, 512>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
        PEPO_CUDA_OK(cudaFuncSetAttribute(jacobi_c16_kernel<6, 512>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
        PEPO_CUDA_OK(cudaFuncSetAttribute(jacobi_c16_kernel<8, 512>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
        PEPO_CUDA_OK(cudaFuncSetAttribute(jacobi_c16_kernel<10, 256>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
        PEPO_CUDA_OK(cudaFuncSetAttribute(jacobi_c16_kernel<13, 256>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
      }
      const double early2 = early * early;
      const int kh = (theta > 0.0) ? keep_hint : 0;
      cudaError_t e;
      if (nreg == 2) e = cudaLaunchKernelEx(&cfg, jacobi_c16_kernel<2, 512>, b, tol, max_sweeps, bs, CS, precond_min, pw, early2, kh, 3, theta, orient);
      else if (nreg == 4) e = cudaLaunchKernelEx(&cfg, jacobi_c16_kernel<4, 512>, b, tol, max_sweeps, bs, CS, precond_min, pw, early2, kh, 3, theta, orient);
      else if (nreg == 6) e = cudaLaunchKernelEx(&cfg, jacobi_c16_kernel<6, 512>, b, tol, max_sweeps, bs, CS, precond_min, pw, early2, kh, 3, theta, orient);
      else if (nreg == 8) e = cudaLaunchKernelEx(&cfg, jacobi_c16_kernel<8, 512>, b, tol, max_sweeps, bs, CS, precond_min, pw, early2, kh, 3, theta, orient);
      else if (nreg == 10) e = cudaLaunchKernelEx(&cfg, jacobi_c16_kernel<10, 256>, b, tol, max_sweeps, bs, CS, precond_min, pw, early2, kh, 3, theta, orient);
      else e = cudaLaunchKernelEx(&cfg, jacobi_c16_kernel<13, 256>, b, tol, max_sweeps, bs, CS, precond_min, pw, early2, kh, 3, theta, orient);
      if (e != cudaSuccess) { set_error("svd: cluster launch failed: %s", cudaGetErrorString(e)); return -3; }
      PEPO_COUNT_LAUNCH();
      return 0;
    }
  }
  for (int CS = cs0; CS <= 16; CS *= 2) {
    int bs = (ncmax + 2 * CS - 1) / (2 * CS);
    const int PW = (2 * bs + 3) & ~3;
    size_t smem0 = ((size_t)2 * bs * lenmax) * 8 + (size_t)(2 * bs + 4) * 4 + 64 +
                   ((size_t)4 * bs * PW + 4 * bs) * 8;
    int pw = 0;                                        // Householder panel width (preconditioner)
    if (!with_v && precond_min > 0 && smem0 < JC_SMEM_CAP)
      pw = (int)std::min<size_t>((size_t)bs, (JC_SMEM_CAP - smem0) / ((size_t)(lenmax + 2) * 8));
    size_t smem = smem0 + (size_t)std::max(pw, 1) * (lenmax + 2) * 8;
    bool fits = smem <= JC_SMEM_CAP && (CS == 1 || (size_t)2 * bs * lenmax <= (size_t)JC_STAGE * JC_THREADS);
    if (!fits) continue;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(b.count * CS));
    cfg.blockDim = dim3(JC_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = CS; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    // registers staged per thread during a block exchange: smallest instantiation that holds a CTA's columns
    const size_t need = (CS == 1) ? 0 : ((size_t)2 * bs * lenmax + JC_THREADS - 1) / JC_THREADS;
    const int pmin = (with_v || pw < 1) ? 0 : precond_min;
    const int pwk = std::max(pw, 1), wv = with_v ? 1 : 0;
    cudaError_t e;
    if (need <= 8 && lenmax / 2 <= 128 && bs <= JC_THREADS / 32) {
      static char done84[PEPO_MAX_DEVICES] = {0};
      if (first_use_on_device(done84)) {
        PEPO_CUDA_OK(cudaFuncSetAttribute(jacobi_cluster_kernel<8, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)JC_SMEM_CAP + 1024));
        PEPO_CUDA_OK(cudaFuncSetAttribute(jacobi_cluster_kernel<8, 4>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
      }
      e = cudaLaunchKernelEx(&cfg, jacobi_cluster_kernel<8, 4>, b, tol, max_sweeps, bs, CS, wv, lenmax, pmin, pwk);
    } else if (need <= 8) {
      static char done8[PEPO_MAX_DEVICES] = {0};
      if (first_use_on_device(done8)) {
        PEPO_CUDA_OK(cudaFuncSetAttribute(jacobi_cluster_kernel<8, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)JC_SMEM_CAP + 1024));
        PEPO_CUDA_OK(cudaFuncSetAttribute(jacobi_cluster_kernel<8, 0>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
      }
      e = cudaLaunchKernelEx(&cfg, jacobi_cluster_kernel<8, 0>, b, tol, max_sweeps, bs, CS, wv, lenmax, pmin, pwk);
    } else if (need <= 16) {
      static char done16[PEPO_MAX_DEVICES] = {0};
      if (first_use_on_device(done16)) {
        PEPO_CUDA_OK(cudaFuncSetAttribute(jacobi_cluster_kernel<16, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)JC_SMEM_CAP + 1024));
        PEPO_CUDA_OK(cudaFuncSetAttribute(jacobi_cluster_kernel<16, 0>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
      }
      e = cudaLaunchKernelEx(&cfg, jacobi_cluster_kernel<16, 0>, b, tol, max_sweeps, bs, CS, wv, lenmax, pmin, pwk);
    } else {
      static char done26[PEPO_MAX_DEVICES] = {0};
      if (first_use_on_device(done26)) {
        PEPO_CUDA_OK(cudaFuncSetAttribute(jacobi_cluster_kernel<JC_STAGE, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)JC_SMEM_CAP + 1024));
        PEPO_CUDA_OK(cudaFuncSetAttribute(jacobi_cluster_kernel<JC_STAGE, 0>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
      }
      e = cudaLaunchKernelEx(&cfg, jacobi_cluster_kernel<JC_STAGE, 0>, b, tol, max_sweeps, bs, CS, wv, lenmax, pmin, pwk);
    }
    if (e == cudaSuccess) { PEPO_COUNT_LAUNCH(); return 0; }
    (void)cudaGetLastError();                      // e.g. cluster of 16 not schedulable: try the fallback
    break;
  }
  if (!with_v && precond_min > 0) { set_error("svd: cluster launch failed"); return -3; }
  size_t smem = (size_t)ncmax * sizeof(double);
  jacobi_svd_kernel<<<b.count, 1024, smem, st>>>(b, tol, max_sweeps);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

int launch_svd_truncate(cudaStream_t st, const SvdFinishBatch& b, int chi_max, double eps_cut) {
  if (b.count == 0) return 0;
  svd_truncate_kernel<<<b.count, 32, 0, st>>>(b, chi_max, eps_cut);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

int launch_svd_bridge(cudaStream_t st, const SvdFinishBatch& b, int chi_cap) {
  if (b.count == 0) return 0;
  long long w = 0;
  for (int t = 0; t < b.count; t++) w = std::max(w, (long long)(b.r1[t] + b.r2[t]) * chi_cap);
  long long g = std::min<long long>(std::max<long long>((w + 255) / 256, 1), 148 * 4);
  dim3 grid((unsigned)g, b.count);
  if (b.with_v) svd_bridge_kernel<<<grid, 256, 0, st>>>(b);
  else svd_bridge_nov_kernel<<<dim3(148 * 4, b.count), 256, 0, st>>>(b);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

}  // namespace pepo
