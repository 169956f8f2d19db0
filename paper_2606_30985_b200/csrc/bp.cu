// bp.cu - belief-propagation message sweep (a14: eq. (13), (14), (19) PAPER.md:L243-L256,
// L444-L449; readings R6, R7), the single-site field gate (a1, L313, L339) and the log-space,
// sign-tracked Bethe evaluation (a15: eq. (7)-(9), L112-L128).
//
// A sweep reads the pinned slab T_v = psi_v[..., p_v] of every site ONCE and produces all of
// the site's outgoing messages from that single pass (the paper issues one strided-batched
// GEMV per message, L247): block (l, r) of site v reduces the dU x dD slice
//     pU[u] = sum_d T[u,d,l,r] mD[d],  pD[d] = sum_u T[u,d,l,r] mU[u],  s = sum_u mU[u] pU[u]
// and stores w*pU, w*pD (w = mL[l] mR[r]) and s as partials; `bp_finalize_kernel` sums the
// partials in a fixed order (deterministic, no floating-point atomics), L2-normalises,
// sign-aligns, damps and takes delta = max |m_new - m_old| (atomicMax on the bit pattern of a
// non-negative double is order-independent).
#include "bp.cuh"
#include <algorithm>

namespace pepo {
namespace {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

constexpr int BP_THREADS = 256;
constexpr int BP_MAXK = 8;     // dU <= 256 (kernel instantiated for 32*KU >= dU, KU in {2,4,8}: fewer
                               // registers -> more resident CTAs -> more bytes in flight)

template <int KU>
__global__ void __launch_bounds__(BP_THREADS) bp_partial_kernel(BpBatch b) {
  if (b.skip_if && __longlong_as_double((long long)*b.skip_if) < b.skip_tol) return;
  constexpr int nw = BP_THREADS / 32;
  __shared__ double sU[nw][32 * KU];
  __shared__ double sS[PEPO_BP_MAXCHUNK][nw];
  const int t = blockIdx.y;
  const BpSite& S = b.s[t];
  const int blk = blockIdx.x;
  if (blk >= S.nchunks) return;
  const int dU = S.d[0], dD = S.d[1], dL = S.d[2], dR = S.d[3];
  const int nlr = dL * dR;
  const int lr0 = blk * S.chunk, lr1 = min(nlr, lr0 + S.chunk);
  const double* mU = S.in[0];
  const double* mD = S.in[1];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double accU[KU];
  double mu[KU];
#pragma unroll
  for (int k = 0; k < KU; k++) {
    accU[k] = 0.0;
    int u = lane + 32 * k;
    mu[k] = (u < dU) ? mU[u] : 0.0;
  }
  // lane j of warp wp owns pD[d] for d = wp + nw*j (dD <= 256)
  double accD = 0.0;
  const double myD = (warp + nw * lane < dD) ? mD[warp + nw * lane] : 0.0;
  for (int lr = lr0; lr < lr1; lr++) {
    const int l = lr % dL, r = lr / dL;
    const double w = S.in[2][l] * S.in[3][r];
    const double* T = S.T + (long long)lr * dU * dD;
    double ssum = 0.0;
    int j = 0;
    for (int d = warp; d < dD; d += 2 * nw, j += 2) {
      const int d2 = d + nw;
      const bool has2 = d2 < dD;
      const double md = __shfl_sync(0xffffffffu, myD, j);
      const double md2 = __shfl_sync(0xffffffffu, myD, (j + 1) & 31);
      const double* col = T + (long long)d * dU;
      const double* col2 = T + (long long)(has2 ? d2 : d) * dU;
      const double mdw = md * w, mdw2 = has2 ? md2 * w : 0.0;
      double cs = 0.0, cs2 = 0.0;
#pragma unroll
      for (int k = 0; k < KU; k++) {
        int u = lane + 32 * k;
        if (u < dU) {
          double tv = col[u], tv2 = col2[u];
          accU[k] += tv * mdw;
          cs += tv * mu[k];
          accU[k] += tv2 * mdw2;
          cs2 += tv2 * mu[k];
        }
      }
      cs = warp_sum(cs);
      cs2 = warp_sum(cs2);
      if (lane == j) accD += w * cs;
      ssum += md * cs;
      if (has2) {
        if (lane == j + 1) accD += w * cs2;
        ssum += md2 * cs2;
      }
    }
    if (lane == 0) sS[lr - lr0][warp] = ssum;
  }
#pragma unroll
  for (int k = 0; k < KU; k++) sU[warp][lane + 32 * k] = accU[k];
  __syncthreads();
  for (int u = threadIdx.x; u < dU; u += BP_THREADS) {
    double p = 0.0;
#pragma unroll
    for (int w2 = 0; w2 < nw; w2++) p += sU[w2][u];
    S.partU[(long long)blk * dU + u] = p;
  }
  {
    const int d = warp + nw * lane;
    if (d < dD) S.partD[(long long)blk * dD + d] = accD;
  }
  // s(l,r) = sum_d mD[d] (sum_u T[u,d,l,r] mU[u])
  for (int i = threadIdx.x; i < lr1 - lr0; i += BP_THREADS) {
    double sv = 0.0;
#pragma unroll
    for (int w2 = 0; w2 < nw; w2++) sv += sS[i][w2];
    S.partS[lr0 + i] = sv;
  }
}

// Second form of the partial sweep (the one launched): the reduction over u that pD[d] needs is
// NOT taken per column.  Warp w owns the columns d = w + nw j (j < KD) of every slice of its
// chunk; each lane accumulates its own share of pD[d] in a register across all slices of the
// chunk (weight w_lr folded in), and the KD warp reductions happen once per chunk.  Per slice only
// s(l,r) needs one warp reduction.  Per column that leaves two loads and four FMAs per lane and no
// shuffle (the first form spent ~30 of its ~45 instructions per column pair on reductions and was
// issue-bound at 0.35 of the HBM rate); the KD columns of a slice are KU*KD independent loads in
// flight per lane.  Sums are in a fixed order: deterministic.
template <int KU, int KD>
__global__ void __launch_bounds__(BP_THREADS) bp_partial2_kernel(BpBatch b) {
  if (b.skip_if && __longlong_as_double((long long)*b.skip_if) < b.skip_tol) return;
  constexpr int nw = BP_THREADS / 32;
  __shared__ double sU[nw][32 * KU];
  __shared__ double sS[PEPO_BP_MAXCHUNK][nw];
  const int t = blockIdx.y;
  const BpSite& S = b.s[t];
  const int blk = blockIdx.x;
  if (blk >= S.nchunks) return;
  const int dU = S.d[0], dD = S.d[1], dL = S.d[2], dR = S.d[3];
  const int nlr = dL * dR;
  const int lr0 = blk * S.chunk, lr1 = min(nlr, lr0 + S.chunk);
  const double* mU = S.in[0];
  const double* mD = S.in[1];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double accU[KU], mu[KU], accD[KD], md[KD];
#pragma unroll
  for (int k = 0; k < KU; k++) {
    accU[k] = 0.0;
    const int u = lane + 32 * k;
    mu[k] = (u < dU) ? mU[u] : 0.0;
  }
#pragma unroll
  for (int j = 0; j < KD; j++) {
    accD[j] = 0.0;
    const int d = warp + nw * j;
    md[j] = (d < dD) ? mD[d] : 0.0;
  }
  for (int lr = lr0; lr < lr1; lr++) {
    const int l = lr % dL, r = lr / dL;
    const double w = S.in[2][l] * S.in[3][r];
    const double* T = S.T + (long long)lr * dU * dD;
    double ps[KU], wmu[KU];
#pragma unroll
    for (int k = 0; k < KU; k++) { ps[k] = 0.0; wmu[k] = w * mu[k]; }
    // all loads of the slice first (columns past dD are clamped to a valid one: their md is 0 and
    // their accD is never stored), then the arithmetic: KU*KD independent loads in flight per lane
    constexpr int JB = (KD * KU <= 16) ? KD : (16 / KU);     // columns per load batch (16 loads per lane)
#pragma unroll
    for (int j0 = 0; j0 < KD; j0 += JB) {
      double tv[JB][KU];
#pragma unroll
      for (int j = 0; j < JB; j++) {
        const int d = min(warp + nw * (j0 + j), dD - 1);
        const double* col = T + (long long)d * dU;
#pragma unroll
        for (int k = 0; k < KU; k++) {
          const int u = lane + 32 * k;
          tv[j][k] = (u < dU) ? __ldg(col + u) : 0.0;
        }
      }
#pragma unroll
      for (int j = 0; j < JB; j++) {
#pragma unroll
        for (int k = 0; k < KU; k++) {
          ps[k] = fma(tv[j][k], md[j0 + j], ps[k]);
          accD[j0 + j] = fma(tv[j][k], wmu[k], accD[j0 + j]);
        }
      }
    }
    double sp = 0.0;
#pragma unroll
    for (int k = 0; k < KU; k++) { accU[k] = fma(w, ps[k], accU[k]); sp = fma(mu[k], ps[k], sp); }
    sp = warp_sum(sp);
    if (lane == 0) sS[lr - lr0][warp] = sp;
  }
#pragma unroll
  for (int k = 0; k < KU; k++) sU[warp][lane + 32 * k] = accU[k];
#pragma unroll
  for (int j = 0; j < KD; j++) {
    const int d = warp + nw * j;
    const double v = warp_sum(accD[j]);
    if (lane == 0 && d < dD) S.partD[(long long)blk * dD + d] = v;
  }
  __syncthreads();
  for (int u = threadIdx.x; u < dU; u += BP_THREADS) {
    double p = 0.0;
#pragma unroll
    for (int w2 = 0; w2 < nw; w2++) p += sU[w2][u];
    S.partU[(long long)blk * dU + u] = p;
  }
  for (int i = threadIdx.x; i < lr1 - lr0; i += BP_THREADS) {
    double sv = 0.0;
#pragma unroll
    for (int w2 = 0; w2 < nw; w2++) sv += sS[i][w2];
    S.partS[lr0 + i] = sv;
  }
}

// one block per (site, leg slot)
__global__ void __launch_bounds__(256) bp_finalize_kernel(BpBatch b, double damping, int update,
                                                          unsigned long long* delta_bits,
                                                          int* flag) {
  if (b.skip_if && __longlong_as_double((long long)*b.skip_if) < b.skip_tol) return;
  __shared__ double sred[8];
  __shared__ double s_bcast[2];
  const int t = blockIdx.y;
  const int slot = blockIdx.x;
  const BpSite& S = b.s[t];
  if (!S.present[slot]) return;
  const int dU = S.d[0], dD = S.d[1], dL = S.d[2], dR = S.d[3];
  const int dl = S.d[slot];
  const int nlr = dL * dR;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  extern __shared__ double mhat[];      // dl doubles
  double nrm2 = 0.0, dot_old = 0.0, dot_in = 0.0;
  const double* old = S.out_old[slot];
  const double* inc = S.in[slot];
  // slots 0/1: sum of the per-chunk partial vectors, 4 thread groups per entry, fixed order
  __shared__ double sgrp[4][64];
  const bool split = (slot < 2) && dl <= 64;
  if (split) {
    const int i = threadIdx.x & 63, gq = threadIdx.x >> 6;
    const double* part = slot == 0 ? S.partU : S.partD;
    double v = 0.0;
    if (i < dl) for (int k = gq; k < S.nchunks; k += 4) v += part[(long long)k * dl + i];
    sgrp[gq][i] = v;
    __syncthreads();
  }
  for (int i = threadIdx.x; i < dl; i += blockDim.x) {
    double v = 0.0;
    if (split) {
      v = (sgrp[0][i] + sgrp[1][i]) + (sgrp[2][i] + sgrp[3][i]);
    } else if (slot == 0) {
      for (int k = 0; k < S.nchunks; k++) v += S.partU[(long long)k * dU + i];
    } else if (slot == 1) {
      for (int k = 0; k < S.nchunks; k++) v += S.partD[(long long)k * dD + i];
    } else if (slot == 2) {
      for (int r = 0; r < dR; r++) v += S.in[3][r] * S.partS[i + dL * r];
    } else {
      for (int l = 0; l < dL; l++) v += S.in[2][l] * S.partS[l + dL * i];
    }
    mhat[i] = v;
    nrm2 += v * v;
    dot_old += v * old[i];
    dot_in += v * inc[i];
  }
  // block reductions (fixed order)
  double vals[3] = {nrm2, dot_old, dot_in};
  double red[3];
  for (int q = 0; q < 3; q++) {
    double v = warp_sum(vals[q]);
    __syncthreads();
    if (lane == 0) sred[warp] = v;
    __syncthreads();
    double s = 0.0;
    for (int w = 0; w < 8; w++) s += sred[w];
    red[q] = s;
  }
  if (threadIdx.x == 0 && slot == S.first_slot) *S.vs = red[2];     // eq. (7): site value
  if (!update) return;
  const double nrm = sqrt(red[0]);
  double* outn = S.out_new[slot];
  if (!(nrm > 0.0) || !isfinite(nrm)) {
    // R7: a zero-norm update keeps the old message and is flagged (bit 0); a non-finite norm (bit 1)
    // also poisons delta with +inf so that the sweep can never count as converged
    for (int i = threadIdx.x; i < dl; i += blockDim.x) outn[i] = old[i];
    if (threadIdx.x == 0) {
      const bool bad = !isfinite(nrm);
      atomicOr(flag, bad ? 2 : 1);
      if (bad) atomicMax(delta_bits, 0x7ff0000000000000ull);
    }
    return;
  }
  const double sgn = (red[1] < 0.0) ? -1.0 : 1.0;
  double dmax = 0.0;
  for (int i = threadIdx.x; i < dl; i += blockDim.x) {
    double mh = sgn * (mhat[i] / nrm);
    double o = old[i];
    double mn = damping * o + (1.0 - damping) * mh;
    outn[i] = mn;
    const double ch = fabs(mn - o);
    dmax = (ch == ch) ? fmax(dmax, ch) : INFINITY;        // fmax would drop a NaN change
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) dmax = fmax(dmax, __shfl_xor_sync(0xffffffffu, dmax, o));
  if (lane == 0) atomicMax(delta_bits, (unsigned long long)__double_as_longlong(dmax));
  (void)0;
  (void)s_bcast;
}

// mode 0 (R7): m = (1, .., 1)/sqrt(chi); mode 1: m = e_0, the leading Schmidt vector of the bond
__global__ void bp_init_kernel(double* msgs, const int* chi_of_msg, int n_msgs, int chi_max, int mode) {
  const int mIdx = blockIdx.x;
  if (mIdx >= n_msgs) return;
  const int chi = chi_of_msg[mIdx];
  const double v = 1.0 / sqrt((double)chi);
  for (int i = threadIdx.x; i < chi_max; i += blockDim.x)
    msgs[(long long)mIdx * chi_max + i] = mode == 1 ? (i == 0 ? 1.0 : 0.0) : ((i < chi) ? v : 0.0);
}

// eq. (8), (9): C = prod vs_v / prod Z_e in log space with sign tracking
__global__ void __launch_bounds__(256) bethe_kernel(const double* vs, int n_sites,
                                                    const double* msgs, const int* chi_of_msg,
                                                    int n_bonds, int chi_max, double* out_C,
                                                    int* out_status) {
  extern __shared__ double Ze[];
  for (int e = threadIdx.x; e < n_bonds; e += blockDim.x) {
    const double* a = msgs + (long long)(2 * e) * chi_max;
    const double* c = msgs + (long long)(2 * e + 1) * chi_max;
    const int chi = chi_of_msg[2 * e];
    double s = 0.0;
    for (int i = 0; i < chi; i++) s += a[i] * c[i];
    Ze[e] = s;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double lognum = 0.0, logden = 0.0, sign = 1.0;
    int status = 0;
    bool zero = false;
    for (int v = 0; v < n_sites; v++) {
      double x = vs[v];
      if (!isfinite(x)) status = -4;
      if (x == 0.0) { zero = true; continue; }
      lognum += log(fabs(x));
      if (x < 0.0) sign = -sign;
    }
    for (int e = 0; e < n_bonds; e++) {
      double z = Ze[e];
      if (z == 0.0 || !isfinite(z)) { status = -4; continue; }
      logden += log(fabs(z));
      if (z < 0.0) sign = -sign;
    }
    *out_C = zero ? 0.0 : exp(lognum - logden) * sign;
    *out_status = status;
  }
}

// a1: psi[.., p'] = sum_p G1[p', p] psi[.., p] on the four contiguous Pauli slabs; rows of G1
// equal to the identity row are skipped (X field: only the Y and Z slabs move).
__global__ void __launch_bounds__(256) field_gate_kernel(FieldBatch b) {
  const int t = blockIdx.y;
  double* psi = b.psi[t];
  const long long slab = b.slab[t];
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < slab;
       i += (long long)gridDim.x * blockDim.x) {
    double v[4], o[4];
#pragma unroll
    for (int p = 0; p < 4; p++) v[p] = (b.col_mask >> p & 1) ? psi[i + p * slab] : 0.0;
#pragma unroll
    for (int q = 0; q < 4; q++) {
      if (b.row_mask >> q & 1) {
        o[q] = 0.0;
#pragma unroll
        for (int p = 0; p < 4; p++) o[q] += b.G[q * 4 + p] * v[p];
      }
    }
#pragma unroll
    for (int q = 0; q < 4; q++)
      if (b.row_mask >> q & 1) psi[i + q * slab] = o[q];
  }
}

}  // namespace

int launch_bp_partial(cudaStream_t st, const BpBatch& b) {
  if (b.count == 0) return 0;
  int maxlr = 1;
  for (int t = 0; t < b.count; t++) maxlr = std::max(maxlr, b.s[t].nchunks);
  dim3 grid(maxlr, b.count);
  int dumax = 1;
  for (int t = 0; t < b.count; t++) dumax = std::max(dumax, b.s[t].d[0]);
  int ddmax = 1;
  for (int t = 0; t < b.count; t++) ddmax = std::max(ddmax, b.s[t].d[1]);
  if (dumax <= 64 && ddmax <= 64) bp_partial2_kernel<2, 8><<<grid, BP_THREADS, 0, st>>>(b);
  else if (dumax <= 128 && ddmax <= 128) bp_partial2_kernel<4, 16><<<grid, BP_THREADS, 0, st>>>(b);
  else bp_partial_kernel<8><<<grid, BP_THREADS, 0, st>>>(b);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

int launch_bp_finalize(cudaStream_t st, const BpBatch& b, double damping, int update,
                       unsigned long long* delta_bits, int* flag) {
  if (b.count == 0) return 0;
  int dmax = 1;
  for (int t = 0; t < b.count; t++)
    for (int k = 0; k < 4; k++) dmax = std::max(dmax, b.s[t].d[k]);
  dim3 grid(4, b.count);
  bp_finalize_kernel<<<grid, 256, dmax * sizeof(double), st>>>(b, damping, update, delta_bits, flag);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

__global__ void __launch_bounds__(256) site_weights_partial_kernel(SiteWeightBatch b) {
  const int t = blockIdx.y, ch = blockIdx.x;
  const int d0 = b.d[t][0], d1 = b.d[t][1], d2 = b.d[t][2], d3 = b.d[t][3];
  const long long slab = (long long)d0 * d1 * d2 * d3;
  const long long per = (slab + PEPO_SW_CHUNKS - 1) / PEPO_SW_CHUNKS;
  const long long i0 = ch * per, i1 = min(slab, i0 + per);
  const double* psi = b.psi[t];
  double w[4] = {0.0, 0.0, 0.0, 0.0};
  for (long long i = i0 + threadIdx.x; i < i1; i += blockDim.x) {
    long long r = i;
    const int a0 = (int)(r % d0); r /= d0;
    const int a1 = (int)(r % d1); r /= d1;
    const int a2 = (int)(r % d2); r /= d2;
    const double lw = b.lam[t][0][a0] * b.lam[t][1][a1] * b.lam[t][2][a2] * b.lam[t][3][(int)r];
#pragma unroll
    for (int p = 0; p < 4; p++) { const double v = psi[i + p * slab]; w[p] = fma(v * v, lw, w[p]); }
  }
  __shared__ double sred[8][4];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int p = 0; p < 4; p++) { const double v = warp_sum(w[p]); if (lane == 0) sred[warp][p] = v; }
  __syncthreads();
  if (threadIdx.x < 4) {
    double s = 0.0;
    for (int q = 0; q < 8; q++) s += sred[q][threadIdx.x];
    b.part[t][ch * 4 + threadIdx.x] = s;
  }
}
__global__ void site_weights_final_kernel(SiteWeightBatch b) {
  const int t = blockIdx.x, p = threadIdx.x;
  if (p >= 4) return;
  double s = 0.0;
  for (int ch = 0; ch < PEPO_SW_CHUNKS; ch++) s += b.part[t][ch * 4 + p];
  b.out[t][p] = s;
}

int launch_site_weights(cudaStream_t st, const SiteWeightBatch& b) {
  if (b.count == 0) return 0;
  site_weights_partial_kernel<<<dim3(PEPO_SW_CHUNKS, b.count), 256, 0, st>>>(b);
  PEPO_COUNT_LAUNCH();
  site_weights_final_kernel<<<b.count, 32, 0, st>>>(b);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

// Bond entanglement entropy of the diagnostics table: S_e = -sum_k l_k^2 log l_k^2
// over the live Schmidt weights of bond e (lambda is normalised, eq. (12)); one warp per bond,
// fixed-order reduction.  chi_of_msg[2e] = live dimension of bond e.
__global__ void bond_entropy_kernel(const double* lambda, const int* chi_of_msg, int n_bonds, int chi_max,
                                    double* out) {
  const int e = blockIdx.x;
  if (e >= n_bonds) return;
  const int chi = chi_of_msg[2 * e];
  const double* l = lambda + (size_t)e * chi_max;
  double s = 0.0;
  for (int k = threadIdx.x; k < chi; k += 32) {
    const double w = l[k] * l[k];
    if (w > 0.0) s -= w * log(w);
  }
  s = warp_sum(s);
  if (threadIdx.x == 0) out[e] = s;
}

int launch_bond_entropy(cudaStream_t st, const double* lambda, const int* chi_of_msg, int n_bonds, int chi_max,
                        double* out) {
  if (n_bonds == 0) return 0;
  bond_entropy_kernel<<<n_bonds, 32, 0, st>>>(lambda, chi_of_msg, n_bonds, chi_max, out);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

int launch_bp_init(cudaStream_t st, double* msgs, const int* chi_of_msg, int n_msgs, int chi_max, int mode) {
  if (n_msgs == 0) return 0;
  bp_init_kernel<<<n_msgs, 128, 0, st>>>(msgs, chi_of_msg, n_msgs, chi_max, mode);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

int launch_bethe(cudaStream_t st, const double* vs, int n_sites, const double* msgs,
                 const int* chi_of_msg, int n_bonds, int chi_max, double* out_C, int* out_status) {
  bethe_kernel<<<1, 256, std::max(1, n_bonds) * sizeof(double), st>>>(vs, n_sites, msgs, chi_of_msg,
                                                                     n_bonds, chi_max, out_C, out_status);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

int launch_field_gate(cudaStream_t st, const FieldBatch& b) {
  if (b.count == 0) return 0;
  long long smax = 1;
  for (int t = 0; t < b.count; t++) smax = std::max(smax, b.slab[t]);
  long long g = std::min<long long>((smax + 255) / 256, 148 * 8);
  dim3 grid((unsigned)g, b.count);
  field_gate_kernel<<<grid, 256, 0, st>>>(b);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

}  // namespace pepo
