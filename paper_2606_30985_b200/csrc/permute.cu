// permute.cu - device-side stride-remapping tensor permutation (section 4.1,
// Listing 1; a4/a11 of the hot path), optionally fused with the diagonal
// environment absorption / de-absorption (a3/a12, L93, L103).
//
// The paper's kernel is one thread per element: peel the column-major coordinates of the
// source index, dot with the destination strides, scatter.  That is coalesced on the read side
// only.  Here:
//   * dims that stay adjacent are merged on the host, size-1 dims dropped;
//   * if the fastest dim stays fastest -> `permute_rows_kernel`: both sides are runs of the
//     (merged) fastest dim, index arithmetic by multiply-shift division;
//   * otherwise -> `permute_tiled_kernel`: a shared-memory tile spanning the input-fastest
//     dim, the output-fastest dim and (when one of them is short, e.g. the Pauli dim of size 4)
//     a third dim that lengthens the short side; reads run along the input-fastest dim,
//     writes along the output-fastest dim; odd smem pitch -> conflict-free transposed access.
// Values are moved as 64-bit words (bit-exact); scaling multiplies by per-dim device vectors.
#include "common.cuh"
#include <algorithm>
#include <cstdio>

namespace pepo {
namespace {

constexpr int MAXD = PEPO_MAX_RANK;

struct RowsParams {
  int rank;
  uint32_t total;
  FastDiv fd[MAXD];
  long long ss[MAXD], ds[MAXD];
  const double* scale[MAXD];
};

// generic gather/scatter with fast index arithmetic (fastest dim preserved => coalesced)
template <bool SCALED>
__global__ void __launch_bounds__(256) permute_rows_kernel(const double* __restrict__ src,
                                                           double* __restrict__ dst,
                                                           RowsParams P) {
  constexpr int UNROLL = 4;
  uint32_t base = (blockIdx.x * (uint32_t)blockDim.x * UNROLL) + threadIdx.x;
  double v[UNROLL];
  long long doff[UNROLL];
#pragma unroll
  for (int u = 0; u < UNROLL; u++) {
    uint32_t idx = base + u * blockDim.x;
    doff[u] = -1;
    if (idx < P.total) {
      uint32_t rem = idx;
      long long so = 0, dof = 0;
      double f = 1.0;
#pragma unroll
      for (int d = 0; d < MAXD; d++) {
        if (d < P.rank) {
          uint32_t q = fd_div(rem, P.fd[d]);
          uint32_t c = rem - q * P.fd[d].d;
          rem = q;
          so += (long long)c * P.ss[d];
          dof += (long long)c * P.ds[d];
          if (SCALED && P.scale[d]) f *= __ldg(P.scale[d] + c);
        }
      }
      double x = src[so];
      v[u] = SCALED ? x * f : x;
      doff[u] = dof;
    }
  }
#pragma unroll
  for (int u = 0; u < UNROLL; u++)
    if (doff[u] >= 0) dst[doff[u]] = v[u];
}

struct TiledParams {
  int n_other;                       // dims enumerated by the grid besides the 3 tile dims
  int T[3];                          // tile extents: [0] in-fastest dim, [1] out-fastest dim, [2] third
  int n[3];                          // full sizes of the three tile dims
  FastDiv tiles[3];                  // number of tiles along each tile dim
  FastDiv fdT[3], fdR[3];            // division by the full tile extent / by the remainder extent
  FastDiv fdHT[3], fdHR[3];          // ... by half of them (128-bit variant)
  int rem[3];                        // extent of the last (ragged) tile, = T if it divides
  long long ss[3], ds[3];
  const double* scale[3];
  FastDiv ofd[MAXD];
  long long oss[MAXD], ods[MAXD];
  const double* oscale[MAXD];
  int pitch0;                        // odd smem pitch of tile dim 0
  int in_b_before_a;                 // input enumeration order of dims 1,2 after dim 0
  int out_b_before_0;                // output enumeration order of dims 0,2 after dim 1
};

template <bool SCALED>
__global__ void __launch_bounds__(256) permute_tiled_kernel(const double* __restrict__ src,
                                                            double* __restrict__ dst,
                                                            TiledParams P) {
  extern __shared__ double tile[];
  uint32_t b = blockIdx.x;
  int tc[3], ext[3];
  FastDiv fde[3];
#pragma unroll
  for (int d = 0; d < 3; d++) {
    uint32_t q = fd_div(b, P.tiles[d]);
    tc[d] = b - q * P.tiles[d].d;
    b = q;
    bool last = (tc[d] == (int)P.tiles[d].d - 1);
    ext[d] = last ? P.rem[d] : P.T[d];
    fde[d] = (last && P.rem[d] != P.T[d]) ? P.fdR[d] : P.fdT[d];
  }
  long long sbase = 0, dbase = 0;
  double fo = 1.0;
#pragma unroll
  for (int d = 0; d < 3; d++) {
    sbase += (long long)tc[d] * P.T[d] * P.ss[d];
    dbase += (long long)tc[d] * P.T[d] * P.ds[d];
  }
  for (int d = 0; d < P.n_other; d++) {
    uint32_t q = fd_div(b, P.ofd[d]);
    uint32_t c = b - q * P.ofd[d].d;
    b = q;
    sbase += (long long)c * P.oss[d];
    dbase += (long long)c * P.ods[d];
    if (SCALED && P.oscale[d]) fo *= __ldg(P.oscale[d] + c);
  }
  const int E = ext[0] * ext[1] * ext[2];
  const int pitch0 = P.pitch0, T1 = P.T[1];
  // phase 1: read along the input-fastest dim
  for (int e = threadIdx.x; e < E; e += blockDim.x) {
    uint32_t q = fd_div(e, fde[0]);
    int i0 = e - q * ext[0];
    int i1, i2;
    if (P.in_b_before_a) {
      uint32_t q2 = fd_div(q, fde[2]);
      i2 = q - q2 * ext[2]; i1 = q2;
    } else {
      uint32_t q2 = fd_div(q, fde[1]);
      i1 = q - q2 * ext[1]; i2 = q2;
    }
    double x = src[sbase + i0 * P.ss[0] + i1 * P.ss[1] + i2 * P.ss[2]];
    if (SCALED) {
      double f = fo;
      if (P.scale[0]) f *= __ldg(P.scale[0] + tc[0] * P.T[0] + i0);
      if (P.scale[1]) f *= __ldg(P.scale[1] + tc[1] * P.T[1] + i1);
      if (P.scale[2]) f *= __ldg(P.scale[2] + tc[2] * P.T[2] + i2);
      x *= f;
    }
    tile[i0 + pitch0 * (i1 + T1 * i2)] = x;
  }
  __syncthreads();
  // phase 2: write along the output-fastest dim
  for (int e = threadIdx.x; e < E; e += blockDim.x) {
    uint32_t q = fd_div(e, fde[1]);
    int i1 = e - q * ext[1];
    int i0, i2;
    if (P.out_b_before_0) {
      uint32_t q2 = fd_div(q, fde[2]);
      i2 = q - q2 * ext[2]; i0 = q2;
    } else {
      uint32_t q2 = fd_div(q, fde[0]);
      i0 = q - q2 * ext[0]; i2 = q2;
    }
    dst[dbase + i0 * P.ds[0] + i1 * P.ds[1] + i2 * P.ds[2]] = tile[i0 + pitch0 * (i1 + T1 * i2)];
  }
}

// ---------------------------------------------------------------------------------------------
// 128-bit variants (the fast path): every global access is a 16-byte vector of two doubles.
// Preconditions (checked by launch_permute): 16-byte aligned base pointers; the input-fastest
// and the output-fastest (merged) dims have even extents; every other stride is even.
// ---------------------------------------------------------------------------------------------
struct RowsV2Params {
  int rank;                          // dims incl. dim 0 (counted in double2 units)
  uint32_t total2;                   // number of double2
  FastDiv fd[MAXD];                  // fd[0] divides by n0/2
  long long ss[MAXD], ds[MAXD];      // strides in doubles (ss[0] = ds[0] = 1 -> 2 per vector)
  const double* scale[MAXD];
};

// VPT consecutive double2 of one row per thread: the index decomposition and the product of the
// outer scale factors are shared by VPT vectors (VPT divides n0/2).
template <bool SCALED, int VPT>
__global__ void __launch_bounds__(256) permute_rows_v2_kernel(const double* __restrict__ src,
                                                              double* __restrict__ dst,
                                                              RowsV2Params P) {
  constexpr int UNROLL = (VPT >= 4) ? 2 : 4;
  const uint32_t base = (blockIdx.x * (uint32_t)blockDim.x * UNROLL) + threadIdx.x;
  double2 v[UNROLL][VPT];
  long long doff[UNROLL];
#pragma unroll
  for (int u = 0; u < UNROLL; u++) {
    const uint32_t idx = base + u * blockDim.x;          // index of a group of VPT vectors
    doff[u] = -1;
    if (idx < P.total2) {
      uint32_t rem = fd_div(idx, P.fd[0]);               // fd[0] divides by n0/(2 VPT)
      const uint32_t j0 = (idx - rem * P.fd[0].d) * VPT;
      long long so = 2ll * j0, dof = 2ll * j0;
      double f = 1.0;
#pragma unroll
      for (int d = 1; d < MAXD; d++) {
        if (d < P.rank) {
          uint32_t q = fd_div(rem, P.fd[d]);
          uint32_t c = rem - q * P.fd[d].d;
          rem = q;
          so += (long long)c * P.ss[d];
          dof += (long long)c * P.ds[d];
          if (SCALED && P.scale[d]) f *= __ldg(P.scale[d] + c);
        }
      }
      const double2* sp = reinterpret_cast<const double2*>(src + so);
#pragma unroll
      for (int w = 0; w < VPT; w++) v[u][w] = sp[w];
      if (SCALED) {
        if (P.scale[0]) {
          const double2* s0 = reinterpret_cast<const double2*>(P.scale[0] + 2 * j0);   // 16-byte aligned: checked on the host
#pragma unroll
          for (int w = 0; w < VPT; w++) { const double2 g = __ldg(s0 + w); v[u][w].x *= f * g.x; v[u][w].y *= f * g.y; }
        } else {
#pragma unroll
          for (int w = 0; w < VPT; w++) { v[u][w].x *= f; v[u][w].y *= f; }
        }
      }
      doff[u] = dof;
    }
  }
#pragma unroll
  for (int u = 0; u < UNROLL; u++)
    if (doff[u] >= 0) {
      double2* dp = reinterpret_cast<double2*>(dst + doff[u]);
#pragma unroll
      for (int w = 0; w < VPT; w++) dp[w] = v[u][w];
    }
}

// Tiled transpose, same tile geometry as permute_tiled_kernel (TiledParams); T[0], T[1] and the
// ragged remainders are even.  Phase 1 reads double2 along the input-fastest dim and stores the
// two halves as 64-bit shared stores (odd pitch: conflict-free); phase 2 gathers two 64-bit
// values one pitch apart and writes a double2 along the output-fastest dim.
template <bool SCALED>
__global__ void __launch_bounds__(256) permute_tiled_v2_kernel(const double* __restrict__ src,
                                                               double* __restrict__ dst,
                                                               TiledParams P) {
  extern __shared__ double tile[];
  uint32_t b = blockIdx.x;
  int tc[3], ext[3];
  bool ragged[3];
#pragma unroll
  for (int d = 0; d < 3; d++) {
    uint32_t q = fd_div(b, P.tiles[d]);
    tc[d] = b - q * P.tiles[d].d;
    b = q;
    bool last = (tc[d] == (int)P.tiles[d].d - 1);
    ext[d] = last ? P.rem[d] : P.T[d];
    ragged[d] = last && P.rem[d] != P.T[d];
  }
  const FastDiv fh0 = ragged[0] ? P.fdHR[0] : P.fdHT[0];   // divide by ext[0]/2
  const FastDiv fh1 = ragged[1] ? P.fdHR[1] : P.fdHT[1];   // divide by ext[1]/2
  const FastDiv fe0 = ragged[0] ? P.fdR[0] : P.fdT[0];
  const FastDiv fe1 = ragged[1] ? P.fdR[1] : P.fdT[1];
  const FastDiv fe2 = ragged[2] ? P.fdR[2] : P.fdT[2];
  long long sbase = 0, dbase = 0;
#pragma unroll
  for (int d = 0; d < 3; d++) {
    sbase += (long long)tc[d] * P.T[d] * P.ss[d];
    dbase += (long long)tc[d] * P.T[d] * P.ds[d];
  }
  // scale factors of the dims enumerated by the grid: the loads are issued here, the product is
  // formed only after the first batch of tile loads is in flight (in-order issue would otherwise
  // stall the whole tile on two dependent L2 round trips)
  double fsc[MAXD];
#pragma unroll
  for (int d = 0; d < MAXD; d++) fsc[d] = 1.0;
#pragma unroll
  for (int d = 0; d < MAXD; d++) {
    if (d < P.n_other) {
      uint32_t q = fd_div(b, P.ofd[d]);
      uint32_t c = b - q * P.ofd[d].d;
      b = q;
      sbase += (long long)c * P.oss[d];
      dbase += (long long)c * P.ods[d];
      if (SCALED && P.oscale[d]) fsc[d] = __ldg(P.oscale[d] + c);
    }
  }
  const int pitch0 = P.pitch0, T1 = P.T[1];
  constexpr int UN = 4;
  // ---- phase 1 -------------------------------------------------------------------------------
  {
    const int E2 = (ext[0] >> 1) * ext[1] * ext[2];
    for (int e0 = threadIdx.x; e0 < E2; e0 += 256 * UN) {
      double2 x[UN];
      int so[UN];
      int c0[UN], c1[UN], c2[UN];
#pragma unroll
      for (int u = 0; u < UN; u++) {
        const int e = e0 + u * 256;
        so[u] = -1;
        if (e < E2) {
          uint32_t q = fd_div(e, fh0);
          const int j0 = e - q * fh0.d;
          int i1, i2;
          if (P.in_b_before_a) { uint32_t q2 = fd_div(q, fe2); i2 = q - q2 * fe2.d; i1 = q2; }
          else { uint32_t q2 = fd_div(q, fe1); i1 = q - q2 * fe1.d; i2 = q2; }
          x[u] = *reinterpret_cast<const double2*>(src + sbase + 2 * j0 + i1 * P.ss[1] + i2 * P.ss[2]);
          so[u] = 2 * j0 + pitch0 * (i1 + T1 * i2);
          c0[u] = 2 * j0; c1[u] = i1; c2[u] = i2;
        }
      }
      double fo = 1.0;
      if (SCALED) {
#pragma unroll
        for (int d = 0; d < MAXD; d++) fo *= fsc[d];
      }
#pragma unroll
      for (int u = 0; u < UN; u++)
        if (so[u] >= 0) {
          double2 v = x[u];
          if (SCALED) {
            double f = fo;
            if (P.scale[1]) f *= __ldg(P.scale[1] + tc[1] * P.T[1] + c1[u]);
            if (P.scale[2]) f *= __ldg(P.scale[2] + tc[2] * P.T[2] + c2[u]);
            double f0 = f, f1 = f;
            if (P.scale[0]) {
              f0 *= __ldg(P.scale[0] + tc[0] * P.T[0] + c0[u]);
              f1 *= __ldg(P.scale[0] + tc[0] * P.T[0] + c0[u] + 1);
            }
            v.x *= f0; v.y *= f1;
          }
          tile[so[u]] = v.x; tile[so[u] + 1] = v.y;
        }
    }
  }
  __syncthreads();
  // ---- phase 2 -------------------------------------------------------------------------------
  {
    const int E2 = ext[0] * (ext[1] >> 1) * ext[2];
    for (int e = threadIdx.x; e < E2; e += 256) {
      uint32_t q = fd_div(e, fh1);
      const int j1 = e - q * fh1.d;
      int i0, i2;
      if (P.out_b_before_0) { uint32_t q2 = fd_div(q, fe2); i2 = q - q2 * fe2.d; i0 = q2; }
      else { uint32_t q2 = fd_div(q, fe0); i0 = q - q2 * fe0.d; i2 = q2; }
      const int so = i0 + pitch0 * (2 * j1 + T1 * i2);
      double2 v;
      v.x = tile[so];
      v.y = tile[so + pitch0];
      *reinterpret_cast<double2*>(dst + dbase + i0 * P.ds[0] + 2 * j1 + i2 * P.ds[2]) = v;
    }
  }
}

inline int even_tile(int n, int cap) {      // n even: balanced even tile extent <= ~cap
  int parts = (n + cap - 1) / cap;
  int t = (n + parts - 1) / parts;
  return (t + 1) & ~1;
}

inline int balanced_tile(int n, int cap) {
  int parts = (n + cap - 1) / cap;
  return (n + parts - 1) / parts;
}

}  // namespace

int launch_permute(cudaStream_t st, const double* src, double* dst, const PermuteDesc& D) {
  if (D.rank < 1 || D.rank > MAXD) { set_error("permute: rank %d unsupported", D.rank); return -1; }
  // inverse perm: position of input dim d in the output
  int pos[MAXD];
  for (int j = 0; j < D.rank; j++) {
    if (D.perm[j] < 0 || D.perm[j] >= D.rank) { set_error("permute: bad perm"); return -1; }
    pos[D.perm[j]] = j;
  }
  long long total = 1;
  for (int d = 0; d < D.rank; d++) {
    if (D.shape[d] < 0) { set_error("permute: negative extent"); return -1; }
    total *= D.shape[d];
  }
  if (total == 0) return 0;
  if (total >= (1ll << 31)) { set_error("permute: tensor too large (%lld elements)", total); return -1; }
  // simplified dims in input order
  int n[MAXD]; long long ss[MAXD], ds[MAXD]; const double* sc[MAXD]; int opos[MAXD];
  int r = 0;
  bool scaled = false;
  for (int d = 0; d < D.rank; d++) {
    if (D.shape[d] == 1) continue;
    long long s_s = D.src_stride[d], d_s = D.dst_stride[pos[d]];
    const double* scl = D.scale[d];
    if (scl) scaled = true;
    if (r > 0 && !scl && !sc[r - 1] && ss[r - 1] * n[r - 1] == s_s && ds[r - 1] * n[r - 1] == d_s &&
        (long long)n[r - 1] * D.shape[d] < (1 << 30)) {
      n[r - 1] *= D.shape[d];           // merge with the previous dim
      continue;
    }
    n[r] = D.shape[d]; ss[r] = s_s; ds[r] = d_s; sc[r] = scl; opos[r] = pos[d]; r++;
  }
  if (r == 0) {                          // single element
    n[0] = 1; ss[0] = 1; ds[0] = 1; sc[0] = nullptr; r = 1;
  }
  // out-fastest dim among the simplified dims
  int a = 0;
  for (int d = 1; d < r; d++) if (ds[d] < ds[a]) a = d;

  // ---- 128-bit fast paths ---------------------------------------------------------------------
  bool vec = (((uintptr_t)src | (uintptr_t)dst) & 15) == 0 && ss[0] == 1 && ds[a] == 1 &&
             (n[0] % 2 == 0) && (n[a] % 2 == 0);
  for (int d = 0; d < r && vec; d++) {
    if (d != 0 && (ss[d] & 1)) vec = false;
    if (d != a && (ds[d] & 1)) vec = false;
  }
  if (vec && a == 0) {
    RowsV2Params P;
    const int h0 = n[0] / 2;
    const bool s0_al = !sc[0] || (((uintptr_t)sc[0] & 15) == 0);
    // measured: sharing the index / scale arithmetic between two vectors pays only in the scaled
    // variant (0.72 -> 0.80 of HBM peak); plain copies are fastest with one vector per thread
    const int vpt = (scaled && h0 % 2 == 0 && s0_al) ? 2 : 1;
    const long long groups = total / 2 / vpt;
    P.rank = r; P.total2 = (uint32_t)groups;
    for (int d = 0; d < MAXD; d++) {
      if (d < r) { P.fd[d] = make_fastdiv(d == 0 ? h0 / vpt : n[d]); P.ss[d] = ss[d]; P.ds[d] = ds[d]; P.scale[d] = sc[d]; }
      else { P.fd[d] = make_fastdiv(1); P.ss[d] = 0; P.ds[d] = 0; P.scale[d] = nullptr; }
    }
    const int per_block = 256 * (vpt >= 4 ? 2 : 4);
    unsigned blocks = (unsigned)((groups + per_block - 1) / per_block);
    if (vpt == 4) {
      if (scaled) permute_rows_v2_kernel<true, 4><<<blocks, 256, 0, st>>>(src, dst, P);
      else permute_rows_v2_kernel<false, 4><<<blocks, 256, 0, st>>>(src, dst, P);
    } else if (vpt == 2) {
      if (scaled) permute_rows_v2_kernel<true, 2><<<blocks, 256, 0, st>>>(src, dst, P);
      else permute_rows_v2_kernel<false, 2><<<blocks, 256, 0, st>>>(src, dst, P);
    } else {
      if (scaled) permute_rows_v2_kernel<true, 1><<<blocks, 256, 0, st>>>(src, dst, P);
      else permute_rows_v2_kernel<false, 1><<<blocks, 256, 0, st>>>(src, dst, P);
    }
    PEPO_COUNT_LAUNCH();
    PEPO_CUDA_OK(cudaGetLastError());
    return 0;
  }
  if (vec && total >= 4096) {
    // tile = (dim 0) x (dim a) [x third dim when the tile would be small]: ~2048-4096 elements
    // a short side (e.g. the Pauli dim, extent 4) is compensated by a longer other side
    const int cap0 = (n[a] < 32) ? std::min(1024, 2048 / n[a]) : 64;
    const int capa = (n[0] < 32) ? std::min(1024, 2048 / n[0]) : 64;
    const int T0 = even_tile(n[0], cap0), Ta = even_tile(n[a], capa);
    int bdim = -1, Tb = 1;
    if (T0 * Ta < 2048 && r > 2) {
      int ob = -1, ib = -1;              // next dim in output order after a / in input order after 0
      for (int d = 0; d < r; d++) {
        if (d == a || d == 0) continue;
        if (ob < 0 || ds[d] < ds[ob]) ob = d;
        if (ib < 0 || ss[d] < ss[ib]) ib = d;
      }
      // a short output run is lengthened by the next output dim unless that is dim 0 itself
      // (then the run is already n[a]*n[0] long); otherwise lengthen the input side
      bool out_next_is_0 = true;
      for (int d = 1; d < r; d++) if (d != a && ds[d] < ds[0]) out_next_is_0 = false;
      if (Ta < 32 && !out_next_is_0) bdim = ob; else bdim = ib;
      if (bdim >= 0) {
        int want = (2048 + T0 * Ta - 1) / (T0 * Ta);
        Tb = balanced_tile(n[bdim], std::min(n[bdim], want));
      }
    }
    TiledParams P;
    const int td[3] = {0, a, bdim};
    const int Tt[3] = {T0, Ta, Tb};
    long long nblocks = 1;
    for (int k = 0; k < 3; k++) {
      int d = td[k];
      int nn = (d >= 0) ? n[d] : 1;
      P.T[k] = Tt[k]; P.n[k] = nn;
      int nt = (nn + Tt[k] - 1) / Tt[k];
      P.tiles[k] = make_fastdiv(nt);
      P.rem[k] = nn - (nt - 1) * Tt[k];
      P.fdT[k] = make_fastdiv(Tt[k]);
      P.fdR[k] = make_fastdiv(P.rem[k]);
      P.fdHT[k] = make_fastdiv(std::max(Tt[k] / 2, 1));
      P.fdHR[k] = make_fastdiv(std::max(P.rem[k] / 2, 1));
      P.ss[k] = (d >= 0) ? ss[d] : 0;
      P.ds[k] = (d >= 0) ? ds[d] : 0;
      P.scale[k] = (d >= 0) ? sc[d] : nullptr;
      nblocks *= nt;
    }
    P.n_other = 0;
    for (int d = 0; d < MAXD; d++) { P.ofd[d] = make_fastdiv(1); P.oss[d] = 0; P.ods[d] = 0; P.oscale[d] = nullptr; }
    for (int d = 1; d < r; d++) {
      if (d == a || d == bdim) continue;
      int k = P.n_other++;
      P.ofd[k] = make_fastdiv(n[d]); P.oss[k] = ss[d]; P.ods[k] = ds[d]; P.oscale[k] = sc[d];
      nblocks *= n[d];
    }
    if (nblocks >= (1ll << 31)) { set_error("permute: grid too large"); return -1; }
    P.pitch0 = T0 | 1;
    P.in_b_before_a = (bdim >= 0 && ss[bdim] < ss[a]) ? 1 : 0;
    P.out_b_before_0 = (bdim >= 0 && ds[bdim] < ds[0]) ? 1 : 0;
    size_t smem = (size_t)P.pitch0 * Ta * Tb * sizeof(double);
    if (scaled) permute_tiled_v2_kernel<true><<<(unsigned)nblocks, 256, smem, st>>>(src, dst, P);
    else permute_tiled_v2_kernel<false><<<(unsigned)nblocks, 256, smem, st>>>(src, dst, P);
    PEPO_COUNT_LAUNCH();
    PEPO_CUDA_OK(cudaGetLastError());
    return 0;
  }
  // ---- generic 64-bit paths (odd extents / misaligned) ---------------------------------------
  const bool tiled = (a != 0) && ss[0] == 1 && ds[a] == 1 && total >= 4096;
  if (!tiled) {
    RowsParams P;
    P.rank = r; P.total = (uint32_t)total;
    for (int d = 0; d < MAXD; d++) {
      if (d < r) { P.fd[d] = make_fastdiv(n[d]); P.ss[d] = ss[d]; P.ds[d] = ds[d]; P.scale[d] = sc[d]; }
      else { P.fd[d] = make_fastdiv(1); P.ss[d] = 0; P.ds[d] = 0; P.scale[d] = nullptr; }
    }
    unsigned blocks = (unsigned)((total + 1023) / 1024);
    if (scaled) permute_rows_kernel<true><<<blocks, 256, 0, st>>>(src, dst, P);
    else permute_rows_kernel<false><<<blocks, 256, 0, st>>>(src, dst, P);
    PEPO_COUNT_LAUNCH();
    PEPO_CUDA_OK(cudaGetLastError());
    return 0;
  }
  // ---- tiled path -------------------------------------------------------------------------
  // third dim: lengthen the short side
  int bdim = -1;
  if (n[a] < 32) {
    // next output dim after a
    int best = -1;
    for (int d = 0; d < r; d++) if (d != a && (best < 0 || ds[d] < ds[best])) best = d;
    if (best > 0) bdim = best;               // (best == 0: the output run is already a*dim0)
  } else if (n[0] < 32) {
    int best = -1;
    for (int d = 1; d < r; d++) if (best < 0 || ss[d] < ss[best]) best = d;
    if (best != a) bdim = best;
  }
  TiledParams P;
  int td[3] = {0, a, bdim};
  int T0 = balanced_tile(n[0], 64), Ta = balanced_tile(n[a], 64), Tb = 1;
  if (bdim >= 0) {
    int shortside = (n[a] < 32) ? Ta : T0;
    int want = (64 + shortside - 1) / shortside;
    Tb = std::min(n[bdim], want);
    Tb = balanced_tile(n[bdim], Tb);
  }
  int Tt[3] = {T0, Ta, Tb};
  long long nblocks = 1;
  for (int k = 0; k < 3; k++) {
    int d = td[k];
    int nn = (d >= 0) ? n[d] : 1;
    P.T[k] = Tt[k]; P.n[k] = nn;
    int nt = (nn + Tt[k] - 1) / Tt[k];
    P.tiles[k] = make_fastdiv(nt);
    P.rem[k] = nn - (nt - 1) * Tt[k];
    P.fdT[k] = make_fastdiv(Tt[k]);
    P.fdR[k] = make_fastdiv(P.rem[k]);
    P.ss[k] = (d >= 0) ? ss[d] : 0;
    P.ds[k] = (d >= 0) ? ds[d] : 0;
    P.scale[k] = (d >= 0) ? sc[d] : nullptr;
    nblocks *= nt;
  }
  P.n_other = 0;
  for (int d = 0; d < MAXD; d++) { P.ofd[d] = make_fastdiv(1); P.oss[d] = 0; P.ods[d] = 0; P.oscale[d] = nullptr; }
  for (int d = 1; d < r; d++) {
    if (d == a || d == bdim) continue;
    int k = P.n_other++;
    P.ofd[k] = make_fastdiv(n[d]); P.oss[k] = ss[d]; P.ods[k] = ds[d]; P.oscale[k] = sc[d];
    nblocks *= n[d];
  }
  if (nblocks >= (1ll << 31)) { set_error("permute: grid too large"); return -1; }
  P.pitch0 = T0 | 1;
  P.in_b_before_a = (bdim >= 0 && ss[bdim] < ss[a]) ? 1 : 0;
  P.out_b_before_0 = (bdim >= 0 && ds[bdim] < ds[0]) ? 1 : 0;
  size_t smem = (size_t)P.pitch0 * Ta * Tb * sizeof(double);
  if (scaled) permute_tiled_kernel<true><<<(unsigned)nblocks, 256, smem, st>>>(src, dst, P);
  else permute_tiled_kernel<false><<<(unsigned)nblocks, 256, smem, st>>>(src, dst, P);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  (void)opos;
  return 0;
}

}  // namespace pepo
