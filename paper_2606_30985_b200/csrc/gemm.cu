// gemm.cu - fp64 tensor-core (DMMA, mma.sync.m8n8k4.f64) GEMM for the three dense
// contractions of the hot path: the Gram matrix C = cv^T cv of eq. (10),
// the reconstruction cv_new = cv (R^-1 M) of a10 (L102, L331-L333) and the small core
// products (a7).  sm_100a lowers every f64 mma shape to DMMA.8x8x4, measured 36.9 TFLOP/s
// on B200 (= the DFMA peak), so the tile loop is built on m8n8k4 directly.
//
// Tiling: CTA tile BM x BN x 16, warp tile WM x WN built from 8x8 accumulator fragments,
// operands staged global -> shared with cp.async (16-byte when aligned, 8-byte otherwise,
// zero-filled outside the matrix) through a STAGES-deep ring; shared tiles are XOR-swizzled
// so that the 64-bit fragment loads of a half-warp hit 16 distinct bank pairs.
#include "common.cuh"
#include <cstdlib>
#include <cstring>

namespace pepo {

namespace {

constexpr int BK = 16;

__device__ __forceinline__ void dmma8x8x4(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, int src_bytes) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async8(void* smem, const void* gmem, int src_bytes) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}

// Copy one operand tile of `ROWS` "outer" indices x 16 k into shared memory.
//  KCONTIG = true : element (r, k) at g[(k0+k) + (r0+r)*ld]; smem s[r*16 + (k ^ 4*(r&3))]
//  KCONTIG = false: element (r, k) at g[(r0+r) + (k0+k)*ld]; smem s[k*ROWS + (r ^ 4*(k&3))]
// rows >= nrows or k >= kend are zero-filled.
template <int ROWS, bool KCONTIG, int NT>
__device__ __forceinline__ void load_tile(double* s, const double* __restrict__ g, long long ld,
                                          long long r0, long long nrows, int k0, int kend,
                                          bool aligned, int tid) {
  constexpr int CHUNKS = ROWS * 8;   // 16-byte chunks
#pragma unroll
  for (int c = tid; c < CHUNKS; c += NT) {
    if (KCONTIG) {
      int r = c >> 3, kk = (c & 7) * 2;
      long long gr = r0 + r;
      int gk = k0 + kk;
      int nvalid = (gr < nrows) ? max(0, min(2, kend - gk)) : 0;
      double* dst = s + r * 16 + (kk ^ (4 * (r & 3)));
      const double* src = g + (nvalid ? ((long long)gk + gr * ld) : 0);
      if (aligned) {
        cp_async16(dst, src, nvalid * 8);
      } else {
        cp_async8(dst, src, nvalid >= 1 ? 8 : 0);
        cp_async8(dst + 1, nvalid >= 2 ? src + 1 : src, nvalid >= 2 ? 8 : 0);
      }
    } else {
      int k = c / (ROWS / 2), rr = (c % (ROWS / 2)) * 2;
      long long gr = r0 + rr;
      int gk = k0 + k;
      int nvalid = (gk < kend) ? (int)max(0ll, min(2ll, nrows - gr)) : 0;
      double* dst = s + k * ROWS + (rr ^ (4 * (k & 3)));
      const double* src = g + (nvalid ? (gr + (long long)gk * ld) : 0);
      if (aligned) {
        cp_async16(dst, src, nvalid * 8);
      } else {
        cp_async8(dst, src, nvalid >= 1 ? 8 : 0);
        cp_async8(dst + 1, nvalid >= 2 ? src + 1 : src, nvalid >= 2 ? 8 : 0);
      }
    }
  }
}

__device__ __forceinline__ long long idx2_off(const Idx2& f, uint32_t i) {
  if (f.E.d == 0) return f.s * (long long)i;
  const uint32_t q = fd_div(i, f.E), r = i - q * f.E.d;
  return f.s * (long long)r + f.T * (long long)q;
}

// Gathered operand tile (see GemmGather in common.cuh).  What is fixed over the k loop lives in
// registers: the address of every chunk's first element at k = 0 (p0), the distance to its second
// element (d1, only read on the unaligned path) and how many of the two are inside the matrix (nb).
// Per stage only the k part of the offset is added: one value per thread for a K-contiguous operand
// (all chunks of a thread share their k pair), one per chunk otherwise - s * k for a plain stride, or a
// look-up in a per-CTA table of the two-level offsets (ktab, built once at kernel start; the operand
// of the reconstruction GEMM whose k index is (cut, P)).  Same shared-memory layout as load_tile.
template <int ROWS, bool KCONTIG, int NT>
struct GatherSlots {
  static constexpr int S = (ROWS * 8 + NT - 1) / NT;
  const double* p0[S];
  long long d1[S];
  int nb[S];
};
template <int ROWS, bool KCONTIG, int NT>
__device__ __forceinline__ void gather_init(GatherSlots<ROWS, KCONTIG, NT>& G, const double* g, const Idx2& fo,
                                            long long r0, long long nrows, int tid) {
#pragma unroll
  for (int i = 0; i < GatherSlots<ROWS, KCONTIG, NT>::S; i++) {
    const int c = tid + i * NT;
    G.p0[i] = g; G.d1[i] = 0; G.nb[i] = 0;
    if (c >= ROWS * 8) continue;
    if (KCONTIG) {
      const long long gr = r0 + (c >> 3);
      if (gr < nrows) { G.p0[i] = g + idx2_off(fo, (uint32_t)gr); G.nb[i] = 2; }
    } else {
      const long long gr = r0 + (c % (ROWS / 2)) * 2;
      if (gr < nrows) {
        const long long o0 = idx2_off(fo, (uint32_t)gr);
        G.p0[i] = g + o0; G.nb[i] = 1;
        if (gr + 1 < nrows) { G.d1[i] = idx2_off(fo, (uint32_t)(gr + 1)) - o0; G.nb[i] = 2; }
      }
    }
  }
}
// KTAB (non-K-contiguous operand only): the k offsets come from the per-CTA table, with no run-time choice
// between table / plain stride / two-level arithmetic inside the chunk loop (that choice compiled to three
// divergence-guarded branches per 16-byte chunk: ~45 instructions, against ~12 for the look-up)
template <int ROWS, bool KCONTIG, int NT, bool KTAB = false>
__device__ __forceinline__ void load_tile_gather(double* s, const GatherSlots<ROWS, KCONTIG, NT>& G,
                                                 const Idx2& fk, const long long* __restrict__ ktab, int kbeg,
                                                 int k0, int kend, bool aligned, int tid) {
  static_assert(NT % 8 == 0, "a thread keeps one k pair for all its chunks");
  if (KCONTIG) {
    const int kk = (tid & 7) * 2;
    const int gk = k0 + kk;
    const int kvalid = max(0, min(2, kend - gk));
    const long long ok0 = kvalid ? idx2_off(fk, (uint32_t)gk) : 0;
    const long long dk = (!aligned && kvalid >= 2) ? idx2_off(fk, (uint32_t)(gk + 1)) - ok0 : 0;
#pragma unroll
    for (int i = 0; i < GatherSlots<ROWS, KCONTIG, NT>::S; i++) {
      const int c = tid + i * NT;
      if (c >= ROWS * 8) continue;
      const int r = c >> 3;
      const int nvalid = G.nb[i] ? kvalid : 0;
      double* dst = s + r * 16 + (kk ^ (4 * (r & 3)));
      const double* src = G.p0[i] + (nvalid ? ok0 : 0);
      if (aligned) {
        cp_async16(dst, src, nvalid * 8);
      } else {
        cp_async8(dst, src, nvalid >= 1 ? 8 : 0);
        cp_async8(dst + 1, nvalid >= 2 ? src + dk : src, nvalid >= 2 ? 8 : 0);
      }
    }
  } else {
#pragma unroll
    for (int i = 0; i < GatherSlots<ROWS, KCONTIG, NT>::S; i++) {
      const int c = tid + i * NT;
      if (c >= ROWS * 8) continue;
      const int k = c / (ROWS / 2), rr = (c % (ROWS / 2)) * 2;
      const int gk = k0 + k;
      const int nvalid = (gk < kend) ? G.nb[i] : 0;
      double* dst = s + k * ROWS + (rr ^ (4 * (k & 3)));
      long long okk = 0;
      if (KTAB) okk = ktab[nvalid ? gk - kbeg : 0];
      else if (nvalid) okk = (fk.E.d == 0) ? fk.s * (long long)gk : (ktab ? ktab[gk - kbeg] : idx2_off(fk, (uint32_t)gk));
      const double* src = G.p0[i] + okk;
      if (aligned) {
        cp_async16(dst, src, nvalid * 8);
      } else {
        cp_async8(dst, src, nvalid >= 1 ? 8 : 0);
        cp_async8(dst + 1, nvalid >= 2 ? src + G.d1[i] : src, nvalid >= 2 ? 8 : 0);
      }
    }
  }
}

constexpr int GW_MAXLEN = 256;      // longest weight vector (chi_max <= 256)

// MINB: resident CTAs per SM the register allocation must allow (3 for the 64 x 80 tile: 170 registers)
// AL: the host has checked that both operands take the 16-byte cp.async path in every stage (the
// 8-byte fallback is then not compiled in: the unrolled main loop is half the size, which matters for
// the instruction cache of the short-K reconstruction CTAs)
// WGT: row weights on the k index (the weighted Gram); a run-time test of it in the main loop is
// if-converted into a multiply by 1.0 that every kernel would execute
template <int TA, int TB, int BM, int BN, int WM, int WN, int STAGES, bool GATHER, bool AL, bool WGT>
__global__ void __launch_bounds__((BM / WM) * (BN / WN) * 32, (BM == 64 && BN == 80) ? 3 : 1)
dgemm_dmma_kernel(GemmProb p0, const GemmProb* __restrict__ probs, int ksplit, int kchunk,
                  double* __restrict__ part, int upper_only, GemmGather gg) {
  constexpr int NT = (BM / WM) * (BN / WN) * 32;
  constexpr int MI = WM / 8, NI = WN / 8;
  constexpr bool A_KC = (TA == 1), B_KC = (TB == 0);
  extern __shared__ __align__(16) double smem[];
  double* sA = smem;                       // STAGES * BM*16
  double* sB = smem + STAGES * BM * BK;    // STAGES * BN*16
  // GATHER extras: weighted Gram: STAGES * 16 row weights + 3 weight vectors; reconstruction: the
  // table of the two-level k offsets of operand A (never both)
  double* sW = sB + STAGES * BN * BK;
  double* sV = sW + STAGES * BK;
  long long* sK = reinterpret_cast<long long*>(sW);

  GemmProb p = p0;
  int split = 0;
  if (probs) {
    p = probs[blockIdx.z];
  } else {
    split = blockIdx.z;
  }
  const long long M = p.M;
  const int N = p.N, K = p.K;
  const int tilesN = (N + BN - 1) / BN;
  const long long tilesM = (M + BM - 1) / BM;
  const long long tile = blockIdx.x;
  if (tile >= tilesM * tilesN) return;
  const long long tm = tile / tilesN;
  const int tn = (int)(tile % tilesN);
  if (upper_only && tn < tm) return;
  const long long m0 = tm * BM;
  const int n0 = tn * BN;
  int kbeg = 0, kend = K;
  if (ksplit > 1) {
    kbeg = split * kchunk;
    kend = min(K, kbeg + kchunk);
  }
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g = lane >> 2, t = lane & 3;
  const int wm0 = (warp % (BM / WM)) * WM, wn0 = (warp / (BM / WM)) * WN;

  const bool alignedA = AL ? true : GATHER ? (gg.alignedA != 0 && (kbeg & 1) == 0)
                               : ((((uintptr_t)p.A & 15) == 0) && ((p.lda & 1) == 0) && ((kbeg & 1) == 0));
  const bool alignedB = AL ? true : GATHER ? (gg.alignedB != 0 && (kbeg & 1) == 0)
                               : ((((uintptr_t)p.B & 15) == 0) && ((p.ldb & 1) == 0) && ((kbeg & 1) == 0));
  GatherSlots<BM, A_KC, NT> gsA;
  GatherSlots<BN, B_KC, NT> gsB;
  constexpr bool weighted = GATHER && WGT;
  if (GATHER) {
    gather_init<BM, A_KC, NT>(gsA, p.A, gg.a_outer, m0, M, tid);
    gather_init<BN, B_KC, NT>(gsB, p.B, gg.b_outer, n0, N, tid);
    if (gg.ktabA) {
      for (int k = tid; k < kend - kbeg; k += NT) sK[k] = idx2_off(gg.a_k, (uint32_t)(kbeg + k));
      __syncthreads();
    }
    if (weighted) {
      for (int v = 0; v < 3; v++)
        for (int i = tid; i < GW_MAXLEN; i += NT) sV[v * GW_MAXLEN + i] = (v < gg.nw && i < gg.wlen[v]) ? gg.wv[v][i] : 1.0;
      __syncthreads();
    }
  }

  // Gram (upper_only) diagonal tiles: a warp tile strictly below the diagonal is never read by the
  // reducer, so its warp only helps with the loads (frees its DMMA issue slots for co-resident CTAs)
  const bool skip_warp = upper_only && tn == tm && BM == BN && (wm0 >= wn0 + WN);
  double acc[MI][NI][2];
#pragma unroll
  for (int i = 0; i < MI; i++)
#pragma unroll
    for (int j = 0; j < NI; j++) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }

  const int nk = (kend - kbeg + BK - 1) / BK;
  auto issue = [&](int it, int st) {
    if (it < nk) {
      int k0 = kbeg + it * BK;
      if (GATHER) {
        if (!A_KC && gg.ktabA) load_tile_gather<BM, A_KC, NT, true>(sA + st * BM * BK, gsA, gg.a_k, sK, kbeg, k0, kend, alignedA, tid);
        else load_tile_gather<BM, A_KC, NT>(sA + st * BM * BK, gsA, gg.a_k, nullptr, kbeg, k0, kend, alignedA, tid);
        load_tile_gather<BN, B_KC, NT>(sB + st * BN * BK, gsB, gg.b_k, nullptr, kbeg, k0, kend, alignedB, tid);
        if (weighted && tid < BK) {
          const int k = k0 + tid;
          double w = 0.0;
          if (k < kend) {
            const uint32_t q0 = fd_div((uint32_t)k, gg.wE[0]), d0 = (uint32_t)k - q0 * gg.wE[0].d;
            const uint32_t q1 = fd_div(q0, gg.wE[1]), d1 = q0 - q1 * gg.wE[1].d;
            w = sV[d0] * sV[GW_MAXLEN + d1] * sV[2 * GW_MAXLEN + q1];
          }
          sW[st * BK + tid] = w;
        }
      } else {
        load_tile<BM, A_KC, NT>(sA + st * BM * BK, p.A, p.lda, m0, M, k0, kend, alignedA, tid);
        load_tile<BN, B_KC, NT>(sB + st * BN * BK, p.B, p.ldb, n0, N, k0, kend, alignedB, tid);
      }
    }
    cp_async_commit();
  };
#pragma unroll
  for (int s = 0; s < STAGES - 1; s++) issue(s, s);

  // the ring position of a stage is a compile-time constant in each of the STAGES unrolled copies of the body
  for (int it0 = 0; it0 < nk; it0 += STAGES) {
#pragma unroll
   for (int sidx = 0; sidx < STAGES; sidx++) {
    const int it = it0 + sidx;
    if (it >= nk) break;
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    issue(it + STAGES - 1, (sidx + STAGES - 1) % STAGES);
    const double* a_s = sA + sidx * BM * BK;
    const double* b_s = sB + sidx * BN * BK;
    const double* w_s = sW + sidx * BK;
    if (!skip_warp) {
#pragma unroll
      for (int kk = 0; kk < BK; kk += 4) {
        double af[MI], bf[NI];
#pragma unroll
        for (int i = 0; i < MI; i++) {
          int m = wm0 + i * 8 + g;
          if (A_KC) af[i] = a_s[m * 16 + ((kk + t) ^ (4 * (m & 3)))];
          else      af[i] = a_s[(kk + t) * BM + (m ^ (4 * t))];
        }
        if (weighted) {                      // a3 fused: row weight lambda_env of this k
          const double w = w_s[kk + t];
#pragma unroll
          for (int i = 0; i < MI; i++) af[i] *= w;
        }
#pragma unroll
        for (int j = 0; j < NI; j++) {
          int n = wn0 + j * 8 + g;
          if (B_KC) bf[j] = b_s[n * 16 + ((kk + t) ^ (4 * (n & 3)))];
          else      bf[j] = b_s[(kk + t) * BN + (n ^ (4 * t))];
        }
#pragma unroll
        for (int i = 0; i < MI; i++)
#pragma unroll
          for (int j = 0; j < NI; j++) dmma8x8x4(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
      }
    }
   }
  }
  cp_async_wait<0>();

  if (skip_warp) return;
  double* Cb = p.C;
  long long ldc = p.ldc;
  if (ksplit > 1) { Cb = part + (long long)split * M * N; ldc = M; }
  const bool gout = GATHER && ksplit <= 1;
  long long on[NI][2];
#pragma unroll
  for (int j = 0; j < NI; j++) {
    const int n = n0 + wn0 + j * 8 + 2 * t;
    on[j][0] = (gout && n < N) ? idx2_off(gg.c_n, (uint32_t)n) : (long long)n * ldc;
    on[j][1] = (gout && n + 1 < N) ? idx2_off(gg.c_n, (uint32_t)(n + 1)) : (long long)(n + 1) * ldc;
  }
#pragma unroll
  for (int i = 0; i < MI; i++) {
    long long m = m0 + wm0 + i * 8 + g;
    if (m >= M) continue;
    const long long om = gout ? idx2_off(gg.c_m, (uint32_t)m) : m;
#pragma unroll
    for (int j = 0; j < NI; j++) {
      int n = n0 + wn0 + j * 8 + 2 * t;
      if (n < N) Cb[om + on[j][0]] = acc[i][j][0];
      if (n + 1 < N) Cb[om + on[j][1]] = acc[i][j][1];
    }
  }
}

// fp64 tensor-pipe yardstick: every warp issues `iters` x 16 register-only DMMA.8x8x4 on 8 independent
// accumulator pairs (no memory traffic).  flops = CTAs x warps x iters x 16 x 512.
__global__ void __launch_bounds__(256) dmma_peak_kernel(int iters, double* sink) {
  double acc[8][2];
#pragma unroll
  for (int i = 0; i < 8; i++) { acc[i][0] = 0.0; acc[i][1] = 0.0; }
  double a = 1.0 + 1e-9 * threadIdx.x, b = 1.0 - 1e-9 * threadIdx.x;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int r = 0; r < 2; r++)
#pragma unroll
      for (int i = 0; i < 8; i++) dmma8x8x4(acc[i][0], acc[i][1], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 8; i++) s += acc[i][0] + acc[i][1];
  if (s == 12345.678) sink[0] = s;                 // keeps the loop alive; never true in practice
}

__global__ void gram_reduce_kernel(const double* part, int ksplit, int n, double* C,
                                   long long ldc) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  int j = blockIdx.y;
  if (i >= n || i > j) return;
  double s = 0.0;
  for (int k = 0; k < ksplit; k++) s += part[(long long)k * n * n + i + (long long)j * n];
  C[i + (long long)j * ldc] = s;
  C[j + (long long)i * ldc] = s;
}

template <int TA, int TB, int BM, int BN, int WM, int WN, int STAGES, bool GATHER = false>
int launch_cfg(cudaStream_t st, const GemmProb& p, const GemmProb* probs, int gz, long long maxM,
               int maxN, int ksplit, int kchunk, double* part, bool upper_only,
               const GemmGather* gg = nullptr) {
  constexpr int NT = (BM / WM) * (BN / WN) * 32;
  size_t smem = (size_t)STAGES * (BM + BN) * BK * sizeof(double);
  // row weights (weighted Gram only): the extra shared memory must not cost a resident CTA elsewhere
  if (GATHER && gg && gg->nw > 0) smem += (size_t)(STAGES * BK + 3 * GW_MAXLEN) * sizeof(double);
  else if (GATHER && gg && gg->ktabA) smem += (size_t)((p.K + 1) & ~1) * sizeof(long long);
  // all-aligned flavour: same tests as the kernel's, made here (single problem; every split starts at an even k)
  bool al = !probs && (ksplit <= 1 || (kchunk & 1) == 0);
  if (al) {
    if (GATHER) al = gg && gg->alignedA != 0 && gg->alignedB != 0;
    else al = (((uintptr_t)p.A & 15) == 0) && ((p.lda & 1) == 0) && (((uintptr_t)p.B & 15) == 0) && ((p.ldb & 1) == 0);
  }
  const bool wg = GATHER && gg && gg->nw > 0;
  auto kern = dgemm_dmma_kernel<TA, TB, BM, BN, WM, WN, STAGES, GATHER, false, false>;
  if (GATHER && wg) kern = al ? dgemm_dmma_kernel<TA, TB, BM, BN, WM, WN, STAGES, GATHER, true, GATHER>
                              : dgemm_dmma_kernel<TA, TB, BM, BN, WM, WN, STAGES, GATHER, false, GATHER>;
  else if (al) kern = dgemm_dmma_kernel<TA, TB, BM, BN, WM, WN, STAGES, GATHER, true, false>;
  static char attr_set[PEPO_MAX_DEVICES] = {0};
  if (first_use_on_device(attr_set)) {
    const size_t smem_max = (size_t)STAGES * (BM + BN) * BK * sizeof(double) +
                            (GATHER ? (size_t)(STAGES * BK + 3 * GW_MAXLEN) * sizeof(double) : 0);
    PEPO_CUDA_OK(cudaFuncSetAttribute(dgemm_dmma_kernel<TA, TB, BM, BN, WM, WN, STAGES, GATHER, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max));
    PEPO_CUDA_OK(cudaFuncSetAttribute(dgemm_dmma_kernel<TA, TB, BM, BN, WM, WN, STAGES, GATHER, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max));
    PEPO_CUDA_OK(cudaFuncSetAttribute(dgemm_dmma_kernel<TA, TB, BM, BN, WM, WN, STAGES, GATHER, true, GATHER>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max));
    PEPO_CUDA_OK(cudaFuncSetAttribute(dgemm_dmma_kernel<TA, TB, BM, BN, WM, WN, STAGES, GATHER, false, GATHER>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max));
  }
  long long tiles = ((maxM + BM - 1) / BM) * ((maxN + BN - 1) / BN);
  if (tiles <= 0 || gz <= 0) return 0;
  dim3 grid((unsigned)tiles, 1, (unsigned)gz);
  GemmGather g0;
  if (gg) g0 = *gg; else memset(&g0, 0, sizeof(g0));
  kern<<<grid, NT, smem, st>>>(p, probs, ksplit, kchunk, part, upper_only ? 1 : 0, g0);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

template <int BM, int BN, int WM, int WN, int STAGES>
int launch_trans(cudaStream_t st, int ta, int tb, const GemmProb& p, const GemmProb* probs, int gz,
                 long long maxM, int maxN, int ksplit, int kchunk, double* part, bool upper) {
  if (ta == 0 && tb == 0) return launch_cfg<0, 0, BM, BN, WM, WN, STAGES>(st, p, probs, gz, maxM, maxN, ksplit, kchunk, part, upper);
  if (ta == 1 && tb == 0) return launch_cfg<1, 0, BM, BN, WM, WN, STAGES>(st, p, probs, gz, maxM, maxN, ksplit, kchunk, part, upper);
  if (ta == 0 && tb == 1) return launch_cfg<0, 1, BM, BN, WM, WN, STAGES>(st, p, probs, gz, maxM, maxN, ksplit, kchunk, part, upper);
  return launch_cfg<1, 1, BM, BN, WM, WN, STAGES>(st, p, probs, gz, maxM, maxN, ksplit, kchunk, part, upper);
}

}  // namespace

// Tile shapes (measured on B200, 216000 x 240 x 240 and 256000 x 160 x 160): two or three
// resident CTAs per SM matter more than a large tile, because the k loop of these products is
// short (K = n = 4 chi for the reconstruction GEMM) and one CTA's epilogue must overlap another's
// main loop; tiles that divide n exactly (80 | 4 chi for chi = 20, 40, 60, 100) waste no DMMA.
enum TileCfg { T_64x64, T_128x128, T_128x64, T_64x80, T_80x80 };

static TileCfg pick_tile(long long M, int N, int ksplit, bool upper_only) {
  const long long tiles128 = ((M + 127) / 128) * ((N + 127) / 128) * ksplit;
  if (upper_only) {
    if (M == N && N % 80 == 0) return T_80x80;
    return (tiles128 >= 120 && N > 64) ? T_128x128 : T_64x64;
  }
  if (tiles128 < 120 || N <= 64) return T_64x64;
  if (N % 80 == 0) return T_64x80;
  return T_128x64;
}

int launch_dgemm(cudaStream_t st, int transA, int transB, const GemmProb& p, int ksplit,
                 int kchunk, double* part, bool upper_only) {
  if (p.M <= 0 || p.N <= 0) return 0;
  if (ksplit < 1) ksplit = 1;
  switch (pick_tile(p.M, p.N, ksplit, upper_only)) {
    case T_80x80:
      return launch_trans<80, 80, 40, 40, 4>(st, transA, transB, p, nullptr, ksplit, p.M, p.N, ksplit, kchunk, part, upper_only);
    case T_64x80:
      return launch_trans<64, 80, 32, 40, 4>(st, transA, transB, p, nullptr, ksplit, p.M, p.N, ksplit, kchunk, part, upper_only);
    case T_128x64:
      return launch_trans<128, 64, 32, 32, 4>(st, transA, transB, p, nullptr, ksplit, p.M, p.N, ksplit, kchunk, part, upper_only);
    case T_128x128:
      return launch_trans<128, 128, 64, 32, 4>(st, transA, transB, p, nullptr, ksplit, p.M, p.N, ksplit, kchunk, part, upper_only);
    default:
      return launch_trans<64, 64, 32, 32, 4>(st, transA, transB, p, nullptr, ksplit, p.M, p.N, ksplit, kchunk, part, upper_only);
  }
}

// Gathered variant (GemmGather): the tile shapes the bond gate uses.  transA/transB as launch_dgemm
// (they select which operand index is the contiguous one); lda / ldb / ldc of p are ignored.
int launch_dgemm_gather(cudaStream_t st, int transA, int transB, const GemmProb& p, const GemmGather& g,
                        int ksplit, int kchunk, double* part, bool upper_only) {
  if (p.M <= 0 || p.N <= 0) return 0;
  if (ksplit < 1) ksplit = 1;
  TileCfg tc = pick_tile(p.M, p.N, ksplit, upper_only);
  // short M (the swapped reconstruction, M = 4 chi_new): a tile that divides it wastes no DMMA
  if (!upper_only && tc == T_64x80 && p.M % 80 == 0 && p.M <= 1024) tc = T_80x80;
#define PEPO_GATHER_CASE(TA_, TB_)                                                                              \
  switch (tc) {                                                                                                 \
    case T_80x80: return launch_cfg<TA_, TB_, 80, 80, 40, 40, 4, true>(st, p, nullptr, ksplit, p.M, p.N, ksplit, kchunk, part, upper_only, &g);   \
    case T_64x80: return launch_cfg<TA_, TB_, 64, 80, 32, 40, 4, true>(st, p, nullptr, ksplit, p.M, p.N, ksplit, kchunk, part, upper_only, &g);   \
    case T_128x64: return launch_cfg<TA_, TB_, 128, 64, 32, 32, 4, true>(st, p, nullptr, ksplit, p.M, p.N, ksplit, kchunk, part, upper_only, &g); \
    case T_128x128: return launch_cfg<TA_, TB_, 128, 128, 64, 32, 4, true>(st, p, nullptr, ksplit, p.M, p.N, ksplit, kchunk, part, upper_only, &g); \
    default: return launch_cfg<TA_, TB_, 64, 64, 32, 32, 4, true>(st, p, nullptr, ksplit, p.M, p.N, ksplit, kchunk, part, upper_only, &g);         \
  }
  if (transA == 1 && transB == 0) { PEPO_GATHER_CASE(1, 0) }
  if (transA == 0 && transB == 1) { PEPO_GATHER_CASE(0, 1) }
  if (transA == 0 && transB == 0) { PEPO_GATHER_CASE(0, 0) }
#undef PEPO_GATHER_CASE
  set_error("dgemm_gather: unsupported operand layout");
  return -1;
}

static void site_geometry(const SiteView& v, long long& run, long long& slab) {
  run = 1; slab = 1;
  for (int l = 0; l < v.cut; l++) run *= v.dims[l];
  for (int l = 0; l < v.nlegs; l++) slab *= v.dims[l];
}

int launch_site_gram(cudaStream_t st, const double* psi, const SiteView& v, const double* const* w2,
                     double* C, double* part, const double* psiB) {
  long long run, slab;
  site_geometry(v, run, slab);
  const long long m = v.m();
  const int n = v.n(), chic = v.dims[v.cut];
  GemmGather g; memset(&g, 0, sizeof(g));
  const Idx2 col = make_idx2(chic, run, slab);                 // (c, p) -> c * run + p * slab
  // contiguous run of the legs before the cut, then the rest (run = 1: plain stride chi_c)
  const Idx2 row = run >= 2 ? make_idx2(run, 1, run * chic) : make_idx2(0, chic, 0);
  g.a_outer = col; g.b_outer = col; g.a_k = row; g.b_k = row;
  g.c_m = make_idx2(0, 1, 0); g.c_n = make_idx2(0, n, 0);      // plain n x n output (single split)
  g.nw = 0;
  int ext[3] = {1, 1, 1};
  for (int l = 0; l < v.nlegs; l++) {
    if (l == v.cut) continue;
    g.wv[g.nw] = w2 ? w2[l] : nullptr; g.wlen[g.nw] = v.dims[l]; ext[g.nw] = v.dims[l]; g.nw++;
  }
  bool any = false;
  for (int i = 0; i < g.nw; i++) any |= (g.wv[i] != nullptr);
  if (!any) g.nw = 0;
  else for (int i = 0; i < g.nw; i++) if (!g.wv[i]) { set_error("site_gram: weights must be given for all environment legs or none"); return -1; }
  g.wE[0] = make_fastdiv((uint32_t)ext[0]); g.wE[1] = make_fastdiv((uint32_t)ext[1]);
  for (int i = 0; i < 3; i++) if (ext[i] > GW_MAXLEN) { set_error("site_gram: bond dimension %d > %d", ext[i], GW_MAXLEN); return -1; }
  const bool base16 = ((((uintptr_t)psi) & 15) == 0) && (!psiB || (((uintptr_t)psiB) & 15) == 0);
  int ks, kc;
  gram_plan(m, n, &ks, &kc);
  GemmProb p; p.A = psi; p.B = psiB ? psiB : psi; p.C = C; p.lda = p.ldb = 0; p.ldc = n; p.M = n; p.N = n; p.K = (int)m;
  int rc;
  if (run >= 2) {
    // rows contiguous in runs: both operands K-contiguous (the layout of the explicit cv)
    g.alignedA = g.alignedB = base16 && (run % 2 == 0) && (slab % 2 == 0);
    rc = launch_dgemm_gather(st, 1, 0, p, g, ks, kc, part, true);
  } else {
    // the cut leg is the fastest one: columns contiguous, rows strided
    g.alignedA = g.alignedB = base16 && (chic % 2 == 0) && (slab % 2 == 0);
    rc = launch_dgemm_gather(st, 0, 1, p, g, ks, kc, part, true);
  }
  if (rc) return rc;
  return launch_gram_reduce(st, ks > 1 ? part : C, ks > 1 ? ks : 1, n, C, n);
}

int launch_site_apply(cudaStream_t st, const double* psi, const SiteView& v, const double* W, long long ldw,
                      int chi_new, double* out) {
  long long run, slab;
  site_geometry(v, run, slab);
  const long long m = v.m();
  const int n = v.n(), chic = v.dims[v.cut];
  const long long slab_new = slab / chic * chi_new;
  GemmGather g; memset(&g, 0, sizeof(g));
  const Idx2 col = make_idx2(chic, run, slab), row = make_idx2(run, 1, run * chic);
  const Idx2 col_new = make_idx2(chi_new, run, slab_new), row_new = make_idx2(run, 1, run * chi_new);
  const bool base16 = (((uintptr_t)psi) & 15) == 0, w16 = ((((uintptr_t)W) & 15) == 0) && (ldw % 2 == 0);
  GemmProb p; p.lda = p.ldb = p.ldc = 0;
  if (run >= 2) {
    // out (m x 4 chi_new) = cv (m x n) W: rows contiguous in runs on both sides
    p.A = psi; p.B = W; p.C = out; p.M = m; p.N = 4 * chi_new; p.K = n;
    g.a_outer = row; g.a_k = col;
    g.b_outer = make_idx2(0, ldw, 0); g.b_k = make_idx2(0, 1, 0);
    g.c_m = row_new; g.c_n = col_new;
    g.alignedA = base16 && (run % 2 == 0) && (slab % 2 == 0);
    g.alignedB = w16;
    g.ktabA = (n <= 768) ? 1 : 0;            // two-level k offsets of psi from a per-CTA table (6 KB at most)
    return launch_dgemm_gather(st, 0, 0, p, g, 1, 0, nullptr, false);
  }
  // cut leg fastest: out^T (4 chi_new x m) = W^T cv^T, so that both psi and out move along their
  // contiguous direction (the cut index)
  p.A = W; p.B = psi; p.C = out; p.M = 4 * chi_new; p.N = (int)m; p.K = n;
  if (m > 0x7fffffffll) { set_error("site_apply: too many rows"); return -1; }
  g.a_outer = make_idx2(0, ldw, 0); g.a_k = make_idx2(0, 1, 0);
  g.b_outer = make_idx2(0, chic, 0); g.b_k = make_idx2(chic, 1, slab);
  g.c_m = make_idx2(chi_new, 1, slab_new); g.c_n = make_idx2(0, chi_new, 0);
  g.alignedA = w16;
  g.alignedB = base16 && (chic % 2 == 0) && (slab % 2 == 0);
  return launch_dgemm_gather(st, 1, 0, p, g, 1, 0, nullptr, false);
}

int launch_dmma_peak(cudaStream_t st, int iters, int ctas_per_sm, double* sink, double* flops) {
  if (iters < 1 || ctas_per_sm < 1 || ctas_per_sm > 8) { set_error("dmma_peak: bad argument"); return -1; }
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int ctas = sms * ctas_per_sm;
  dmma_peak_kernel<<<ctas, 256, 0, st>>>(iters, sink);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  if (flops) *flops = (double)ctas * 8.0 * iters * 16.0 * 512.0;
  return 0;
}

int launch_dgemm_batched(cudaStream_t st, int transA, int transB, const GemmProb* probs_dev,
                         int batch, long long max_M, int max_N) {
  GemmProb dummy{};
  return launch_trans<64, 64, 32, 32, 4>(st, transA, transB, dummy, probs_dev, batch, max_M, max_N, 1, 0, nullptr, false);
}

constexpr int GRAM_WAVES = 2;      // waves of resident CTAs of the 80x80 Gram kernel (1 and 2 measured equal, 3+ slower)

// Upper bound of gram_plan's split count over every row count <= m: the count before the chunk is rounded
// up to 16 rows.  (The rounded count is NOT monotone in m - 62400 rows give 195 splits of 320, 64000 rows
// 191 of 336 - so a workspace shared by all sites of a run is sized with this bound, not with gram_plan
// of the largest m.)
int gram_max_splits(long long m, int n) {
  int ks, kc;
  gram_plan(m, n, &ks, &kc);
  long long best = ks;
  // ks = ceil(m' / kc) <= the unrounded count, which grows with m' through the 256-rows-per-split rule only
  int bt = 128, target = 148 * 2, cap = 128; bool whole = false;
  if (n % 80 == 0) { bt = 80; target = 148 * 2 * GRAM_WAVES; cap = 100 * GRAM_WAVES; whole = true; }
  else if (n <= 64) { bt = 64; target = 148 * 4; cap = 1024; }
  const int tn = (n + bt - 1) / bt, upper = tn * (tn + 1) / 2;
  long long k0 = whole ? std::max(1, target / upper) : (target + upper - 1) / upper;
  k0 = std::min<long long>(k0, (m + 255) / 256);
  k0 = std::max<long long>(1, std::min<long long>(k0, cap));
  return (int)std::max(best, k0);
}

void gram_plan(long long m, int n, int* ksplit, int* kchunk) {
  // upper-triangle tiles at the tile size launch_dgemm will pick (the choice between the 128 and
  // 64 tiles depends on ksplit itself: plan with the 128 tile first, as before)
  int bt = 128, target = 148 * 2, cap = 128;
  bool whole_waves = false;
  if (n % 80 == 0) {
    // 80x80 tile kernel: 197 registers x 128 threads -> 2 resident CTAs per SM = 296 slots.  The
    // working CTAs (upper tiles x splits) must fill a whole number of waves: 99 splits x 6 tiles =
    // 594 CTAs ran as two waves plus a third one of 2 CTAs (ncu: 558 us against 2/3 of that).
    bt = 80; target = 148 * 2 * GRAM_WAVES; cap = 100 * GRAM_WAVES; whole_waves = true;
  }
  else if (n <= 64) {
    // one tile: the product is HBM-bound (5 - 10 flop / byte): enough splits for 4 resident CTAs per SM
    // (128 splits streamed 256000 x 40 at 0.64 TB/s)
    bt = 64; target = 148 * 4; cap = 1024;
  }
  const int tn = (n + bt - 1) / bt;
  const int upper = tn * (tn + 1) / 2;
  int ks = whole_waves ? std::max(1, target / upper) : (target + upper - 1) / upper;
  long long maxsplit = (m + 255) / 256;             // at least 256 rows per split
  if (ks > maxsplit) ks = (int)maxsplit;
  if (ks > cap) ks = cap;
  if (ks < 1) ks = 1;
  long long kc = (m + ks - 1) / ks;
  kc = (kc + 15) / 16 * 16;
  ks = (int)((m + kc - 1) / kc);
  *ksplit = ks;
  *kchunk = (int)kc;
}

int launch_gram_reduce(cudaStream_t st, const double* part, int ksplit, int n, double* C,
                       long long ldc) {
  dim3 grid((n + 127) / 128, n);
  gram_reduce_kernel<<<grid, 128, 0, st>>>(part, ksplit, n, C, ldc);
  PEPO_COUNT_LAUNCH();
  PEPO_CUDA_OK(cudaGetLastError());
  return 0;
}

}  // namespace pepo
