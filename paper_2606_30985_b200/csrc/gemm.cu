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

template <int TA, int TB, int BM, int BN, int WM, int WN, int STAGES>
__global__ void __launch_bounds__((BM / WM) * (BN / WN) * 32)
dgemm_dmma_kernel(GemmProb p0, const GemmProb* __restrict__ probs, int ksplit, int kchunk,
                  double* __restrict__ part, int upper_only) {
  constexpr int NT = (BM / WM) * (BN / WN) * 32;
  constexpr int MI = WM / 8, NI = WN / 8;
  constexpr bool A_KC = (TA == 1), B_KC = (TB == 0);
  extern __shared__ __align__(16) double smem[];
  double* sA = smem;                       // STAGES * BM*16
  double* sB = smem + STAGES * BM * BK;    // STAGES * BN*16

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

  const bool alignedA = (((uintptr_t)p.A & 15) == 0) && ((p.lda & 1) == 0) && ((kbeg & 1) == 0);
  const bool alignedB = (((uintptr_t)p.B & 15) == 0) && ((p.ldb & 1) == 0) && ((kbeg & 1) == 0);

  // Gram (upper_only) diagonal tiles: a warp tile strictly below the diagonal is never read by the
  // reducer, so its warp only helps with the loads (frees its DMMA issue slots for co-resident CTAs)
  const bool skip_warp = upper_only && tn == tm && BM == BN && (wm0 >= wn0 + WN);
  double acc[MI][NI][2];
#pragma unroll
  for (int i = 0; i < MI; i++)
#pragma unroll
    for (int j = 0; j < NI; j++) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }

  const int nk = (kend - kbeg + BK - 1) / BK;
  auto issue = [&](int it) {
    if (it < nk) {
      int st = it % STAGES;
      int k0 = kbeg + it * BK;
      load_tile<BM, A_KC, NT>(sA + st * BM * BK, p.A, p.lda, m0, M, k0, kend, alignedA, tid);
      load_tile<BN, B_KC, NT>(sB + st * BN * BK, p.B, p.ldb, n0, N, k0, kend, alignedB, tid);
    }
    cp_async_commit();
  };
#pragma unroll
  for (int s = 0; s < STAGES - 1; s++) issue(s);

  for (int it = 0; it < nk; it++) {
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    issue(it + STAGES - 1);
    const double* a_s = sA + (it % STAGES) * BM * BK;
    const double* b_s = sB + (it % STAGES) * BN * BK;
    if (skip_warp) continue;
#pragma unroll
    for (int kk = 0; kk < BK; kk += 4) {
      double af[MI], bf[NI];
#pragma unroll
      for (int i = 0; i < MI; i++) {
        int m = wm0 + i * 8 + g;
        if (A_KC) af[i] = a_s[m * 16 + ((kk + t) ^ (4 * (m & 3)))];
        else      af[i] = a_s[(kk + t) * BM + (m ^ (4 * t))];
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
  cp_async_wait<0>();

  if (skip_warp) return;
  double* Cb = p.C;
  long long ldc = p.ldc;
  if (ksplit > 1) { Cb = part + (long long)split * M * N; ldc = M; }
#pragma unroll
  for (int i = 0; i < MI; i++) {
    long long m = m0 + wm0 + i * 8 + g;
    if (m >= M) continue;
#pragma unroll
    for (int j = 0; j < NI; j++) {
      int n = n0 + wn0 + j * 8 + 2 * t;
      if (n < N) Cb[m + (long long)n * ldc] = acc[i][j][0];
      if (n + 1 < N) Cb[m + (long long)(n + 1) * ldc] = acc[i][j][1];
    }
  }
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

template <int TA, int TB, int BM, int BN, int WM, int WN, int STAGES>
int launch_cfg(cudaStream_t st, const GemmProb& p, const GemmProb* probs, int gz, long long maxM,
               int maxN, int ksplit, int kchunk, double* part, bool upper_only) {
  constexpr int NT = (BM / WM) * (BN / WN) * 32;
  size_t smem = (size_t)STAGES * (BM + BN) * BK * sizeof(double);
  auto kern = dgemm_dmma_kernel<TA, TB, BM, BN, WM, WN, STAGES>;
  static char attr_set[PEPO_MAX_DEVICES] = {0};
  if (first_use_on_device(attr_set))
    PEPO_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  long long tiles = ((maxM + BM - 1) / BM) * ((maxN + BN - 1) / BN);
  if (tiles <= 0 || gz <= 0) return 0;
  dim3 grid((unsigned)tiles, 1, (unsigned)gz);
  kern<<<grid, NT, smem, st>>>(p, probs, ksplit, kchunk, part, upper_only ? 1 : 0);
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

int launch_dgemm_batched(cudaStream_t st, int transA, int transB, const GemmProb* probs_dev,
                         int batch, long long max_M, int max_N) {
  GemmProb dummy{};
  return launch_trans<64, 64, 32, 32, 4>(st, transA, transB, dummy, probs_dev, batch, max_M, max_N, 1, 0, nullptr, false);
}

constexpr int GRAM_WAVES = 2;      // waves of resident CTAs of the 80x80 Gram kernel (1 and 2 measured equal, 3+ slower)

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
  else if (n <= 64) bt = 64;
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
