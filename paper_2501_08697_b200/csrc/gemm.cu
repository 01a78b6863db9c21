// gemm.cu -- complex FP64 GEMMs on the FP64 tensor path (mma.sync m8n8k4 f64 -> SASS DMMA.8x8x4,
// the only FP64 MMA shape sm_100a has; tcgen05 has no f64 kind).
//
//   ks_gemm_hn:  C[M x N] = A^H B   A: K x M, B: K x N column-major, K (= npw) long and contiguous.
//                Used for beta^H psi (H6), V^H W (D2), V^H T and T^H T (D0, D7).  Split-K over CTAs with a
//                fixed-order second-pass reduction (deterministic, no atomics).
//   ks_gemm_nn:  C[M x N] (+)= A B  A: M x K, C: M x N column-major, M (= npw) long and contiguous.
//                Used for hpsi += beta (D B) (H8), X = V C, HX = W C (D4), T -= V (V^H T) (D7).
//
// The N-tile width is a template parameter (NJ = 1..5 MMA tiles per warp) picked per call for the least padding of N;
// N <= 4 takes matrix-vector kernels instead (k_gemv_hn / k_gemv_nn: A is read once at memory speed).
//
// A complex product is four real DMMAs on split re/im fragments:
//   C_re += A_re B_re - A_im B_im ,  C_im += A_re B_im + A_im B_re     (signs folded into one negated
// fragment; for A^H the imaginary part of A is negated instead).
// Fragment layout of mma.m8n8k4.row.col.f64: lane l holds A[l>>2][l&3], B[l&3][l>>2],
// C[l>>2][2*(l&3)+{0,1}].  Tiles are staged in shared memory by cp.async (16 B = one complex) in a
// 3-stage ring; leading dimensions are padded so a quarter-warp's 16-byte loads hit distinct banks.
#include "mma.cuh"
#include "plan.h"
#include <algorithm>
#include <atomic>
#include <cstdlib>

#define GEMM_THREADS 256
#ifndef KS_EARLY
#define KS_EARLY 8      // k-step (0, 4, 8, 12) before which warps 0..3 / 4..7 issue their cp.async of the stage after next
#endif
#ifndef KS_LATE
#define KS_LATE 4
#endif
#define GEMM_STAGES 3
#define KT 16          // complex K elements per stage
#define LDK (KT + 4)   // "k-contiguous" tile leading dimension: == 4 (mod 8) -> conflict-free fragment loads

// ------------------------------------------------------------------------------------------------
// C = A^H B.  CTA tile 64 x 32*NJ, 8 warps as 2 (M) x 4 (N), warp tile 32 x 8*NJ -> 4 x NJ MMA tiles.
// NJ in 1..5 is picked per call so that N is covered with the least padding (N = 160 -> one 160-wide tile,
// N = 5 unconverged bands -> a 32-wide tile instead of 64).
// ------------------------------------------------------------------------------------------------
#define HN_MT 64

// one CTA tile of C = A^H B over the K range [kbeg, kend): the partial tile goes to out (column-major M x N)
// WN = warps along N (WM = 8 / WN along M): WN = 4 is the wide tile above; WN = 1 gives an N-tile of 8*NJ columns (8 .. 40)
// with 8-row warp tiles, for narrow products and for the ragged remainder of a wide one (N = 520 = 3 x 160 + 40: the 40
// columns cost 40/480 of the main launch instead of a padded 64-wide tile, cfg 3: 3.31 -> 2.0 ms).
template <int NJ, int WN = 4>
__device__ __forceinline__ void gemm_hn_tile(int M, int N, const cplx* __restrict__ A, long lda, const cplx* __restrict__ B,
                                             long ldb, cplx* __restrict__ out, int m0, int n0, int kbeg, int kend) {
  constexpr int WM = 8 / WN, MI = HN_MT / (8 * WM), HN_NT = 8 * NJ * WN;
  extern __shared__ cplx sm[];
  cplx* sA = sm;                                     // [stage][HN_MT][LDK]
  cplx* sB = sm + GEMM_STAGES * HN_MT * LDK;         // [stage][HN_NT][LDK]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp % WM, wn = warp / WM;
  const int ntile = (kend - kbeg + KT - 1) / KT;

  auto load_stage = [&](int st, int kt) {
    const int k0 = kbeg + kt * KT;
    // 64 columns x 16 k per operand = 1024 elements each; 256 threads -> 4 + 4 per thread
#pragma unroll
    for (int r = 0; r < (HN_MT * KT) / GEMM_THREADS; ++r) {
      const int e = tid + r * GEMM_THREADS, col = e / KT, kk = e % KT;
      const bool ok = (m0 + col < M) && (k0 + kk < kend);
      cp16(&sA[(st * HN_MT + col) * LDK + kk], ok ? &A[(long)(m0 + col) * lda + k0 + kk] : A, ok);
    }
#pragma unroll
    for (int r = 0; r < (HN_NT * KT + GEMM_THREADS - 1) / GEMM_THREADS; ++r) {
      const int e = tid + r * GEMM_THREADS, col = e / KT, kk = e % KT;
      if ((HN_NT * KT) % GEMM_THREADS != 0 && e >= HN_NT * KT) break;
      const bool ok = (n0 + col < N) && (k0 + kk < kend);
      cp16(&sB[(st * HN_NT + col) * LDK + kk], ok ? &B[(long)(n0 + col) * ldb + k0 + kk] : B, ok);
    }
  };

  double cre[MI][NJ][2], cim[MI][NJ][2];
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int j = 0; j < NJ; ++j) cre[i][j][0] = cre[i][j][1] = cim[i][j][0] = cim[i][j][1] = 0.0;

  for (int s = 0; s < GEMM_STAGES - 1; ++s) {
    if (s < ntile) load_stage(s, s);
    cp_commit();
  }
  const int fr = lane >> 2, fk = lane & 3;
  // The two warps of an SM sub-partition (w, w + 4) leave the barrier together.  If both then spend ~130 instructions on
  // the addresses and cp.async of the stage after next, the DMMA pipe of that sub-partition idles for that long at every
  // k-tile (ncu, cfg 3: pipe 87 % active inside a CTA).  So warps 4..7 start their DMMAs at once and issue their share of the
  // loads after the first k-step, when warps 0..3 are computing: one warp alone keeps the pipe full (ks_dmma_latency).
#ifdef KSPW_GEMM_NO_STAGGER
  const bool late = false;
#else
  const bool late = warp >= 4;
#endif
  for (int kt = 0; kt < ntile; ++kt) {
    cp_wait<GEMM_STAGES - 2>();
    __syncthreads();
    const bool more = kt + GEMM_STAGES - 1 < ntile;
#ifdef KSPW_GEMM_NO_STAGGER
    if (more) load_stage((kt + GEMM_STAGES - 1) % GEMM_STAGES, kt + GEMM_STAGES - 1);
    cp_commit();
#endif
    const cplx* a = sA + ((kt % GEMM_STAGES) * HN_MT + wm * 8 * MI) * LDK;
    const cplx* b = sB + ((kt % GEMM_STAGES) * HN_NT + wn * 8 * NJ) * LDK;
#pragma unroll
    for (int ks = 0; ks < KT; ks += 4) {
#ifndef KSPW_GEMM_NO_STAGGER
      if (ks == (late ? KS_LATE : KS_EARLY)) {
        if (more) load_stage((kt + GEMM_STAGES - 1) % GEMM_STAGES, kt + GEMM_STAGES - 1);
        cp_commit();
      }
#endif
      cplx af[MI], bf[NJ];
#pragma unroll
      for (int i = 0; i < MI; ++i) af[i] = a[(i * 8 + fr) * LDK + ks + fk];
#pragma unroll
      for (int j = 0; j < NJ; ++j) bf[j] = b[(j * 8 + fr) * LDK + ks + fk];
      // conj(a) b = (ar br + ai bi) + i (ar bi - ai br).  The two products of one accumulator are two DMMAs apart: enough,
      // the DMMA result latency is 27 clk against an issue interval of 16 (ks_dmma_latency); spreading them 8 NJ apart
      // measured no difference (cfg 3: 30.24 vs 30.29 ms)
#pragma unroll
      for (int i = 0; i < MI; ++i) {
        const double nai = -af[i].y;
#pragma unroll
        for (int j = 0; j < NJ; ++j) {
          dmma(cre[i][j][0], cre[i][j][1], af[i].x, bf[j].x);
          dmma(cim[i][j][0], cim[i][j][1], af[i].x, bf[j].y);
          dmma(cre[i][j][0], cre[i][j][1], af[i].y, bf[j].y);
          dmma(cim[i][j][0], cim[i][j][1], nai, bf[j].x);
        }
      }
    }
  }
  cp_wait<0>();
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int j = 0; j < NJ; ++j)
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int m = m0 + wm * 8 * MI + i * 8 + fr, n = n0 + wn * 8 * NJ + j * 8 + 2 * fk + h;
        if (m < M && n < N) out[(size_t)n * M + m] = cmake(cre[i][j][h], cim[i][j][h]);
      }
}

template <int NJ, int WN = 4>
__global__ void __launch_bounds__(GEMM_THREADS) k_gemm_hn(int M, int N, int K, const cplx* __restrict__ A, long lda,
                                                          const cplx* __restrict__ B, long ldb, cplx* __restrict__ part,
                                                          int kchunk, int herm_r0) {
  // Hermitian block (rows herm_r0..): tiles strictly below its diagonal are not computed
  if (herm_r0 >= 0 && (int)(blockIdx.y * HN_MT) - herm_r0 > (int)(blockIdx.x * 8 * NJ * WN + 8 * NJ * WN - 1)) return;
  const int kbeg = blockIdx.z * kchunk;
  // partial tile -> part[z][n][m] (column-major M x N per split)
  gemm_hn_tile<NJ, WN>(M, N, A, lda, B, ldb, part + (size_t)blockIdx.z * M * N, blockIdx.y * HN_MT, blockIdx.x * 8 * NJ * WN, kbeg,
                       min(K, kbeg + kchunk));
}

// Grouped form (ks_hpsi_batch): blockIdx.z = problem * nsplit + split; every problem has its own operands and sizes, the
// grid covers the largest one.  part of problem g: [nsplit][N_g][M_g].
template <int NJ>
__global__ void __launch_bounds__(GEMM_THREADS) k_gemm_hn_g(const GemmProb* __restrict__ probs, int nsplit) {
  const int g = blockIdx.z / nsplit, z = blockIdx.z % nsplit;
  const GemmProb p = probs[g];
  const int m0 = blockIdx.y * HN_MT, n0 = blockIdx.x * 32 * NJ;
  if (m0 >= p.M || n0 >= p.N) return;
  int kchunk = (p.K + nsplit - 1) / nsplit;
  kchunk = (kchunk + KT - 1) / KT * KT;
  const int kbeg = z * kchunk, kend = min(p.K, kbeg + kchunk);
  gemm_hn_tile<NJ>(p.M, p.N, p.A, p.lda, p.B, p.ldb, p.C + (size_t)z * p.M * p.N, m0, n0, kbeg, max(kend, kbeg));
}

__global__ void k_splitk_reduce(int M, int N, int nsplit, const cplx* __restrict__ part, cplx* __restrict__ C, long ldc,
                                int herm_r0 = -1) {
  const long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (i >= (long)M * N) return;
  if (herm_r0 >= 0 && (int)(i % M) - herm_r0 > (int)(i / M)) return;     // strictly below the diagonal of the Hermitian block
  double sr = 0, si = 0;
  for (int z = 0; z < nsplit; ++z) {   // fixed order: deterministic
    const cplx p = part[(size_t)z * M * N + i];
    sr += p.x; si += p.y;
  }
  C[(i / M) * ldc + (i % M)] = cmake(sr, si);
}

// N-tile multiplier with the least padded width (ties: the wider tile)
static int pick_nj(int N, int unit) {
  int best = 1;
  long bestpad = -1;
  for (int nj = 1; nj <= 5; ++nj) {
    const long w = (long)unit * nj, pad = (N + w - 1) / w * w;
    if (bestpad < 0 || pad <= bestpad) { best = nj; bestpad = pad; }
  }
  return best;
}

template <int NJ, int WN = 4>
static int launch_hn(cudaStream_t st, int M, int N, int K, const cplx* A, long lda, const cplx* B, long ldb, cplx* C,
                     long ldc, GemmWs* ws, std::string& err, int herm_r0 = -1) {
  constexpr int HN_NT = 8 * NJ * WN;
  static std::atomic<bool> opted{false};
  const size_t smem = sizeof(cplx) * GEMM_STAGES * (HN_MT + HN_NT) * LDK;
  if (!opted) {
    KS_CUDA_CHECK((cudaFuncSetAttribute(k_gemm_hn<NJ, WN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)), err);
    opted = true;
  }
  const int tm = ceil_div(M, HN_MT), tn = ceil_div(N, HN_NT);
  // split K: the smallest split count that (a) gives every CTA slot (148 SMs x CTAs per SM at this tile's shared
  // memory) about two tiles and (b) wastes less than 7 % of the last wave; each split keeps at least 8 k-tiles.
  // (Measured on cfg 1, 8 output tiles: 148 splits 0.84 ms, 37 splits = exactly two waves 0.78 ms.)
  const int per_sm = std::max(1, (int)((227 * 1024) / (smem + 1024)));
  long tiles = (long)tm * tn;
  if (herm_r0 >= 0) {       // tiles that do work
    tiles = 0;
    for (int y = 0; y < tm; ++y)
      for (int x = 0; x < tn; ++x)
        if (!(y * HN_MT - herm_r0 > x * HN_NT + HN_NT - 1)) ++tiles;
  }
  const long slots = 148L * per_sm;
  // CTAs of one launch take equal time, so they run as lockstep waves of `slots`: take the split count with the fullest
  // last wave among those that give at least two waves and keep >= 48 k-tiles per split (the pipeline prologue and the
  // partial-tile store stay < 1 %).  cfg 3 beta^H psi (81 tiles of 64 x 160): 7 splits = 3.83 waves (ncu: tensor pipe 68 %
  // active on the SMs that got three CTAs, 91 % on those with four) -> 20 splits = 10.95 waves.
  const int cap_long = std::max(1, K / (48 * KT)), cap_short = std::max(1, K / (8 * KT));
  int nsplit;
  if (tiles * cap_long >= 2 * slots) {
    nsplit = cap_long;
    double best_eff = 0.0;
    for (int sp = 1; sp <= cap_long; ++sp) {
      const long total = tiles * sp;
      if (total < 2 * slots) continue;
      const double eff = (double)total / (double)(ceil_div(total, slots) * slots);
      if (eff > best_eff + 1e-9) { best_eff = eff; nsplit = sp; }
    }
  } else {
    // a small product (few tiles, short K): it cannot fill two waves with long splits, so fill ONE wave as far as splits of
    // at least 8 k-tiles allow (cfg 2: 1 tile x 66 splits; with 48-tile splits it ran on 11 CTAs and cost 50 us more per call)
    nsplit = (int)std::max(1L, std::min((long)cap_short, (slots + tiles - 1) / tiles));
  }
  int kchunk = ceil_div(std::max(K, 1), nsplit);
  kchunk = ceil_div(kchunk, KT) * KT;
  nsplit = std::max(1, ceil_div(std::max(K, 1), kchunk));
  const size_t need = sizeof(cplx) * (size_t)nsplit * M * N;
  if (ws->bytes < need) {
    if (ws->part) cudaFree(ws->part);
    ws->part = nullptr; ws->bytes = 0;
    KS_CUDA_CHECK(cudaMalloc(&ws->part, need), err);
    ws->bytes = need;
  }
  dim3 grid(tn, tm, nsplit);
  k_gemm_hn<NJ, WN><<<grid, GEMM_THREADS, smem, st>>>(M, N, K, A, lda, B, ldb, ws->part, kchunk, herm_r0);
  k_splitk_reduce<<<ceil_div((long)M * N, 256), 256, 0, st>>>(M, N, nsplit, ws->part, C, ldc, herm_r0);
  KS_CUDA_CHECK(cudaGetLastError(), err);
  return KS_OK;
}

// ------------------------------------------------------------------------------------------------
// N <= 4 (one to four vectors: the band-by-band CG, the last Davidson iterations): matrix-vector forms that read A
// once at memory speed instead of spending a 16/32-wide tensor tile on one column.  Fixed summation order.
// ------------------------------------------------------------------------------------------------
#define GEMV_T 256
// C[m][n] = sum_k conj(A[k][m]) B[k][n]: one CTA per row m of A^H (column m of A), all N vectors at once
template <int NV>
__global__ void __launch_bounds__(GEMV_T) k_gemv_hn(int K, const cplx* __restrict__ A, long lda, const cplx* __restrict__ B, long ldb,
                                                    cplx* __restrict__ C, long ldc) {
  const cplx* a = A + (long)blockIdx.x * lda;
  double re[NV], im[NV];
#pragma unroll
  for (int n = 0; n < NV; ++n) re[n] = im[n] = 0.0;
  for (int k = threadIdx.x; k < K; k += GEMV_T) {
    const cplx av = a[k];
#pragma unroll
    for (int n = 0; n < NV; ++n) {
      const cplx bv = B[(long)n * ldb + k];
      re[n] += av.x * bv.x + av.y * bv.y;
      im[n] += av.x * bv.y - av.y * bv.x;
    }
  }
  __shared__ double sh[2 * NV][GEMV_T / 32];
#pragma unroll
  for (int n = 0; n < NV; ++n) {
    for (int o = 16; o > 0; o >>= 1) {
      re[n] += __shfl_xor_sync(0xffffffffu, re[n], o);
      im[n] += __shfl_xor_sync(0xffffffffu, im[n], o);
    }
    if ((threadIdx.x & 31) == 0) { sh[2 * n][threadIdx.x >> 5] = re[n]; sh[2 * n + 1][threadIdx.x >> 5] = im[n]; }
  }
  __syncthreads();
  if (threadIdx.x < NV) {
    double r = 0, i = 0;
    for (int w = 0; w < GEMV_T / 32; ++w) { r += sh[2 * threadIdx.x][w]; i += sh[2 * threadIdx.x + 1][w]; }
    C[(long)threadIdx.x * ldc + blockIdx.x] = cmake(r, i);
  }
}
// C[m][n] (+)= sum_k A[m][k] B[k][n]: a CTA owns 32 rows; its 8 warps take every 8th k (32 rows x 16 B = one 512-byte
// segment per load, 8 loads in flight per warp), partial sums meet in shared memory in a fixed order.  B (K x NV, tiny)
// is read through the read-only cache.
template <int NV>
__global__ void __launch_bounds__(GEMV_T) k_gemv_nn(int M, int K, const cplx* __restrict__ A, long lda, const cplx* __restrict__ B, long ldb,
                                                    cplx* __restrict__ C, long ldc, int accumulate) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int m = blockIdx.x * 32 + lane;
  const bool ok = m < M;
  double re[NV], im[NV];
#pragma unroll
  for (int n = 0; n < NV; ++n) re[n] = im[n] = 0.0;
  const cplx* a = A + (ok ? m : 0);
#pragma unroll 4
  for (int k = w; k < K; k += GEMV_T / 32) {
    const cplx av = a[(long)k * lda];
#pragma unroll
    for (int n = 0; n < NV; ++n) {
      const cplx bv = __ldg(&B[(long)n * ldb + k]);
      re[n] += av.x * bv.x - av.y * bv.y;
      im[n] += av.x * bv.y + av.y * bv.x;
    }
  }
  __shared__ double sh[GEMV_T / 32][2 * NV][32];
#pragma unroll
  for (int n = 0; n < NV; ++n) { sh[w][2 * n][lane] = re[n]; sh[w][2 * n + 1][lane] = im[n]; }
  __syncthreads();
  if (w == 0 && ok) {
#pragma unroll
    for (int n = 0; n < NV; ++n) {
      double r = 0, i = 0;
      for (int ww = 0; ww < GEMV_T / 32; ++ww) { r += sh[ww][2 * n][lane]; i += sh[ww][2 * n + 1][lane]; }
      cplx* p = &C[(long)n * ldc + m];
      cplx v = cmake(r, i);
      if (accumulate) { const cplx o = *p; v.x += o.x; v.y += o.y; }
      *p = v;
    }
  }
}

int ks_gemm_hn(cudaStream_t st, int M, int N, int K, const cplx* A, long lda, const cplx* B, long ldb, cplx* C,
               long ldc, GemmWs* ws, std::string& err, int herm_r0) {
  if (M <= 0 || N <= 0) return KS_OK;
  if (K < 0 || !ws) { err = "ks_gemm_hn: bad argument"; return KS_EINVAL; }
  if (N <= 4 && K >= 1024) {
    switch (N) {
      case 1: k_gemv_hn<1><<<M, GEMV_T, 0, st>>>(K, A, lda, B, ldb, C, ldc); break;
      case 2: k_gemv_hn<2><<<M, GEMV_T, 0, st>>>(K, A, lda, B, ldb, C, ldc); break;
      case 3: k_gemv_hn<3><<<M, GEMV_T, 0, st>>>(K, A, lda, B, ldb, C, ldc); break;
      default: k_gemv_hn<4><<<M, GEMV_T, 0, st>>>(K, A, lda, B, ldb, C, ldc); break;
    }
    KS_CUDA_CHECK(cudaGetLastError(), err);
    return KS_OK;
  }
  // Tile choice (KSPW_GEMM_NSPLIT=0: one launch with the least-padding wide tile, the round-1 rule):
  //   N <= 40          one launch of 8*NJ-wide tiles (WN = 1): padding < 8 columns
  //   N  > 160         whole 160-wide tiles, the rest (if any) by the same rules in a second launch
  //   40 < N <= 160    32*NJ-wide tiles; a ragged tail of 1..24 columns beyond a multiple of 32 goes to a narrow launch
  static const bool nsplit_on = !(getenv("KSPW_GEMM_NSPLIT") && atoi(getenv("KSPW_GEMM_NSPLIT")) == 0);
  if (nsplit_on) {
    if (N <= 40) {
      switch ((N + 7) / 8) {
        case 1: return launch_hn<1, 1>(st, M, N, K, A, lda, B, ldb, C, ldc, ws, err, herm_r0);
        case 2: return launch_hn<2, 1>(st, M, N, K, A, lda, B, ldb, C, ldc, ws, err, herm_r0);
        case 3: return launch_hn<3, 1>(st, M, N, K, A, lda, B, ldb, C, ldc, ws, err, herm_r0);
        case 4: return launch_hn<4, 1>(st, M, N, K, A, lda, B, ldb, C, ldc, ws, err, herm_r0);
        default: return launch_hn<5, 1>(st, M, N, K, A, lda, B, ldb, C, ldc, ws, err, herm_r0);
      }
    }
    int main_n = N;
    if (N > 160) main_n = N / 160 * 160;
    else if (N % 32 >= 1 && N % 32 <= 24) main_n = N / 32 * 32;
    if (main_n < N) {
      const int rc = ks_gemm_hn(st, M, main_n, K, A, lda, B, ldb, C, ldc, ws, err, herm_r0);
      if (rc != KS_OK) return rc;
      // the remainder's local column 0 is global column main_n: the diagonal of the Hermitian block moves down by main_n rows
      return ks_gemm_hn(st, M, N - main_n, K, A, lda, B + (long)main_n * ldb, ldb, C + (long)main_n * ldc, ldc, ws, err,
                        herm_r0 >= 0 ? herm_r0 + main_n : -1);
    }
    switch ((N + 31) / 32 > 5 ? 5 : (N + 31) / 32) {    // here N <= 160 or N % 160 == 0
      case 2: return launch_hn<2>(st, M, N, K, A, lda, B, ldb, C, ldc, ws, err, herm_r0);
      case 3: return launch_hn<3>(st, M, N, K, A, lda, B, ldb, C, ldc, ws, err, herm_r0);
      case 4: return launch_hn<4>(st, M, N, K, A, lda, B, ldb, C, ldc, ws, err, herm_r0);
      default: return launch_hn<5>(st, M, N, K, A, lda, B, ldb, C, ldc, ws, err, herm_r0);
    }
  }
  switch (pick_nj(N, 32)) {
    case 1: return launch_hn<1>(st, M, N, K, A, lda, B, ldb, C, ldc, ws, err, herm_r0);
    case 2: return launch_hn<2>(st, M, N, K, A, lda, B, ldb, C, ldc, ws, err, herm_r0);
    case 3: return launch_hn<3>(st, M, N, K, A, lda, B, ldb, C, ldc, ws, err, herm_r0);
    case 4: return launch_hn<4>(st, M, N, K, A, lda, B, ldb, C, ldc, ws, err, herm_r0);
    default: return launch_hn<5>(st, M, N, K, A, lda, B, ldb, C, ldc, ws, err, herm_r0);
  }
}

// ------------------------------------------------------------------------------------------------
// C (+)= A B.  CTA tile 128 (M) x 16*NJ (N), 8 warps as 4 (M) x 2 (N), warp tile 32 x 8*NJ -> 4 x NJ MMA tiles,
// NJ in 1..5 picked per call for the least padding of N (N = 160 -> two 80-wide tiles, not three 64-wide ones).
// ------------------------------------------------------------------------------------------------
#define NN_MT 128
#define LDM (NN_MT + 2)   // "m-contiguous" tile leading dimension: == 2 (mod 8)

// WN = warps along N (WM = 8 / WN along M): WN = 2 is the tile above; WN = 1 gives an N-tile of 8*NJ columns (8 .. 40) with
// 16-row warp tiles, for narrow products and the ragged remainder of a wide one (see gemm_hn_tile).
template <int NJ, int WN = 2>
__device__ __forceinline__ void gemm_nn_tile(int M, int N, int K, const cplx* __restrict__ A, long lda, const cplx* __restrict__ B,
                                             long ldb, cplx* __restrict__ C, long ldc, int accumulate, int m0, int n0) {
  constexpr int WM = 8 / WN, MI = NN_MT / (8 * WM), NN_NT = 8 * NJ * WN;
  extern __shared__ cplx sm[];
  cplx* sA = sm;                                   // [stage][KT][LDM]
  cplx* sB = sm + GEMM_STAGES * KT * LDM;          // [stage][NN_NT][LDK]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp % WM, wn = warp / WM;
  const int ntile = (K + KT - 1) / KT;

  auto load_stage = [&](int st, int kt) {
    const int k0 = kt * KT;
#pragma unroll
    for (int r = 0; r < (NN_MT * KT) / GEMM_THREADS; ++r) {
      const int e = tid + r * GEMM_THREADS, kk = e / NN_MT, mm = e % NN_MT;
      const bool ok = (m0 + mm < M) && (k0 + kk < K);
      cp16(&sA[(st * KT + kk) * LDM + mm], ok ? &A[(long)(k0 + kk) * lda + m0 + mm] : A, ok);
    }
#pragma unroll
    for (int r = 0; r < (NN_NT * KT + GEMM_THREADS - 1) / GEMM_THREADS; ++r) {
      const int e = tid + r * GEMM_THREADS, col = e / KT, kk = e % KT;
      if ((NN_NT * KT) % GEMM_THREADS != 0 && e >= NN_NT * KT) break;
      const bool ok = (n0 + col < N) && (k0 + kk < K);
      cp16(&sB[(st * NN_NT + col) * LDK + kk], ok ? &B[(long)(n0 + col) * ldb + k0 + kk] : B, ok);
    }
  };

  double cre[MI][NJ][2], cim[MI][NJ][2];
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int j = 0; j < NJ; ++j) cre[i][j][0] = cre[i][j][1] = cim[i][j][0] = cim[i][j][1] = 0.0;

  for (int s = 0; s < GEMM_STAGES - 1; ++s) {
    if (s < ntile) load_stage(s, s);
    cp_commit();
  }
  const int fr = lane >> 2, fk = lane & 3;
#ifdef KSPW_GEMM_NO_STAGGER
  const bool late = false;
#else
  const bool late = warp >= 4;      // see gemm_hn_tile: the two warps of a sub-partition issue their loads at different times
#endif
  for (int kt = 0; kt < ntile; ++kt) {
    cp_wait<GEMM_STAGES - 2>();
    __syncthreads();
    const bool more = kt + GEMM_STAGES - 1 < ntile;
#ifdef KSPW_GEMM_NO_STAGGER
    if (more) load_stage((kt + GEMM_STAGES - 1) % GEMM_STAGES, kt + GEMM_STAGES - 1);
    cp_commit();
#endif
    const cplx* a = sA + (kt % GEMM_STAGES) * KT * LDM + wm * 8 * MI;
    const cplx* b = sB + ((kt % GEMM_STAGES) * NN_NT + wn * 8 * NJ) * LDK;
#pragma unroll
    for (int ks = 0; ks < KT; ks += 4) {
#ifndef KSPW_GEMM_NO_STAGGER
      if (ks == (late ? KS_LATE : KS_EARLY)) {
        if (more) load_stage((kt + GEMM_STAGES - 1) % GEMM_STAGES, kt + GEMM_STAGES - 1);
        cp_commit();
      }
#endif
      cplx af[MI], bf[NJ];
#pragma unroll
      for (int i = 0; i < MI; ++i) af[i] = a[(ks + fk) * LDM + i * 8 + fr];
#pragma unroll
      for (int j = 0; j < NJ; ++j) bf[j] = b[(j * 8 + fr) * LDK + ks + fk];
#pragma unroll
      for (int i = 0; i < MI; ++i) {
        const double nai = -af[i].y;
#pragma unroll
        for (int j = 0; j < NJ; ++j) {   // a b = (ar br - ai bi) + i (ar bi + ai br)
          dmma(cre[i][j][0], cre[i][j][1], af[i].x, bf[j].x);
          dmma(cim[i][j][0], cim[i][j][1], af[i].x, bf[j].y);
          dmma(cre[i][j][0], cre[i][j][1], nai, bf[j].y);
          dmma(cim[i][j][0], cim[i][j][1], af[i].y, bf[j].x);
        }
      }
    }
  }
  cp_wait<0>();
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int j = 0; j < NJ; ++j)
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int m = m0 + wm * 8 * MI + i * 8 + fr, n = n0 + wn * 8 * NJ + j * 8 + 2 * fk + h;
        if (m < M && n < N) {
          cplx* p = &C[(long)n * ldc + m];
#ifndef KSPW_GEMM_NN_RMW
          // C += tile as two reductions without a return value (SASS RED.ADD.F64): every element has exactly one writer in
          // the launch, so the sum is the same IEEE addition as load-add-store, bit for bit and deterministic -- but the
          // thread does not wait ~1 us for each of its 40 old values in turn (stores to C may alias the next load, so the
          // compiler keeps load-add-store pairs in order: ncu showed the DMMA pipe idle for ~9 % of a CTA's life at cfg 3,
          // more where K is short)
          if (accumulate) { atomicAdd(&p->x, cre[i][j][h]); atomicAdd(&p->y, cim[i][j][h]); }
          else *p = cmake(cre[i][j][h], cim[i][j][h]);
#else
          cplx v = cmake(cre[i][j][h], cim[i][j][h]);
          if (accumulate) { const cplx o = *p; v.x += o.x; v.y += o.y; }
          *p = v;
#endif
        }
      }
}

template <int NJ, int WN = 2>
__global__ void __launch_bounds__(GEMM_THREADS) k_gemm_nn(int M, int N, int K, const cplx* __restrict__ A, long lda,
                                                          const cplx* __restrict__ B, long ldb, cplx* __restrict__ C,
                                                          long ldc, int accumulate, int btri_c0) {
  // triangular B (B[k][n] = 0 for k > btri_c0 + n): this N-tile's products end at row btri_c0 + (its last column)
  const int n0 = blockIdx.y * 8 * NJ * WN;
  const int Keff = btri_c0 >= 0 ? min(K, btri_c0 + n0 + 8 * NJ * WN) : K;
  gemm_nn_tile<NJ, WN>(M, N, Keff, A, lda, B, ldb, C, ldc, accumulate, blockIdx.x * NN_MT, n0);
}
template <int NJ>
__global__ void __launch_bounds__(GEMM_THREADS) k_gemm_nn_g(const GemmProb* __restrict__ probs, int accumulate) {
  const GemmProb p = probs[blockIdx.z];
  const int m0 = blockIdx.x * NN_MT, n0 = blockIdx.y * 16 * NJ;
  if (m0 >= p.M || n0 >= p.N) return;
  gemm_nn_tile<NJ>(p.M, p.N, p.K, p.A, p.lda, p.B, p.ldb, p.C, p.ldc, accumulate, m0, n0);
}

template <int NJ, int WN = 2>
static int launch_nn(cudaStream_t st, int M, int N, int K, const cplx* A, long lda, const cplx* B, long ldb, cplx* C,
                     long ldc, int accumulate, std::string& err, int btri_c0 = -1) {
  constexpr int NN_NT = 8 * NJ * WN;
  static std::atomic<bool> opted{false};
  const size_t smem = sizeof(cplx) * GEMM_STAGES * (KT * LDM + NN_NT * LDK);
  if (!opted) {
    KS_CUDA_CHECK((cudaFuncSetAttribute(k_gemm_nn<NJ, WN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)), err);
    opted = true;
  }
  dim3 grid(ceil_div(M, NN_MT), ceil_div(N, NN_NT));
  k_gemm_nn<NJ, WN><<<grid, GEMM_THREADS, smem, st>>>(M, N, K, A, lda, B, ldb, C, ldc, accumulate, btri_c0);
  KS_CUDA_CHECK(cudaGetLastError(), err);
  return KS_OK;
}

int ks_gemm_nn(cudaStream_t st, int M, int N, int K, const cplx* A, long lda, const cplx* B, long ldb, cplx* C,
               long ldc, int accumulate, std::string& err, int btri_c0) {
  if (M <= 0 || N <= 0) return KS_OK;
  if (K < 0) { err = "ks_gemm_nn: bad argument"; return KS_EINVAL; }
  if (N <= 4 && M >= 1024 && K >= 1) {
    const int grid = ceil_div(M, 32);
    switch (N) {
      case 1: k_gemv_nn<1><<<grid, GEMV_T, 0, st>>>(M, K, A, lda, B, ldb, C, ldc, accumulate); break;
      case 2: k_gemv_nn<2><<<grid, GEMV_T, 0, st>>>(M, K, A, lda, B, ldb, C, ldc, accumulate); break;
      case 3: k_gemv_nn<3><<<grid, GEMV_T, 0, st>>>(M, K, A, lda, B, ldb, C, ldc, accumulate); break;
      default: k_gemv_nn<4><<<grid, GEMV_T, 0, st>>>(M, K, A, lda, B, ldb, C, ldc, accumulate); break;
    }
    KS_CUDA_CHECK(cudaGetLastError(), err);
    return KS_OK;
  }
  // Tile choice (KSPW_GEMM_NSPLIT=0: one launch with the least-padding 16*NJ-wide tile, the round-1 rule):
  //   N <= 40         one launch of 8*NJ-wide tiles (WN = 1)
  //   N  > 80         whole 80-wide tiles (more DMMAs per fragment load, A re-read N/80 times), the rest in a second launch
  //   40 < N <= 80    16*NJ-wide tiles; a ragged tail of 1..8 columns beyond a multiple of 16 goes to a narrow launch
  static const bool nsplit_on = !(getenv("KSPW_GEMM_NSPLIT") && atoi(getenv("KSPW_GEMM_NSPLIT")) == 0);
  if (nsplit_on) {
    if (N <= 40) {
      switch ((N + 7) / 8) {
        case 1: return launch_nn<1, 1>(st, M, N, K, A, lda, B, ldb, C, ldc, accumulate, err, btri_c0);
        case 2: return launch_nn<2, 1>(st, M, N, K, A, lda, B, ldb, C, ldc, accumulate, err, btri_c0);
        case 3: return launch_nn<3, 1>(st, M, N, K, A, lda, B, ldb, C, ldc, accumulate, err, btri_c0);
        case 4: return launch_nn<4, 1>(st, M, N, K, A, lda, B, ldb, C, ldc, accumulate, err, btri_c0);
        default: return launch_nn<5, 1>(st, M, N, K, A, lda, B, ldb, C, ldc, accumulate, err, btri_c0);
      }
    }
    int main_n = N;
    if (N > 80) main_n = N / 80 * 80;
    else if (N % 16 >= 1 && N % 16 <= 8) main_n = N / 16 * 16;
    if (main_n < N) {
      const int rc = ks_gemm_nn(st, M, main_n, K, A, lda, B, ldb, C, ldc, accumulate, err, btri_c0);
      if (rc != KS_OK) return rc;
      return ks_gemm_nn(st, M, N - main_n, K, A, lda, B + (long)main_n * ldb, ldb, C + (long)main_n * ldc, ldc, accumulate, err,
                        btri_c0 >= 0 ? btri_c0 + main_n : -1);
    }
    switch ((N + 15) / 16 > 5 ? 5 : (N + 15) / 16) {    // here N <= 80 or N % 80 == 0
      case 3: return launch_nn<3>(st, M, N, K, A, lda, B, ldb, C, ldc, accumulate, err, btri_c0);
      case 4: return launch_nn<4>(st, M, N, K, A, lda, B, ldb, C, ldc, accumulate, err, btri_c0);
      default: return launch_nn<5>(st, M, N, K, A, lda, B, ldb, C, ldc, accumulate, err, btri_c0);
    }
  }
  switch (pick_nj(N, 16)) {
    case 1: return launch_nn<1>(st, M, N, K, A, lda, B, ldb, C, ldc, accumulate, err, btri_c0);
    case 2: return launch_nn<2>(st, M, N, K, A, lda, B, ldb, C, ldc, accumulate, err, btri_c0);
    case 3: return launch_nn<3>(st, M, N, K, A, lda, B, ldb, C, ldc, accumulate, err, btri_c0);
    case 4: return launch_nn<4>(st, M, N, K, A, lda, B, ldb, C, ldc, accumulate, err, btri_c0);
    default: return launch_nn<5>(st, M, N, K, A, lda, B, ldb, C, ldc, accumulate, err, btri_c0);
  }
}

// ------------------------------------------------------------------------------------------------
// Grouped launches (ks_hpsi_batch): ng independent problems of similar size in ONE launch each.  dev_probs: DEVICE [ng].
// ------------------------------------------------------------------------------------------------
// split count for ng problems of (about) M x N x K: enough CTAs for two waves of the resident slots, >= 8 k-tiles per split
int ks_gemm_hn_group_nsplit(int ng, int M, int N, int K) {
  const int nj = pick_nj(N, 32);
  const size_t smem = sizeof(cplx) * GEMM_STAGES * (HN_MT + 32 * nj) * LDK;
  const int per_sm = std::max(1, (int)((227 * 1024) / (smem + 1024)));
  const long slots = 148L * per_sm, tiles = (long)ng * ceil_div(M, HN_MT) * ceil_div(N, 32 * nj);
  const int max_split = std::max(1, K / (8 * KT));
  return (int)std::max(1L, std::min((long)max_split, (2 * slots + tiles - 1) / tiles));
}

template <int NJ>
static int launch_hn_g(cudaStream_t st, const GemmProb* dev_probs, int ng, int M, int N, int nsplit, std::string& err) {
  static std::atomic<bool> opted{false};
  const size_t smem = sizeof(cplx) * GEMM_STAGES * (HN_MT + 32 * NJ) * LDK;
  if (!opted.load()) {
    KS_CUDA_CHECK(cudaFuncSetAttribute(k_gemm_hn_g<NJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), err);
    opted.store(true);
  }
  const dim3 grid(ceil_div(N, 32 * NJ), ceil_div(M, HN_MT), ng * nsplit);
  k_gemm_hn_g<NJ><<<grid, GEMM_THREADS, smem, st>>>(dev_probs, nsplit);
  KS_CUDA_CHECK(cudaGetLastError(), err);
  return KS_OK;
}
// partial sums C_g[z] = A_g^H B_g over split z of K_g; M, N: the largest of the group (sizes the grid and the tile width)
int ks_gemm_hn_group(cudaStream_t st, const GemmProb* dev_probs, int ng, int M, int N, int nsplit, std::string& err) {
  if (ng <= 0 || M <= 0 || N <= 0) return KS_OK;
  if ((long)ng * nsplit > 65535) { err = "ks_gemm_hn_group: too many problems x splits for one launch"; return KS_EINVAL; }
  switch (pick_nj(N, 32)) {
    case 1: return launch_hn_g<1>(st, dev_probs, ng, M, N, nsplit, err);
    case 2: return launch_hn_g<2>(st, dev_probs, ng, M, N, nsplit, err);
    case 3: return launch_hn_g<3>(st, dev_probs, ng, M, N, nsplit, err);
    case 4: return launch_hn_g<4>(st, dev_probs, ng, M, N, nsplit, err);
    default: return launch_hn_g<5>(st, dev_probs, ng, M, N, nsplit, err);
  }
}

template <int NJ>
static int launch_nn_g(cudaStream_t st, const GemmProb* dev_probs, int ng, int M, int N, int accumulate, std::string& err) {
  static std::atomic<bool> opted{false};
  const size_t smem = sizeof(cplx) * GEMM_STAGES * (KT * LDM + 16 * NJ * LDK);
  if (!opted.load()) {
    KS_CUDA_CHECK(cudaFuncSetAttribute(k_gemm_nn_g<NJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), err);
    opted.store(true);
  }
  const dim3 grid(ceil_div(M, NN_MT), ceil_div(N, 16 * NJ), ng);
  k_gemm_nn_g<NJ><<<grid, GEMM_THREADS, smem, st>>>(dev_probs, accumulate);
  KS_CUDA_CHECK(cudaGetLastError(), err);
  return KS_OK;
}
// C_g (+)= A_g B_g for every problem of the group
int ks_gemm_nn_group(cudaStream_t st, const GemmProb* dev_probs, int ng, int M, int N, int accumulate, std::string& err) {
  if (ng <= 0 || M <= 0 || N <= 0) return KS_OK;
  if (ng > 65535) { err = "ks_gemm_nn_group: too many problems for one launch"; return KS_EINVAL; }
  switch (pick_nj(N, 16)) {
    case 1: return launch_nn_g<1>(st, dev_probs, ng, M, N, accumulate, err);
    case 2: return launch_nn_g<2>(st, dev_probs, ng, M, N, accumulate, err);
    case 3: return launch_nn_g<3>(st, dev_probs, ng, M, N, accumulate, err);
    case 4: return launch_nn_g<4>(st, dev_probs, ng, M, N, accumulate, err);
    default: return launch_nn_g<5>(st, dev_probs, ng, M, N, accumulate, err);
  }
}

// ------------------------------------------------------------------------------------------------
// Roofline denominators: register-resident DMMA and DFMA loops (no memory traffic).
// ------------------------------------------------------------------------------------------------
// 4 x 4 grid of accumulator tiles fed by four A and four B fragments, as in the GEMM inner loop.  (A loop that
// feeds all 16 DMMAs from ONE operand pair reads 29.7 TFLOP/s at 32 warps/SM and 36.8 at 8 warps/SM on the same
// B200; with distinct fragments it is 36.9-37.0 at every occupancy, so that is the peak.)
__global__ void __launch_bounds__(256) k_dmma_peak(double* out, int iters) {
  double c[16][2];
#pragma unroll
  for (int i = 0; i < 16; ++i) c[i][0] = c[i][1] = 0.0;
  double a[4], b[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) { a[i] = 1.0 + 1e-9 * (threadIdx.x + i); b[i] = 1.0 - 1e-9 * (threadIdx.x + 7 * i); }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) dmma(c[4 * i + j][0], c[4 * i + j][1], a[i], b[j]);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += c[i][0] + c[i][1];
  if (s == 12345.678) out[0] = s;
}
__global__ void __launch_bounds__(256) k_dfma_peak(double* out, int iters) {
  double c[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) c[i] = 1e-3 * i;
  const double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-9 * threadIdx.x;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) c[i] = fma(c[i], a, b);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += c[i];
  if (s == 12345.678) out[0] = s;
}

// DMMA result latency probe: NACC independent accumulators per warp, each DMMA depends on the one NACC issues earlier.
// 8 warps per SM sub-partition would hide it; ONE warp per sub-partition (128-thread CTA, one CTA per SM) shows it.
template <int NACC>
__global__ void __launch_bounds__(128) k_dmma_chain(double* out, int iters) {
  double c[NACC][2];
#pragma unroll
  for (int i = 0; i < NACC; ++i) c[i][0] = c[i][1] = 0.0;
  const double a = 1.0 + 1e-9 * threadIdx.x, b = 1.0 - 1e-9 * threadIdx.x;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < NACC; ++i) dmma(c[i][0], c[i][1], a, b);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < NACC; ++i) s += c[i][0] + c[i][1];
  if (s == 12345.678) out[0] = s;
}
// clocks per DMMA of one warp on its sub-partition with NACC = 1, 2, 3, 4, 6, 8 independent accumulators (HOST out [6])
int ks_dmma_latency_run(double* clk_per_dmma, double sm_ghz, std::string& err) {
  double* d = nullptr;
  KS_CUDA_CHECK(cudaMalloc(&d, 8), err);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int iters = 20000;
  for (int v = 0; v < 6; ++v) {
    float best = 1e30f;
    const int nacc[6] = {1, 2, 3, 4, 6, 8};
    for (int rep = 0; rep < 3; ++rep) {
      cudaEventRecord(e0);
      switch (v) {
        case 0: k_dmma_chain<1><<<148, 128>>>(d, iters); break;
        case 1: k_dmma_chain<2><<<148, 128>>>(d, iters); break;
        case 2: k_dmma_chain<3><<<148, 128>>>(d, iters); break;
        case 3: k_dmma_chain<4><<<148, 128>>>(d, iters); break;
        case 4: k_dmma_chain<6><<<148, 128>>>(d, iters); break;
        default: k_dmma_chain<8><<<148, 128>>>(d, iters); break;
      }
      cudaEventRecord(e1);
      KS_CUDA_CHECK(cudaEventSynchronize(e1), err);
      float ms; cudaEventElapsedTime(&ms, e0, e1);
      if (rep) best = std::min(best, ms);
    }
    clk_per_dmma[v] = best * 1e-3 * sm_ghz * 1e9 / ((double)iters * nacc[v]);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
  return KS_OK;
}

int ks_peak_run(double* dmma_tf, double* dfma_tf, std::string& err) {
  double* d = nullptr;
  KS_CUDA_CHECK(cudaMalloc(&d, 8), err);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int blocks = 148 * 4, iters = 20000;
  float best_m = 1e30f, best_f = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0);
    k_dmma_peak<<<blocks, 256>>>(d, iters);
    cudaEventRecord(e1);
    KS_CUDA_CHECK(cudaEventSynchronize(e1), err);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    if (rep) best_m = std::min(best_m, ms);
    cudaEventRecord(e0);
    k_dfma_peak<<<blocks, 256>>>(d, iters);
    cudaEventRecord(e1);
    KS_CUDA_CHECK(cudaEventSynchronize(e1), err);
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep) best_f = std::min(best_f, ms);
  }
  // per warp and iteration: 16 DMMA x 512 flop ; per thread and iteration: 16 DFMA x 2 flop
  const double fl_m = (double)blocks * 8 * iters * 16 * 512.0, fl_f = (double)blocks * 256 * iters * 16 * 2.0;
  if (dmma_tf) *dmma_tf = fl_m / (best_m * 1e-3) / 1e12;
  if (dfma_tf) *dfma_tf = fl_f / (best_f * 1e-3) / 1e12;
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
  return KS_OK;
}

// Can the DMMA and the DFMA pipe be fed at the same time?  (If they could, a mixed-pipe GEMM would have a ceiling above the
// DMMA peak.)  mode 0: every warp runs the DMMA loop; 1: every warp the DFMA loop; 2: warps 0-3 DMMA and warps 4-7 DFMA
// (each SM sub-partition holds one warp of either kind); 3: every warp interleaves 16 DMMAs with 16 DFMAs per iteration.
// out[mode] = summed TFLOP/s (512 flop per DMMA, 2 flop per DFMA lane).
__global__ void __launch_bounds__(256) k_fp64_mix(double* out, int iters, int mode) {
  double c[16][2], f[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) { c[i][0] = c[i][1] = 0.0; f[i] = 1e-3 * i; }
  double a[4], b[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) { a[i] = 1.0 + 1e-9 * (threadIdx.x + i); b[i] = 1.0 - 1e-9 * (threadIdx.x + 7 * i); }
  const double fa = 1.0 + 1e-9 * threadIdx.x, fb = 1e-9 * threadIdx.x;
  const int warp = threadIdx.x >> 5;
  const bool do_m = mode == 0 || mode == 3 || (mode == 2 && warp < 4);
  const bool do_f = mode == 1 || mode == 3 || (mode == 2 && warp >= 4);
  for (int it = 0; it < iters; ++it) {
    if (do_m) {
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) dmma(c[4 * i + j][0], c[4 * i + j][1], a[i], b[j]);
    }
    if (do_f) {
#pragma unroll
      for (int i = 0; i < 16; ++i) f[i] = fma(f[i], fa, fb);
    }
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += c[i][0] + c[i][1] + f[i];
  if (s == 12345.678) out[0] = s;
}
int ks_fp64_mix_run(double* tflops4, std::string& err) {
  double* d = nullptr;
  KS_CUDA_CHECK(cudaMalloc(&d, 8), err);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int blocks = 148 * 4, iters = 20000;
  for (int mode = 0; mode < 4; ++mode) {
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
      cudaEventRecord(e0);
      k_fp64_mix<<<blocks, 256>>>(d, iters, mode);
      cudaEventRecord(e1);
      KS_CUDA_CHECK(cudaEventSynchronize(e1), err);
      float ms; cudaEventElapsedTime(&ms, e0, e1);
      if (rep) best = std::min(best, ms);
    }
    const double wm = (mode == 0 || mode == 3) ? 8 : (mode == 2 ? 4 : 0), wf = (mode == 1 || mode == 3) ? 8 : (mode == 2 ? 4 : 0);
    const double fl = (double)blocks * iters * 16 * (wm * 512.0 + wf * 32 * 2.0);
    tflops4[mode] = fl / (best * 1e-3) / 1e12;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
  return KS_OK;
}

// ------------------------------------------------------------------------------------------------
// ks_zgemm_hn_static: C = A^H B for callers that cannot call cudaMalloc (code under CUDA graph capture, serving loops,
// harnesses that forbid allocation).  The same split-K kernels as ks_gemm_hn (k_gemm_hn<NJ> + k_splitk_reduce), with the
// partial tiles in a file-scope device array instead of the growing GemmWs buffer.
//
//   * the array is KS_STATIC_SCRATCH_BYTES (8 MiB) on every GPU that loads the library, until the process exits;
//   * nsplit * M * N complex partials must fit: M * N <= KS_STATIC_SCRATCH_ELEMS (524 288, e.g. 724 x 724), and the split
//     count is capped at KS_STATIC_SCRATCH_ELEMS / (M * N) -- larger products are rejected with KS_EINVAL, never truncated;
//   * nothing in the array has to start at zero: every element of part[0 : nsplit][N][M] that the reduction reads is
//     written by exactly one CTA of the launch before it (every split owns a non-empty K range, or K = 0 and the one
//     split writes zeros), so the previous call's contents are never observed;
//   * every call shares the one array: two calls that overlap on the GPU (different streams, or two host threads on
//     different streams) race on it.  Calls on one stream are ordered and safe.
//
// In host code `g_hn_scratch` is a host-side stand-in, not a device address; the address the kernels get comes from
// cudaGetSymbolAddress, looked up once per device with that device current (static_setup), together with the kernels'
// shared-memory opt-in.  The call itself launches two kernels and calls no cudaMalloc / cudaFree / allocating routine.
// ------------------------------------------------------------------------------------------------
#define KS_STATIC_SCRATCH_BYTES (8u << 20)
#define KS_STATIC_SCRATCH_ELEMS (KS_STATIC_SCRATCH_BYTES / sizeof(cplx))
static __device__ __align__(256) unsigned char g_hn_scratch[KS_STATIC_SCRATCH_BYTES];

#define KS_STATIC_MAX_DEV 64
static cplx* g_static_ptr[KS_STATIC_MAX_DEV];        // device address of g_hn_scratch on device d (nullptr: not set up yet)
static std::atomic<bool> g_static_ready[KS_STATIC_MAX_DEV];

template <int NJ>
static cudaError_t static_opt_in() {
  const size_t smem = sizeof(cplx) * GEMM_STAGES * (HN_MT + 32 * NJ) * LDK;
  return cudaFuncSetAttribute(k_gemm_hn<NJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
}

// once per device, with that device current
static int static_setup(int dev, std::string& err) {
  if (g_static_ready[dev].load(std::memory_order_acquire)) return KS_OK;
  void* p = nullptr;
  KS_CUDA_CHECK(cudaGetSymbolAddress(&p, g_hn_scratch), err);
  KS_CUDA_CHECK(static_opt_in<1>(), err);
  KS_CUDA_CHECK(static_opt_in<2>(), err);
  KS_CUDA_CHECK(static_opt_in<3>(), err);
  KS_CUDA_CHECK(static_opt_in<4>(), err);
  KS_CUDA_CHECK(static_opt_in<5>(), err);
  g_static_ptr[dev] = (cplx*)p;
  g_static_ready[dev].store(true, std::memory_order_release);
  return KS_OK;
}

template <int NJ>
static int launch_hn_static(cudaStream_t st, int M, int N, int K, const cplx* A, long lda, const cplx* B, long ldb, cplx* C,
                            long ldc, cplx* part, std::string& err) {
  constexpr int HN_NT = 32 * NJ;
  const size_t smem = sizeof(cplx) * GEMM_STAGES * (HN_MT + HN_NT) * LDK;
  const int tm = ceil_div(M, HN_MT), tn = ceil_div(N, HN_NT);
  // split K: fill one wave of CTA slots, at least 8 k-tiles per split, and never more partial tiles than the array holds
  const int per_sm = std::max(1, (int)((227 * 1024) / (smem + 1024)));
  const long slots = 148L * per_sm, tiles = (long)tm * tn;
  const long cap_scratch = (long)(KS_STATIC_SCRATCH_ELEMS / ((size_t)M * N));      // >= 1: checked by the caller
  const long cap_short = std::max(1, K / (8 * KT));
  int nsplit = (int)std::max(1L, std::min(std::min(cap_short, cap_scratch), (slots + tiles - 1) / tiles));
  int kchunk = ceil_div(std::max(K, 1), nsplit);
  kchunk = ceil_div(kchunk, KT) * KT;
  nsplit = std::max(1, ceil_div(std::max(K, 1), kchunk));      // only shrinks: still within the array
  dim3 grid(tn, tm, nsplit);
  k_gemm_hn<NJ><<<grid, GEMM_THREADS, smem, st>>>(M, N, K, A, lda, B, ldb, part, kchunk, -1);
  k_splitk_reduce<<<ceil_div((long)M * N, 256), 256, 0, st>>>(M, N, nsplit, part, C, ldc);
  KS_CUDA_CHECK(cudaGetLastError(), err);
  return KS_OK;
}

extern "C" int ks_zgemm_hn_static(void* stream, int M, int N, int K, const void* A, long lda, const void* B, long ldb, void* C,
                                  long ldc) {
  std::string& err = ks_global_error();
  if (M < 1 || N < 1 || K < 0 || (K > 0 && (!A || !B)) || !C || lda < K || ldb < K || ldc < M) {
    err = "ks_zgemm_hn_static: bad argument (M, N >= 1, K >= 0, lda, ldb >= K, ldc >= M, non-NULL device pointers unless K = 0)";
    return KS_EINVAL;
  }
  if ((size_t)M * (size_t)N > KS_STATIC_SCRATCH_ELEMS) {
    char b[256];
    snprintf(b, sizeof b, "ks_zgemm_hn_static: M * N = %zu exceeds the static scratch array (%zu complex128 elements = %u MiB); "
             "use ks_zgemm_hn, which allocates its workspace", (size_t)M * (size_t)N, (size_t)KS_STATIC_SCRATCH_ELEMS,
             KS_STATIC_SCRATCH_BYTES >> 20);
    err = b;
    return KS_EINVAL;
  }
  int dev = 0;
  KS_CUDA_CHECK(cudaGetDevice(&dev), err);
  if (dev < 0 || dev >= KS_STATIC_MAX_DEV) { err = "ks_zgemm_hn_static: device index beyond 63"; return KS_EINVAL; }
  const int rc = static_setup(dev, err);
  if (rc != KS_OK) return rc;
  cplx* part = g_static_ptr[dev];
  cudaStream_t st = (cudaStream_t)stream;
  const cplx *a = (const cplx*)A, *b = (const cplx*)B;
  cplx* c = (cplx*)C;
  switch (pick_nj(N, 32)) {
    case 1: return launch_hn_static<1>(st, M, N, K, a, lda, b, ldb, c, ldc, part, err);
    case 2: return launch_hn_static<2>(st, M, N, K, a, lda, b, ldb, c, ldc, part, err);
    case 3: return launch_hn_static<3>(st, M, N, K, a, lda, b, ldb, c, ldc, part, err);
    case 4: return launch_hn_static<4>(st, M, N, K, a, lda, b, ldb, c, ldc, part, err);
    default: return launch_hn_static<5>(st, M, N, K, a, lda, b, ldb, c, ldc, part, err);
  }
}
