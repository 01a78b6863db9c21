// eigh.cu -- Jacobi Hermitian eigensolver for the subspace matrix (DESIGN.md step D3) and for the
// Gram matrices of the orthonormalisation (D0, D7).  The paper is silent on the subspace solver
// (north_star: "a Jacobi-style Hermitian eigensolver kernel"); the oracle uses cyclic-by-row Jacobi,
// this file uses parallel (round-robin) ordering -- the results agree to round-off.
//
//   n <= 64   one CTA: A and the accumulated rotations V live in shared memory; every round applies
//             n/2 disjoint complex Givens rotations (two-sided), n-1 rounds per sweep.
//   n  > 64   two-sided BLOCK Jacobi with 16-wide blocks: every round solves nblk/2 independent 32x32 pair problems
//             with the one-CTA solver (one inner sweep; after round 0 of an outer sweep only the pivots that couple the
//             two blocks), then applies the 32x32 unitary blocks: one CTA per 32x32 tile computes U_a^H A U_b (or V U_b)
//             in place (k_jac_upd32).  For n >= 512 one launch per round does both (k_jac_round32): the solver CTAs of
//             the NEXT round rebuild their pair matrices from the old A and this round's U and run next to the tile
//             CTAs (A double buffered).  (The older 64x64 pair / column + row DMMA kernels remain behind KSPW_JAC_PAIR=64.)
// Rotation for pivot (p,q), a_pq = |a_pq| e^{i phi}:  J = diag(1, e^{-i phi}) [[c, s], [-s, c]],
// tau = (a_qq - a_pp)/(2|a_pq|), t = sign(tau)/(|tau| + sqrt(1 + tau^2))  (the oracle's rotation, evaluated here in the
// division-free form c = sqrt((1 + |d|/r)/2), sg = sign(d) a_pq/(2 r c), d = (a_qq - a_pp)/2, r = sqrt(d^2 + |a_pq|^2)).
#include "mma.cuh"
#include "plan.h"
#include <algorithm>
#include <atomic>
#include <cstdlib>
#include <vector>
#include <cooperative_groups.h>
namespace cg = cooperative_groups;

#define JB 32            // block size of the block method
#define JS (2 * JB)      // pair problem size
#define JTHREADS 1024
#define JPAD 1.0e30      // diagonal of padding rows: decoupled (zero off-diagonals) and sorts last

// round-robin pair k of round r for n (even) players: (n-1, r) for k = 0, else ((r+k) % (n-1), (r-k) % (n-1))
__host__ __device__ __forceinline__ void rr_pair(int n, int r, int k, int* p, int* q) {
  int a, b;
  if (k == 0) { a = n - 1; b = r; }
  else { a = (r + k) % (n - 1); b = (r - k + (n - 1)) % (n - 1); }
  *p = a < b ? a : b;
  *q = a < b ? b : a;
}

// ------------------------------------------------------------------------------------------------
// one CTA per pair problem.  ns = 2*nbk (even, <= 64).  Gathers rows/cols {I*nbk.., J*nbk..} of Ap.
// U (ns x ns, column-major, ld = ns) receives the accumulated rotations; dout (nullable) the diagonal.
//
// A round applies ns/2 disjoint rotations J_k = [[c, sg], [-conj(sg), c]] (sg = s e^{i phi}; this is the
// rotation of the header times diag(1, e^{i phi}), which zeroes the same pivot).  Two barriers per round:
//   phase 1  ns/2 threads: (c, sg) from a_pp, a_qq, a_pq.  With a = |a_pq|^2, d = (a_qq - a_pp)/2,
//            r = sqrt(d^2 + a):  z = sign(d) a_pq / (|d| + r),  c = rsqrt(1 + |z|^2),  sg = c z.
//   phase 2  one thread per 2x2 block (k, l):  A[{p_k,q_k},{p_l,q_l}] <- J_k^H (.) J_l  and
//            V[{p_k,q_k},{p_l,q_l}] <- (.) J_l, all in registers.
// ------------------------------------------------------------------------------------------------
// The solver proper.  Shared memory (caller provides; ns = 2*nbk, LD = ns+1): As[ns*LD] filled with the pair
// problem (As[i*LD + j] = A[i][j]), Vs[ns*LD] (set to the identity here), then `scr`: >= 16*(JS/2) + 8*(JS/2) +
// 2*(ns-1)*(ns/2) bytes.  On return As holds the rotated matrix and Vs the accumulated rotations.
__device__ __forceinline__ void jac_solve_smem(cplx* As, cplx* Vs, void* scr, int nbk, int max_sweeps, double tol2, int cross) {
  const int ns = 2 * nbk, LD = ns + 1, hp = ns / 2;
  cplx* rsg = (cplx*)scr;              // sg[k]
  double* rc = (double*)(rsg + JS / 2);                 // c[k]
  uchar2* sched = (uchar2*)(rc + JS / 2);               // [rounds][hp] pivot pairs of every round
  __shared__ double red[2][JTHREADS / 32];
  __shared__ int stop;
  const int tid = threadIdx.x, nt = blockDim.x;
  for (int e = tid; e < ns * ns; e += nt) {
    const int i = e % ns, j = e / ns;
    Vs[i * LD + j] = cmake(i == j ? 1.0 : 0.0, 0.0);
  }
  // cross != 0: only the pivots that couple the two blocks (p in the first, q in the second): nbk rounds of nbk
  // disjoint rotations.  The pivots inside a block are swept once per outer sweep, by the round-0 launches.
  const int nrounds = cross ? nbk : ns - 1;
  for (int e = tid; e < nrounds * hp; e += nt) {
    int p, q;
    if (cross) { p = e % hp; q = nbk + (e % hp + e / hp) % nbk; }
    else rr_pair(ns, e / hp, e % hp, &p, &q);
    sched[e] = make_uchar2((unsigned char)p, (unsigned char)q);
  }
  __syncthreads();
  for (int sweep = 0; sweep < max_sweeps; ++sweep) {
    // (the block method asks for a fixed number of inner sweeps with tol2 ~ 0: no test needed, two barriers saved)
    if (tol2 > 1e-29) {
      // convergence: off(A)_F^2 <= tol2 * ||A||_F^2 (padding rows: zero off-diagonals, diagonal excluded)
      double off = 0, tot = 0;
      for (int e = tid; e < ns * ns; e += nt) {
        const int i = e / ns, j = e % ns;
        const cplx a = As[i * LD + j];
        const double v = a.x * a.x + a.y * a.y;
        if (i != j) { off += v; tot += v; }
        else if (fabs(a.x) < 0.5 * JPAD) tot += v;
      }
      for (int o = 16; o > 0; o >>= 1) {
        off += __shfl_xor_sync(0xffffffffu, off, o);
        tot += __shfl_xor_sync(0xffffffffu, tot, o);
      }
      if ((tid & 31) == 0) { red[0][tid >> 5] = off; red[1][tid >> 5] = tot; }
      __syncthreads();
      if (tid == 0) {
        double a = 0, b = 0;
        for (int w = 0; w < nt / 32; ++w) { a += red[0][w]; b += red[1][w]; }
        stop = (a <= tol2 * b) ? 1 : 0;
      }
      __syncthreads();
      if (stop) break;
    }
    for (int r = 0; r < nrounds; ++r) {
      const uchar2* sr = sched + r * hp;
      if (tid < hp) {
        const int p = sr[tid].x, q = sr[tid].y;
        const cplx apq = As[p * LD + q];
        const double a = apq.x * apq.x + apq.y * apq.y;
        double c = 1.0;
        cplx sg = cmake(0.0, 0.0);
        if (a > 0.0) {
          // c = sqrt((1 + |d|/r)/2), sg = sign(d) a_pq / (2 r c), r = sqrt(d^2 + |a_pq|^2): the same rotation as
          // z = sign(d) a_pq / (|d| + r), c = 1/sqrt(1+|z|^2), sg = c z, with two rsqrt and no division
          const double d = 0.5 * (As[q * LD + q].x - As[p * LD + p].x);
          const double ir = rsqrt(fma(d, d, a));
          const double x = fma(0.5 * fabs(d), ir, 0.5);
          const double ix = rsqrt(x);
          c = x * ix;
          const double f = (d >= 0.0 ? 0.5 : -0.5) * ir * ix;
          sg = cmake(apq.x * f, apq.y * f);
        }
        rc[tid] = c;
        rsg[tid] = sg;
      }
      __syncthreads();
      for (int it = tid; it < hp * hp; it += nt) {
        const int l = it % hp, k = it / hp;
        const int pk = sr[k].x, qk = sr[k].y, pl = sr[l].x, ql = sr[l].y;
        const double ck = rc[k], cl = rc[l];
        const cplx sk = rsg[k], sl = rsg[l];
        // right multiply by J_l:  x' = c x - conj(sg) y ,  y' = sg x + c y
        cplx a00 = As[pk * LD + pl], a01 = As[pk * LD + ql], a10 = As[qk * LD + pl], a11 = As[qk * LD + ql];
        cplx v00 = Vs[pk * LD + pl], v01 = Vs[pk * LD + ql], v10 = Vs[qk * LD + pl], v11 = Vs[qk * LD + ql];
        const cplx slc = cconj(sl);
#define ROTR(x, y)                                                              \
        {                                                                       \
          const cplx tx = csub(cscale(cl, x), cmul(slc, y));                    \
          const cplx ty = cadd(cmul(sl, x), cscale(cl, y));                     \
          x = tx; y = ty;                                                       \
        }
        ROTR(a00, a01) ROTR(a10, a11) ROTR(v00, v01) ROTR(v10, v11)
#undef ROTR
        // left multiply by J_k^H:  rp' = c rp - sg rq ,  rq' = conj(sg) rp + c rq
        const cplx skc = cconj(sk);
#define ROTL(x, y)                                                              \
        {                                                                       \
          const cplx tx = csub(cscale(ck, x), cmul(sk, y));                     \
          const cplx ty = cadd(cmul(skc, x), cscale(ck, y));                    \
          x = tx; y = ty;                                                       \
        }
        ROTL(a00, a10) ROTL(a01, a11)
#undef ROTL
        if (k == l) {
          if (sk.x != 0.0 || sk.y != 0.0) { a01 = cmake(0.0, 0.0); a10 = cmake(0.0, 0.0); }
          a00.y = 0.0; a11.y = 0.0;
        }
        As[pk * LD + pl] = a00; As[pk * LD + ql] = a01; As[qk * LD + pl] = a10; As[qk * LD + ql] = a11;
        Vs[pk * LD + pl] = v00; Vs[pk * LD + ql] = v01; Vs[qk * LD + pl] = v10; Vs[qk * LD + ql] = v11;
      }
      __syncthreads();
    }
  }
}

__global__ void __launch_bounds__(JTHREADS) k_jacobi_cta(const cplx* __restrict__ Ap, long ld, int nbk,
                                                        const int2* __restrict__ pairs, cplx* __restrict__ U,
                                                        double* __restrict__ dout, int max_sweeps, double tol2, int cross) {
  extern __shared__ cplx sm[];
  const int ns = 2 * nbk, LD = ns + 1;
  cplx* As = sm;                       // As[i*LD + j] = A[i][j]
  cplx* Vs = As + ns * LD;
  const int tid = threadIdx.x, nt = blockDim.x;
  const int2 pr = pairs[blockIdx.x];
  for (int e = tid; e < ns * ns; e += nt) {
    const int i = e % ns, j = e / ns;    // column-major global read: consecutive threads -> consecutive rows
    const int gi = (i < nbk ? pr.x * nbk + i : pr.y * nbk + i - nbk);
    const int gj = (j < nbk ? pr.x * nbk + j : pr.y * nbk + j - nbk);
    As[i * LD + j] = Ap[(long)gj * ld + gi];
  }
  jac_solve_smem(As, Vs, Vs + ns * LD, nbk, max_sweeps, tol2, cross);
  cplx* Uo = U + (size_t)blockIdx.x * ns * ns;
  for (int e = tid; e < ns * ns; e += nt) {
    const int i = e % ns, j = e / ns;
    Uo[(size_t)j * ns + i] = Vs[i * LD + j];
  }
  if (dout)
    for (int i = tid; i < ns; i += nt) dout[(size_t)blockIdx.x * ns + i] = As[i * LD + i].x;
}

// ------------------------------------------------------------------------------------------------
// block updates: (rows x JSZ x JSZ) complex GEMM tiles on DMMA.  JSZ = pair size (2 blocks of JSZ/2).
// 8 warps, warp tile 32 x 16 MMA layout (4 x 2 m8n8k4 tiles, four real DMMAs per complex product).
// ------------------------------------------------------------------------------------------------
template <int JSZ>
__device__ __forceinline__ int blk_index(int2 pr, int i) {
  return i < JSZ / 2 ? pr.x * (JSZ / 2) + i : pr.y * (JSZ / 2) + i - JSZ / 2;
}

// columns: X[:, IJ] <- X[:, IJ] U   for X = A (z = 0) and X = V (z = 1); rows m0 .. m0+MT-1
template <int JSZ>
__global__ void __launch_bounds__(256) k_jac_col(cplx* __restrict__ Ap, cplx* __restrict__ Vp, long ld, int np,
                                                 const int2* __restrict__ pairs, const cplx* __restrict__ U) {
  constexpr int WN = JSZ / 16, WM = 8 / WN, MT = WM * 32, LDMJ = MT + 2, LDKJ = JSZ + 4;
  extern __shared__ cplx sm[];
  cplx* sP = sm;                   // [k][m]
  cplx* sU = sm + JSZ * LDMJ;      // [n][k]
  cplx* X = blockIdx.z ? Vp : Ap;
  const int2 pr = pairs[blockIdx.y];
  const int m0 = blockIdx.x * MT, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const cplx* Up = U + (size_t)blockIdx.y * JSZ * JSZ;
  for (int e = tid; e < JSZ * MT; e += 256) {
    const int a = e % MT, b = e / MT;                            // m = a, k = b
    sP[b * LDMJ + a] = (m0 + a < np) ? X[(long)blk_index<JSZ>(pr, b) * ld + m0 + a] : cmake(0.0, 0.0);
  }
  for (int e = tid; e < JSZ * JSZ; e += 256) sU[(e / JSZ) * LDKJ + (e % JSZ)] = Up[e];   // n = e / JSZ, k = e % JSZ
  __syncthreads();
  const int wm = warp % WM, wn = warp / WM, fr = lane >> 2, fk = lane & 3;
  double cre[4][2][2], cim[4][2][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 2; ++j) cre[i][j][0] = cre[i][j][1] = cim[i][j][0] = cim[i][j][1] = 0.0;
#pragma unroll 4
  for (int ks = 0; ks < JSZ; ks += 4) {
    cplx af[4], bf[2];
#pragma unroll
    for (int i = 0; i < 4; ++i) af[i] = sP[(ks + fk) * LDMJ + wm * 32 + i * 8 + fr];
#pragma unroll
    for (int j = 0; j < 2; ++j) bf[j] = sU[(wn * 16 + j * 8 + fr) * LDKJ + ks + fk];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const double nai = -af[i].y;
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        dmma(cre[i][j][0], cre[i][j][1], af[i].x, bf[j].x);
        dmma(cim[i][j][0], cim[i][j][1], af[i].x, bf[j].y);
        dmma(cre[i][j][0], cre[i][j][1], nai, bf[j].y);
        dmma(cim[i][j][0], cim[i][j][1], af[i].y, bf[j].x);
      }
    }
  }
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 2; ++j)
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int m = m0 + wm * 32 + i * 8 + fr, n = wn * 16 + j * 8 + 2 * fk + h;
        if (m < np) X[(long)blk_index<JSZ>(pr, n) * ld + m] = cmake(cre[i][j][h], cim[i][j][h]);
      }
}

// rows: A[IJ, :] <- U^H A[IJ, :]   for columns n0 .. n0+NT-1
template <int JSZ>
__global__ void __launch_bounds__(256) k_jac_row(cplx* __restrict__ Ap, long ld, int np, const int2* __restrict__ pairs,
                                                 const cplx* __restrict__ U) {
  constexpr int WM = JSZ / 32, WN = 8 / WM, NT = WN * 16, LDKJ = JSZ + 4;
  extern __shared__ cplx sm[];
  cplx* sU = sm;                   // [m][k]  (U column m)
  cplx* sB = sm + JSZ * LDKJ;      // [n][k]  (A[IJ(k)][n0+n])
  const int2 pr = pairs[blockIdx.y];
  const int n0 = blockIdx.x * NT, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const cplx* Up = U + (size_t)blockIdx.y * JSZ * JSZ;
  for (int e = tid; e < JSZ * JSZ; e += 256) sU[(e / JSZ) * LDKJ + (e % JSZ)] = Up[e];
  for (int e = tid; e < JSZ * NT; e += 256) {
    const int a = e % JSZ, b = e / JSZ;                          // k = a, n = b
    sB[b * LDKJ + a] = (n0 + b < np) ? Ap[(long)(n0 + b) * ld + blk_index<JSZ>(pr, a)] : cmake(0.0, 0.0);
  }
  __syncthreads();
  const int wm = warp % WM, wn = warp / WM, fr = lane >> 2, fk = lane & 3;
  double cre[4][2][2], cim[4][2][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 2; ++j) cre[i][j][0] = cre[i][j][1] = cim[i][j][0] = cim[i][j][1] = 0.0;
#pragma unroll 4
  for (int ks = 0; ks < JSZ; ks += 4) {
    cplx af[4], bf[2];
#pragma unroll
    for (int i = 0; i < 4; ++i) af[i] = sU[(wm * 32 + i * 8 + fr) * LDKJ + ks + fk];
#pragma unroll
    for (int j = 0; j < 2; ++j) bf[j] = sB[(wn * 16 + j * 8 + fr) * LDKJ + ks + fk];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const double nai = -af[i].y;
#pragma unroll
      for (int j = 0; j < 2; ++j) {   // conj(u) a
        dmma(cre[i][j][0], cre[i][j][1], af[i].x, bf[j].x);
        dmma(cim[i][j][0], cim[i][j][1], af[i].x, bf[j].y);
        dmma(cre[i][j][0], cre[i][j][1], af[i].y, bf[j].y);
        dmma(cim[i][j][0], cim[i][j][1], nai, bf[j].x);
      }
    }
  }
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 2; ++j)
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int m = wm * 32 + i * 8 + fr, n = n0 + wn * 16 + j * 8 + 2 * fk + h;
        if (n < np) Ap[(long)n * ld + blk_index<JSZ>(pr, m)] = cmake(cre[i][j][h], cim[i][j][h]);
      }
}

// ------------------------------------------------------------------------------------------------
// small helpers
// ------------------------------------------------------------------------------------------------
__global__ void k_pad_copy(const cplx* __restrict__ A, long lda, int n, cplx* __restrict__ Ap, cplx* __restrict__ Vp, int np) {
  const long e = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (e >= (long)np * np) return;
  const int i = (int)(e % np), j = (int)(e / np);
  cplx v = cmake(0.0, 0.0);
  if (i < n && j < n) {
    // Hermitian part of the input: (A + A^H)/2, diagonal real
    const cplx a = A[(long)j * lda + i], b = A[(long)i * lda + j];
    v = cmake(0.5 * (a.x + b.x), 0.5 * (a.y - b.y));
  } else if (i == j) {
    v = cmake(JPAD, 0.0);
  }
  Ap[e] = v;
  if (Vp) Vp[e] = cmake(i == j ? 1.0 : 0.0, 0.0);
}
__global__ void k_offnorm(const cplx* __restrict__ Ap, int np, int n, double* __restrict__ red) {
  double off = 0, tot = 0;
  for (long e = blockIdx.x * (long)blockDim.x + threadIdx.x; e < (long)np * np; e += (long)gridDim.x * blockDim.x) {
    const int i = (int)(e % np), j = (int)(e / np);
    if (i < n && j < n) {
      const cplx a = Ap[e];
      const double v = a.x * a.x + a.y * a.y;
      tot += v;
      if (i != j) off += v;
    }
  }
  for (int o = 16; o > 0; o >>= 1) {
    off += __shfl_xor_sync(0xffffffffu, off, o);
    tot += __shfl_xor_sync(0xffffffffu, tot, o);
  }
  if ((threadIdx.x & 31) == 0) { atomicAdd(&red[0], off); atomicAdd(&red[1], tot); }
}
__global__ void k_diag(const cplx* __restrict__ Ap, int np, double* __restrict__ d) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < np) d[i] = Ap[(long)i * np + i].x;
}
// rank by counting (ties by index): order[rank] = i, theta[rank] = d[i] for rank < n
__global__ void k_rank(const double* __restrict__ d, int np, int n, int* __restrict__ order, double* __restrict__ theta) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= np) return;
  const double di = d[i];
  int r = 0;
  for (int j = 0; j < np; ++j) {
    const double dj = d[j];
    r += (dj < di || (dj == di && j < i)) ? 1 : 0;
  }
  order[r] = i;
  if (r < n) theta[r] = di;
}
__global__ void k_gather_cols(const cplx* __restrict__ Vp, int np, const int* __restrict__ order, int n,
                              cplx* __restrict__ C, long ldc) {
  const long e = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (e >= (long)n * n) return;
  const int i = (int)(e % n), r = (int)(e / n);
  C[(long)r * ldc + i] = Vp[(long)order[r] * np + i];
}

void ks_eigh_free(EighWs* ws) {
  cudaFree(ws->U); cudaFree(ws->Ap); cudaFree(ws->Vp); cudaFree(ws->diag); cudaFree(ws->red);
  cudaFree(ws->order); cudaFree(ws->pairs); cudaFree(ws->where); cudaFree(ws->Ap2); cudaFree(ws->red_sweeps);
  *ws = EighWs();
}

static int eigh_reserve(EighWs* ws, int np, std::string& err) {
  if (np > ws->cap) {
    cudaFree(ws->U); cudaFree(ws->Ap); cudaFree(ws->Vp); cudaFree(ws->diag); cudaFree(ws->order); cudaFree(ws->Ap2);
    ws->U = ws->Ap = ws->Vp = ws->Ap2 = nullptr; ws->diag = nullptr; ws->order = nullptr; ws->cap = 0;
    const size_t nu = std::max<size_t>((size_t)(np / JS + 1) * JS * JS, (size_t)JS * JS);
    KS_CUDA_CHECK(cudaMalloc(&ws->U, sizeof(cplx) * nu), err);
    KS_CUDA_CHECK(cudaMalloc(&ws->Ap, sizeof(cplx) * (size_t)np * np), err);
    KS_CUDA_CHECK(cudaMalloc(&ws->Vp, sizeof(cplx) * (size_t)np * np), err);
    KS_CUDA_CHECK(cudaMalloc(&ws->Ap2, sizeof(cplx) * (size_t)np * np), err);
    KS_CUDA_CHECK(cudaMalloc(&ws->diag, sizeof(double) * np), err);
    KS_CUDA_CHECK(cudaMalloc(&ws->order, sizeof(int) * np), err);
    ws->cap = np;
  }
  if (!ws->red) KS_CUDA_CHECK(cudaMalloc(&ws->red, 2 * sizeof(double)), err);
  return KS_OK;
}

// ------------------------------------------------------------------------------------------------
// fused two-sided update for 32-wide pairs: one CTA per 32 x 32 tile.
//   blockIdx.y <  npair :  A[IJ_a, IJ_b] <- U_a^H A[IJ_a, IJ_b] U_b     (a = blockIdx.y, b = blockIdx.x)
//   blockIdx.y >= npair :  V[rows, IJ_b] <- V[rows, IJ_b] U_b           (rows = 32 (blockIdx.y - npair) ...)
// The pairs of a round partition the blocks, so the tiles partition A (and V): every tile is read and written
// by exactly one CTA and the update is in place with no intermediate pass through global memory.
// 256 threads as 16 x 16, each owning a 2 x 2 block {ti, ti+16} x {tj, tj+16}; operands row-major with an odd
// leading dimension (33) in shared memory: a half-warp reads one row segment, conflict-free.
// ------------------------------------------------------------------------------------------------
#define JU_LD 33
__device__ __forceinline__ void jac_upd_tile(cplx* sm, cplx* Ap, cplx* Vp, long ld, int npair,
                                             const int2* __restrict__ pairs, const cplx* U, int b, int ay) {
  cplx *sT = sm, *sUa = sm + 32 * JU_LD, *sUb = sm + 64 * JU_LD;
  const int tid = threadIdx.x;
  const bool isA = ay < npair;
  const int2 pb = pairs[b];
  const int2 pa = isA ? pairs[ay] : make_int2(0, 0);
  const int r0 = isA ? 0 : (ay - npair) * 32;
  cplx* X = isA ? Ap : Vp;
  // loads: e -> (i = e % 32 fastest: consecutive rows of a column-major matrix)
  for (int e = tid; e < 32 * 32; e += 256) {
    const int i = e & 31, j = e >> 5;
    const int gi = isA ? blk_index<32>(pa, i) : r0 + i;
    const int gj = blk_index<32>(pb, j);
    sT[i * JU_LD + j] = X[(long)gj * ld + gi];
    sUb[i * JU_LD + j] = U[(size_t)b * 1024 + e];                 // U_b[k = i][j]
    if (isA) sUa[i * JU_LD + j] = U[(size_t)ay * 1024 + e];           // U_a[k = i][col = j]
  }
  __syncthreads();
  const int ti = tid >> 4, tj = tid & 15;
  // P = T U_b
  cplx p00 = cmake(0, 0), p01 = p00, p10 = p00, p11 = p00;
#pragma unroll 8
  for (int k = 0; k < 32; ++k) {
    const cplx a0 = sT[ti * JU_LD + k], a1 = sT[(ti + 16) * JU_LD + k];
    const cplx b0 = sUb[k * JU_LD + tj], b1 = sUb[k * JU_LD + tj + 16];
    p00 = cfma(a0, b0, p00); p01 = cfma(a0, b1, p01);
    p10 = cfma(a1, b0, p10); p11 = cfma(a1, b1, p11);
  }
  __syncthreads();
  sT[ti * JU_LD + tj] = p00; sT[ti * JU_LD + tj + 16] = p01;
  sT[(ti + 16) * JU_LD + tj] = p10; sT[(ti + 16) * JU_LD + tj + 16] = p11;
  __syncthreads();
  if (isA) {
    // T' = U_a^H P :  T'[i][j] = sum_k conj(U_a[k][i]) P[k][j]
    cplx q00 = cmake(0, 0), q01 = q00, q10 = q00, q11 = q00;
#pragma unroll 8
    for (int k = 0; k < 32; ++k) {
      const cplx a0 = cconj(sUa[k * JU_LD + ti]), a1 = cconj(sUa[k * JU_LD + ti + 16]);
      const cplx b0 = sT[k * JU_LD + tj], b1 = sT[k * JU_LD + tj + 16];
      q00 = cfma(a0, b0, q00); q01 = cfma(a0, b1, q01);
      q10 = cfma(a1, b0, q10); q11 = cfma(a1, b1, q11);
    }
    __syncthreads();
    sT[ti * JU_LD + tj] = q00; sT[ti * JU_LD + tj + 16] = q01;
    sT[(ti + 16) * JU_LD + tj] = q10; sT[(ti + 16) * JU_LD + tj + 16] = q11;
    __syncthreads();
  }
  for (int e = tid; e < 32 * 32; e += 256) {
    const int i = e & 31, j = e >> 5;
    const int gi = isA ? blk_index<32>(pa, i) : r0 + i;
    const int gj = blk_index<32>(pb, j);
    X[(long)gj * ld + gi] = sT[i * JU_LD + j];
  }
  // A stays Hermitian under U^H A U: the tile (b, ay) is the conjugate transpose of this one and no CTA computes it
  // (jac_tile_decode deals out the tiles with ay <= b only)
  if (isA && ay != b) {
    for (int e = tid; e < 32 * 32; e += 256) {
      const int j = e & 31, i = e >> 5;          // j fastest: consecutive rows of the mirrored tile
      X[(long)blk_index<32>(pa, i) * ld + blk_index<32>(pb, j)] = cconj(sT[i * JU_LD + j]);
    }
  }
}
// tile t of a round -> (b, ay): first the npair (npair + 1) / 2 tiles of A on or above the block diagonal (ay <= b), then
// the npair * nvt tiles of V (ay = npair + row block)
__device__ __forceinline__ void jac_tile_decode(int t, int npair, int* b, int* ay) {
  const int nA = npair * (npair + 1) / 2;
  if (t >= nA) { t -= nA; *b = t % npair; *ay = npair + t / npair; return; }
  int a = 0;
  while (t >= npair - a) { t -= npair - a; ++a; }
  *ay = a; *b = a + t;
}

__global__ void __launch_bounds__(256) k_jac_upd32(cplx* __restrict__ Ap, cplx* __restrict__ Vp, long ld, int npair,
                                                   const int2* __restrict__ pairs, const cplx* __restrict__ U) {
  extern __shared__ cplx sm[];
  if (blockIdx.y < (unsigned)npair && blockIdx.y > blockIdx.x) return;     // below the block diagonal: written by tile (y, x)'s CTA
  jac_upd_tile(sm, Ap, Vp, ld, npair, pairs, U, blockIdx.x, blockIdx.y);
}

// ------------------------------------------------------------------------------------------------
// The whole solve in ONE cooperative launch (64 < n, padded size < 512): every sweep tests the off-diagonal norm on the
// device and every round is [pair solves] grid.sync [tile updates] grid.sync, with the pairs and tiles dealt over the
// resident CTAs.  Launch by launch the same rounds cost ~37 us each at n = 320 (two launches of a few microseconds of work
// plus one blocking host read per sweep); here a round is two grid barriers plus the pair solve.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_jac_coop32(cplx* Ap, cplx* Vp, int np, int n, int nblk, const int2* __restrict__ pairs_all,
                                                    cplx* U, double* red /* [2 * max_sweeps], zeroed */, int inner, int cross_rounds,
                                                    double tol2, int max_sweeps, int* __restrict__ sweeps_out) {
  cg::grid_group grid = cg::this_grid();
  extern __shared__ cplx sm[];
  const int tid = threadIdx.x, npair = nblk / 2, nbk = JB / 2;
  const int ntile = npair * (npair + 1) / 2 + npair * (np / 32);
  int sweep = 0;
  for (; sweep < max_sweeps; ++sweep) {
    // off(A)_F^2 and ||A||_F^2 of the n x n part, fixed partition of the elements over the grid
    double off = 0, tot = 0;
    for (long e = blockIdx.x * 256L + tid; e < (long)np * np; e += (long)gridDim.x * 256) {
      const int i = (int)(e % np), j = (int)(e / np);
      if (i < n && j < n) {
        const cplx a = Ap[e];
        const double v = a.x * a.x + a.y * a.y;
        tot += v;
        if (i != j) off += v;
      }
    }
    for (int o = 16; o > 0; o >>= 1) {
      off += __shfl_xor_sync(0xffffffffu, off, o);
      tot += __shfl_xor_sync(0xffffffffu, tot, o);
    }
    if ((tid & 31) == 0 && tot != 0.0) { atomicAdd(&red[2 * sweep], off); atomicAdd(&red[2 * sweep + 1], tot); }
    grid.sync();
    const double goff = __ldcg(&red[2 * sweep]), gtot = __ldcg(&red[2 * sweep + 1]);
    if (goff <= tol2 * gtot) break;              // the same two numbers in every CTA: a uniform decision
    for (int r = 0; r < nblk - 1; ++r) {
      const int2* pr = pairs_all + (size_t)r * npair;
      const int cross = (r > 0 && cross_rounds) ? 1 : 0;
      for (int p = blockIdx.x; p < npair; p += gridDim.x) {
        // pair problem p: gather the 32 x 32 block, one inner sweep, rotations to U[p]
        const int ns = 2 * nbk, LD = ns + 1;
        cplx* As = sm;
        cplx* Vs = As + ns * LD;
        const int2 pq = pr[p];
        __syncthreads();
        for (int e = tid; e < ns * ns; e += 256) {
          const int i = e % ns, j = e / ns;
          const int gi = (i < nbk ? pq.x * nbk + i : pq.y * nbk + i - nbk);
          const int gj = (j < nbk ? pq.x * nbk + j : pq.y * nbk + j - nbk);
          As[i * LD + j] = Ap[(long)gj * np + gi];
        }
        jac_solve_smem(As, Vs, Vs + ns * LD, nbk, inner, 1e-30, cross);
        cplx* Uo = U + (size_t)p * ns * ns;
        for (int e = tid; e < ns * ns; e += 256) {
          const int i = e % ns, j = e / ns;
          Uo[(size_t)j * ns + i] = Vs[i * LD + j];
        }
      }
      grid.sync();
      for (int t = blockIdx.x; t < ntile; t += gridDim.x) {
        __syncthreads();
        int tb, tay;
        jac_tile_decode(t, npair, &tb, &tay);
        jac_upd_tile(sm, Ap, Vp, np, npair, pr, U, tb, tay);
      }
      grid.sync();
    }
  }
  if (blockIdx.x == 0 && tid == 0) *sweeps_out = sweep;
}

// ------------------------------------------------------------------------------------------------
// One launch per round (32-wide pairs).  CTAs 0 .. npair-1 solve the pair problems of the NEXT round while
// the other CTAs apply THIS round's rotations U_cur to A and V (jac_upd_tile).  A next-round pair (I', J')
// needs only A'[{I',J'},{I',J'}] = four 16 x 16 blocks of U_a^H A[IJ_a, IJ_b] U_b, where a, b are the pairs of
// this round that hold I', J' (table `where`: block -> (pair index, half)); the solver CTA recomputes those
// blocks itself from the not yet updated A (reads only; the tile CTAs write A in place, so the reads below go
// through a snapshot: see the host loop -- A is double buffered).  The pair solves (tens of microseconds on
// npair SMs) therefore overlap the bulk update instead of serialising with it.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_jac_round32(const cplx* __restrict__ Aold, cplx* __restrict__ Anew, cplx* __restrict__ Vp,
                                                     long ld, int npair, int nvt, const int2* __restrict__ pairs_cur,
                                                     const int2* __restrict__ where_cur, const cplx* __restrict__ Ucur,
                                                     const int2* __restrict__ pairs_next, cplx* __restrict__ Unext,
                                                     int inner, int cross_next) {
  extern __shared__ cplx sm[];
  const int tid = threadIdx.x;
  if ((int)blockIdx.x >= npair) {
    // tile CTA: t -> (b, ay); A tiles read Aold and write Anew, V tiles update Vp in place
    int b, ay;
    jac_tile_decode(blockIdx.x - npair, npair, &b, &ay);
    cplx *sT = sm, *sUa = sm + 32 * JU_LD, *sUb = sm + 64 * JU_LD;
    const bool isA = ay < npair;
    const int2 pb = pairs_cur[b];
    const int2 pa = isA ? pairs_cur[ay] : make_int2(0, 0);
    const int r0 = isA ? 0 : (ay - npair) * 32;
    const cplx* Xin = isA ? Aold : Vp;
    cplx* Xout = isA ? Anew : Vp;
    for (int e = tid; e < 32 * 32; e += 256) {
      const int i = e & 31, j = e >> 5;
      const int gi = isA ? blk_index<32>(pa, i) : r0 + i;
      const int gj = blk_index<32>(pb, j);
      sT[i * JU_LD + j] = Xin[(long)gj * ld + gi];
      sUb[i * JU_LD + j] = Ucur[(size_t)b * 1024 + e];
      if (isA) sUa[i * JU_LD + j] = Ucur[(size_t)ay * 1024 + e];
    }
    __syncthreads();
    const int ti = tid >> 4, tj = tid & 15;
    cplx p00 = cmake(0, 0), p01 = p00, p10 = p00, p11 = p00;
#pragma unroll 8
    for (int k = 0; k < 32; ++k) {
      const cplx a0 = sT[ti * JU_LD + k], a1 = sT[(ti + 16) * JU_LD + k];
      const cplx b0 = sUb[k * JU_LD + tj], b1 = sUb[k * JU_LD + tj + 16];
      p00 = cfma(a0, b0, p00); p01 = cfma(a0, b1, p01);
      p10 = cfma(a1, b0, p10); p11 = cfma(a1, b1, p11);
    }
    __syncthreads();
    sT[ti * JU_LD + tj] = p00; sT[ti * JU_LD + tj + 16] = p01;
    sT[(ti + 16) * JU_LD + tj] = p10; sT[(ti + 16) * JU_LD + tj + 16] = p11;
    __syncthreads();
    if (isA) {
      cplx q00 = cmake(0, 0), q01 = q00, q10 = q00, q11 = q00;
#pragma unroll 8
      for (int k = 0; k < 32; ++k) {
        const cplx a0 = cconj(sUa[k * JU_LD + ti]), a1 = cconj(sUa[k * JU_LD + ti + 16]);
        const cplx b0 = sT[k * JU_LD + tj], b1 = sT[k * JU_LD + tj + 16];
        q00 = cfma(a0, b0, q00); q01 = cfma(a0, b1, q01);
        q10 = cfma(a1, b0, q10); q11 = cfma(a1, b1, q11);
      }
      __syncthreads();
      sT[ti * JU_LD + tj] = q00; sT[ti * JU_LD + tj + 16] = q01;
      sT[(ti + 16) * JU_LD + tj] = q10; sT[(ti + 16) * JU_LD + tj + 16] = q11;
      __syncthreads();
    }
    for (int e = tid; e < 32 * 32; e += 256) {
      const int i = e & 31, j = e >> 5;
      const int gi = isA ? blk_index<32>(pa, i) : r0 + i;
      const int gj = blk_index<32>(pb, j);
      Xout[(long)gj * ld + gi] = sT[i * JU_LD + j];
    }
    if (isA && ay != b) {      // the mirror tile (b, ay) of the Hermitian matrix (no CTA computes it)
      for (int e = tid; e < 32 * 32; e += 256) {
        const int j = e & 31, i = e >> 5;
        Xout[(long)blk_index<32>(pa, i) * ld + blk_index<32>(pb, j)] = cconj(sT[i * JU_LD + j]);
      }
    }
    return;
  }
  // solver CTA for next-round pair p
  const int p = blockIdx.x;
  cplx* As = sm;                       // [32][33]
  cplx* sT = sm + 32 * JU_LD;          // doubles as Vs once As is built
  cplx* sUa = sm + 64 * JU_LD;
  cplx* sUb = sm + 96 * JU_LD;
  const int2 pn = pairs_next[p];
  const int ti = tid >> 4, tj = tid & 15;
  for (int bx = 0; bx < 2; ++bx)
    for (int by = 0; by < 2; ++by) {
      const int2 wa = where_cur[bx ? pn.y : pn.x], wb = where_cur[by ? pn.y : pn.x];
      const int2 pa = pairs_cur[wa.x], pb = pairs_cur[wb.x];
      __syncthreads();
      for (int e = tid; e < 32 * 32; e += 256) {
        const int i = e & 31, j = e >> 5;
        sT[i * JU_LD + j] = Aold[(long)blk_index<32>(pb, j) * ld + blk_index<32>(pa, i)];
        sUa[i * JU_LD + j] = Ucur[(size_t)wa.x * 1024 + e];
        sUb[i * JU_LD + j] = Ucur[(size_t)wb.x * 1024 + e];
      }
      __syncthreads();
      // P (32 x 16) = T U_b[:, half_b] : thread (ti, tj) -> rows ti, ti+16, column tj
      cplx p0 = cmake(0, 0), p1 = p0;
      const int cb = wb.y * 16 + tj;
#pragma unroll 8
      for (int k = 0; k < 32; ++k) {
        const cplx bb = sUb[k * JU_LD + cb];
        p0 = cfma(sT[ti * JU_LD + k], bb, p0);
        p1 = cfma(sT[(ti + 16) * JU_LD + k], bb, p1);
      }
      __syncthreads();
      sT[ti * JU_LD + tj] = p0;
      sT[(ti + 16) * JU_LD + tj] = p1;
      __syncthreads();
      // M (16 x 16) = U_a[:, half_a]^H P : thread (ti, tj) -> element (ti, tj)
      cplx q = cmake(0, 0);
      const int ca = wa.y * 16 + ti;
#pragma unroll 8
      for (int k = 0; k < 32; ++k) q = cfma(cconj(sUa[k * JU_LD + ca]), sT[k * JU_LD + tj], q);
      As[(bx * 16 + ti) * JU_LD + by * 16 + tj] = q;
    }
  __syncthreads();
  // exact Hermitian input for the rotations: real diagonal, upper triangle mirrored
  for (int e = tid; e < 32 * 32; e += 256) {
    const int i = e >> 5, j = e & 31;
    if (i == j) As[i * JU_LD + i].y = 0.0;
  }
  __syncthreads();
  for (int e = tid; e < 32 * 32; e += 256) {
    const int i = e >> 5, j = e & 31;
    if (i < j) {
      const cplx u = As[i * JU_LD + j], l = As[j * JU_LD + i];
      const cplx m = cmake(0.5 * (u.x + l.x), 0.5 * (u.y - l.y));
      As[i * JU_LD + j] = m;
      As[j * JU_LD + i] = cconj(m);
    }
  }
  __syncthreads();
  jac_solve_smem(As, sT, sm + 128 * JU_LD, 16, inner, 1e-30, cross_next);
  cplx* Uo = Unext + (size_t)p * 1024;
  for (int e = tid; e < 1024; e += 256) {
    const int i = e & 31, j = e >> 5;
    Uo[(size_t)j * 32 + i] = sT[i * JU_LD + j];
  }
}

template <int JSZ>
static int block_sweeps(cudaStream_t st, int n, const cplx* A, long lda, EighWs* ws, double tol2, int inner, int* sweeps_out,
                        bool want_sweeps, std::string& err) {
  constexpr int JBK = JSZ / 2;
  constexpr int WNc = JSZ / 16, MT = (8 / WNc) * 32;          // k_jac_col tile rows
  constexpr int WMr = JSZ / 32, NT = (8 / WMr) * 16;          // k_jac_row tile columns
  const size_t smem_cta = sizeof(cplx) * 2 * JS * (JS + 1) + sizeof(cplx) * (JS / 2) + sizeof(double) * (JS / 2) + 2 * (JS - 1) * (JS / 2) + 64;
  const size_t smem_col = sizeof(cplx) * (JSZ * (MT + 2) + JSZ * (JSZ + 4));
  const size_t smem_row = sizeof(cplx) * (JSZ * (JSZ + 4) + NT * (JSZ + 4));
  static std::atomic<bool> opted{false};
  if (!opted) {
    KS_CUDA_CHECK(cudaFuncSetAttribute(k_jac_col<JSZ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_col), err);
    KS_CUDA_CHECK(cudaFuncSetAttribute(k_jac_row<JSZ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_row), err);
    KS_CUDA_CHECK(cudaFuncSetAttribute(k_jac_upd32, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(cplx) * 96 * JU_LD)), err);
    opted = true;
  }
  int nblk = ceil_div(n, JBK);
  nblk += nblk & 1;
  const int np = nblk * JBK, npair = nblk / 2;
  int rc = eigh_reserve(ws, np, err);
  if (rc) return rc;
  ws->np = np;
  if (ws->pairs_nblk != nblk) {
    cudaFree(ws->pairs); ws->pairs = nullptr;
    std::vector<int2> h((size_t)(nblk - 1) * npair);
    for (int r = 0; r < nblk - 1; ++r)
      for (int k = 0; k < npair; ++k) {
        int p, q;
        rr_pair(nblk, r, k, &p, &q);
        h[(size_t)r * npair + k] = make_int2(p, q);
      }
    KS_CUDA_CHECK(cudaMalloc(&ws->pairs, sizeof(int2) * h.size()), err);
    KS_CUDA_CHECK(cudaMemcpy(ws->pairs, h.data(), sizeof(int2) * h.size(), cudaMemcpyHostToDevice), err);
    cudaFree(ws->where); ws->where = nullptr;
    std::vector<int2> wh((size_t)(nblk - 1) * nblk);
    for (int r = 0; r < nblk - 1; ++r)
      for (int k = 0; k < npair; ++k) {
        const int2 pq = h[(size_t)r * npair + k];
        wh[(size_t)r * nblk + pq.x] = make_int2(k, 0);
        wh[(size_t)r * nblk + pq.y] = make_int2(k, 1);
      }
    KS_CUDA_CHECK(cudaMalloc(&ws->where, sizeof(int2) * wh.size()), err);
    KS_CUDA_CHECK(cudaMemcpy(ws->where, wh.data(), sizeof(int2) * wh.size(), cudaMemcpyHostToDevice), err);
    ws->pairs_nblk = nblk;
  }
  k_pad_copy<<<ceil_div((long)np * np, 256), 256, 0, st>>>(A, lda, n, ws->Ap, ws->Vp, np);
  static const bool fused_upd = !(getenv("KSPW_JAC_FUSED") && atoi(getenv("KSPW_JAC_FUSED")) == 0);
  static const bool cross_rounds = !(getenv("KSPW_JAC_CROSS") && atoi(getenv("KSPW_JAC_CROSS")) == 0);
  static const bool one_launch = !(getenv("KSPW_JAC_ROUND") && atoi(getenv("KSPW_JAC_ROUND")) == 0);
  int sweeps = 0;
  static const bool coop_on = !(getenv("KSPW_JAC_COOP") && atoi(getenv("KSPW_JAC_COOP")) == 0);
  if (JSZ == 32 && fused_upd && coop_on && np < 512) {
    // one cooperative launch for the whole solve; the sweep count comes back with the next blocking read of the caller
    const size_t smem_coop = std::max(sizeof(cplx) * 96 * JU_LD, smem_cta);
    static std::atomic<int> coop_ctas{0};
    if (coop_ctas.load() == 0) {
      KS_CUDA_CHECK(cudaFuncSetAttribute(k_jac_coop32, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_coop), err);
      int per_sm = 0, dev = 0, nsm = 0, coop = 0;
      KS_CUDA_CHECK(cudaGetDevice(&dev), err);
      KS_CUDA_CHECK(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev), err);
      KS_CUDA_CHECK(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev), err);
      KS_CUDA_CHECK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_jac_coop32, 256, smem_coop), err);
      coop_ctas.store(coop ? std::max(1, per_sm * nsm) : -1);
    }
    if (coop_ctas.load() > 0) {
      if (!ws->red_sweeps) KS_CUDA_CHECK(cudaMalloc(&ws->red_sweeps, sizeof(double) * 2 * 40 + sizeof(int) * 2), err);
      KS_CUDA_CHECK(cudaMemsetAsync(ws->red_sweeps, 0, sizeof(double) * 2 * 40 + sizeof(int) * 2, st), err);
      int* d_sweeps = (int*)(ws->red_sweeps + 2 * 40);
      const int ntile = npair * (npair + 1) / 2 + npair * (np / 32);
      const int grid = std::min(coop_ctas.load(), std::max(ntile, npair));
      cplx *Ap_ = ws->Ap, *Vp_ = ws->Vp, *U_ = ws->U;
      const int2* pairs_ = ws->pairs;
      double* red_ = ws->red_sweeps;
      int np_ = np, n_ = n, nblk_ = nblk, inner_ = inner, cross_ = cross_rounds ? 1 : 0, maxs = 40;
      double tol2_ = tol2;
      void* args[] = {&Ap_, &Vp_, &np_, &n_, &nblk_, &pairs_, &U_, &red_, &inner_, &cross_, &tol2_, &maxs, &d_sweeps};
      KS_CUDA_CHECK(cudaLaunchCooperativeKernel((void*)k_jac_coop32, dim3(grid), dim3(256), args, smem_coop, st), err);
      if (want_sweeps) {
        KS_CUDA_CHECK(cudaMemcpyAsync(&sweeps, d_sweeps, sizeof(int), cudaMemcpyDeviceToHost, st), err);
        KS_CUDA_CHECK(cudaStreamSynchronize(st), err);
      }
      *sweeps_out = sweeps;
      return sweeps >= 40 ? KS_NOTCONV : KS_OK;
    }
  }
  if (JSZ == 32 && fused_upd && one_launch && np >= 512) {   // below ~500 the solver CTAs' own tile products outweigh the overlap
    // one launch per round: the launch that applies round r also solves the pair problems of round r+1
    const size_t smem_round = sizeof(cplx) * 128 * JU_LD + 2048;
    static std::atomic<bool> opted2{false};
    if (!opted2) {
      KS_CUDA_CHECK(cudaFuncSetAttribute(k_jac_round32, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_round), err);
      opted2 = true;
    }
    const int nr = nblk - 1, nvt = np / 32;
    cplx* Ucur = ws->U;
    cplx* Unext = ws->U + (size_t)npair * 1024;
    cplx *Acur = ws->Ap, *Aalt = ws->Ap2;
    k_jacobi_cta<<<npair, 256, smem_cta, st>>>(Acur, np, JBK, ws->pairs, Ucur, nullptr, inner, 1e-30, 0);
    for (; sweeps < 40; ++sweeps) {
      double h[2];
      KS_CUDA_CHECK(cudaMemsetAsync(ws->red, 0, 2 * sizeof(double), st), err);
      k_offnorm<<<148 * 2, 256, 0, st>>>(Acur, np, n, ws->red);
      KS_CUDA_CHECK(cudaMemcpyAsync(h, ws->red, sizeof h, cudaMemcpyDeviceToHost, st), err);
      KS_CUDA_CHECK(cudaStreamSynchronize(st), err);
      if (h[0] <= tol2 * h[1]) break;
      for (int r = 0; r < nr; ++r) {
        const int rn = (r + 1) % nr;
        k_jac_round32<<<npair + npair * (npair + 1) / 2 + npair * nvt, 256, smem_round, st>>>(
            Acur, Aalt, ws->Vp, np, npair, nvt, ws->pairs + (size_t)r * npair, ws->where + (size_t)r * nblk, Ucur,
            ws->pairs + (size_t)rn * npair, Unext, inner, (rn > 0 && cross_rounds) ? 1 : 0);
        std::swap(Acur, Aalt);
        std::swap(Ucur, Unext);
      }
    }
    if (Acur != ws->Ap) std::swap(ws->Ap, ws->Ap2);   // the caller reads the diagonal from ws->Ap
    KS_CUDA_CHECK(cudaGetLastError(), err);
    *sweeps_out = sweeps;
    return sweeps >= 40 ? KS_NOTCONV : KS_OK;       // the loop left at the cap without passing the off-norm test
  }
  for (; sweeps < 40; ++sweeps) {
    double h[2];
    KS_CUDA_CHECK(cudaMemsetAsync(ws->red, 0, 2 * sizeof(double), st), err);
    k_offnorm<<<148 * 2, 256, 0, st>>>(ws->Ap, np, n, ws->red);
    KS_CUDA_CHECK(cudaMemcpyAsync(h, ws->red, sizeof h, cudaMemcpyDeviceToHost, st), err);
    KS_CUDA_CHECK(cudaStreamSynchronize(st), err);
    if (h[0] <= tol2 * h[1]) break;
    for (int r = 0; r < nblk - 1; ++r) {
      const int2* pr = ws->pairs + (size_t)r * npair;
      k_jacobi_cta<<<npair, JSZ * JSZ / 4, smem_cta, st>>>(ws->Ap, np, JBK, pr, ws->U, nullptr, inner, 1e-30, (r > 0 && cross_rounds) ? 1 : 0);
      if (JSZ == 32 && fused_upd) {
        k_jac_upd32<<<dim3(npair, npair + np / 32), 256, sizeof(cplx) * 96 * JU_LD, st>>>(ws->Ap, ws->Vp, np, npair, pr, ws->U);
      } else {
        k_jac_col<JSZ><<<dim3(ceil_div(np, MT), npair, 2), 256, smem_col, st>>>(ws->Ap, ws->Vp, np, np, pr, ws->U);
        k_jac_row<JSZ><<<dim3(ceil_div(np, NT), npair), 256, smem_row, st>>>(ws->Ap, np, np, pr, ws->U);
      }
    }
  }
  KS_CUDA_CHECK(cudaGetLastError(), err);
  *sweeps_out = sweeps;
  return sweeps >= 40 ? KS_NOTCONV : KS_OK;
}

int ks_eigh_run(cudaStream_t st, int n, cplx* A, long lda, double* theta, cplx* C, long ldc, EighWs* ws,
                int* sweeps_out, std::string& err) {
  if (n <= 0) return KS_OK;
  if (!ws) { err = "ks_eigh: no workspace"; return KS_EINVAL; }
  static std::atomic<bool> opted{false};
  const size_t smem_cta = sizeof(cplx) * 2 * JS * (JS + 1) + sizeof(cplx) * (JS / 2) + sizeof(double) * (JS / 2) + 2 * (JS - 1) * (JS / 2) + 64;
  if (!opted) {
    KS_CUDA_CHECK(cudaFuncSetAttribute(k_jacobi_cta, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_cta), err);
    opted = true;
  }
  const double tol2 = 1e-28;   // off_F <= 1e-14 ||A||_F
  static int inner = 0;        // inner sweeps of the 64x64 pair problems in the block method
  if (!inner) {
    const char* e = getenv("KSPW_JAC_INNER");
    inner = (e && atoi(e) > 0) ? atoi(e) : 1;
  }
  int sweeps = 0;
  if (n <= JS) {
    const int ns = n + (n & 1), nbk = ns / 2;
    int rc = eigh_reserve(ws, JS, err);
    if (rc) return rc;
    if (ws->pairs_nblk != 2) {
      cudaFree(ws->pairs); ws->pairs = nullptr;
      KS_CUDA_CHECK(cudaMalloc(&ws->pairs, sizeof(int2)), err);
      const int2 p01 = make_int2(0, 1);
      KS_CUDA_CHECK(cudaMemcpyAsync(ws->pairs, &p01, sizeof p01, cudaMemcpyHostToDevice, st), err);
      KS_CUDA_CHECK(cudaStreamSynchronize(st), err);
      ws->pairs_nblk = 2;
    }
    k_pad_copy<<<ceil_div((long)ns * ns, 256), 256, 0, st>>>(A, lda, n, ws->Ap, nullptr, ns);
    k_jacobi_cta<<<1, JTHREADS, smem_cta, st>>>(ws->Ap, ns, nbk, ws->pairs, ws->Vp, ws->diag, 40, tol2, 0);
    k_rank<<<ceil_div(ns, 128), 128, 0, st>>>(ws->diag, ns, n, ws->order, theta);
    k_gather_cols<<<ceil_div((long)n * n, 256), 256, 0, st>>>(ws->Vp, ns, ws->order, n, C, ldc);
    KS_CUDA_CHECK(cudaGetLastError(), err);
    if (sweeps_out) *sweeps_out = -1;   // inner sweeps are not reported back
    return KS_OK;
  }
  int rc = 0;
  static int force_blk = -1;
  if (force_blk < 0) {
    const char* e = getenv("KSPW_JAC_PAIR");
    force_blk = e ? atoi(e) : 0;
  }
  const bool use32 = force_blk != 64;   // 32-wide pairs win at every size measured (n = 320 .. 1040)
  if (use32) rc = block_sweeps<32>(st, n, A, lda, ws, tol2, inner, &sweeps, sweeps_out != nullptr, err);
  else rc = block_sweeps<64>(st, n, A, lda, ws, tol2, inner, &sweeps, sweeps_out != nullptr, err);
  if (rc < 0) return rc;
  const int notconv = rc;      // KS_NOTCONV: 40 sweeps did not reach off_F <= 1e-14 ||A||_F; the best pairs are still written
  const int np = ws->np;
  k_diag<<<ceil_div(np, 128), 128, 0, st>>>(ws->Ap, np, ws->diag);
  k_rank<<<ceil_div(np, 128), 128, 0, st>>>(ws->diag, np, n, ws->order, theta);
  k_gather_cols<<<ceil_div((long)n * n, 256), 256, 0, st>>>(ws->Vp, np, ws->order, n, C, ldc);
  KS_CUDA_CHECK(cudaGetLastError(), err);
  if (sweeps_out) *sweeps_out = sweeps;
  if (notconv) err = "ks_eigh: 40 Jacobi sweeps did not reach off_F <= 1e-14 ||A||_F";
  return notconv;
}
