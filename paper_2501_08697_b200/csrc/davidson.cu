// davidson.cu -- block Davidson for the lowest nbands eigenpairs of H psi = eps psi (S = I), or of H psi = eps S psi when
// ks_set_overlap gave an overlap (S V, S X carried next to H V, H X; S-metric projections and CholQR)
// (DESIGN.md §3 listing, steps D0-D9; the paper names the method at PAPER.md L326, L547, L578 and prints
// no listing; the residual p - lambda psi and the preconditioner K are Fig. 10, `vecdiv` L578).
//
// Everything runs on the device; the host only sequences launches and reads nbands residual norms (and
// the Gram-matrix eigenvalues of the orthonormalisation) back per iteration.
//   D0  X = orth(psi0)                        Gram matrix + Cholesky (CholQR2)
//   D1  W = H V                               ks_hpsi_impl on the new block only
//   D2  Hc[:, new] = V^H W_new                DMMA GEMM (K = npw), mirrored to keep Hc Hermitian
//   D3  Hc = C Theta C^H                      Jacobi (eigh.cu)
//   D4  X = V C[:, :nb], HX = W C[:, :nb]     DMMA GEMMs (M = npw)
//   D5  rho_i = ||HX_i - eps_i X_i||, Ekin_i  fused reduction, one CTA per band
//   D6  T_i = K_i (HX_i - eps_i X_i)          Teter-Payne-Allan diagonal polynomial, fused, unconverged only
//   D7  T <- (I - V V^H) T (x2, x1) ; G = T^H T = R^H R (Cholesky with the Gram-Schmidt drop rule) ;
//       T <- T R^{-1} ; twice (CholQR2)
//   D8  V <- [V, T], restart V <- X when m + nu > 2 nb
//   D9  psi <- X, eig, residuals
// On top of the listing, none of which changes the converged pairs: D3 is warm-started in the basis of the
// previous Ritz vectors, converged pairs are locked out of the subspace eigenproblem, and D4 rotates only the
// unconverged bands (all bands before a restart and before returning).
// Difference from the oracle listing (reading C10): the orthonormalisation is Gram/Cholesky based (CholQR2,
// the BLAS-3 form of Gram-Schmidt, same column order and the same kind of drop rule) instead of modified
// Gram-Schmidt.  Both span the same space; the converged pairs agree.
#include "ctx.h"
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdlib>
#include <vector>

#define RED_THREADS 256

__device__ __forceinline__ double block_sum(double v, double* sh) {
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
  __syncthreads();
  double s = 0;
  if (threadIdx.x < 32) {
    s = (threadIdx.x < blockDim.x / 32) ? sh[threadIdx.x] : 0.0;
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  }
  __syncthreads();
  return s;   // valid in thread 0
}

// D5: rho_i = ||HX_i - eps_i X_i||_2 , ekin_i = sum_G g2 |X_i|^2
__global__ void __launch_bounds__(RED_THREADS) k_resid_norms(int npw, const cplx* __restrict__ X, const cplx* __restrict__ SX,
                                                             const cplx* __restrict__ HX,
                                                             const double* __restrict__ eps, const double* __restrict__ g2,
                                                             double* __restrict__ rho, double* __restrict__ ekin,
                                                             const int* __restrict__ list) {
  __shared__ double sh[RED_THREADS / 32];
  const int i = list ? list[blockIdx.x] : blockIdx.x;      // list: only the bands whose Ritz vectors changed
  const cplx* x = X + (size_t)i * npw;
  const cplx* sx = SX + (size_t)i * npw;       // = x when S = I
  const cplx* h = HX + (size_t)i * npw;
  const double e = eps[i];
  double r2 = 0, ek = 0;
  for (int j = threadIdx.x; j < npw; j += blockDim.x) {
    const cplx a = x[j], s = sx[j], b = h[j];
    const double rx = b.x - e * s.x, ry = b.y - e * s.y;
    r2 += rx * rx + ry * ry;
    ek += g2[j] * (a.x * a.x + a.y * a.y);
  }
  r2 = block_sum(r2, sh);
  ek = block_sum(ek, sh);
  if (threadIdx.x == 0) { rho[i] = sqrt(r2); ekin[i] = ek; }
}

// D6: T_u = K_i (HX_i - eps_i X_i), i = idx[u];  K = n(x)/(n(x) + 16 x^4), n = 27 + 18x + 12x^2 + 8x^3,
// x = g2 / max(ekin_i, 1e-3)   (Teter-Payne-Allan; reading C11)
__global__ void k_precond(int npw, int nu, const int* __restrict__ idx, const cplx* __restrict__ X /* S X when S != I */, const cplx* __restrict__ HX,
                          const double* __restrict__ eps, const double* __restrict__ ekin, const double* __restrict__ g2,
                          cplx* __restrict__ T) {
  const int u = blockIdx.y, i = idx[u];
  const double e = eps[i], ek = fmax(ekin[i], 1e-3);
  for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < npw; j += gridDim.x * blockDim.x) {
    const cplx a = X[(size_t)i * npw + j], b = HX[(size_t)i * npw + j];
    const double x = g2[j] / ek;
    const double nx = 27.0 + 18.0 * x + 12.0 * x * x + 8.0 * x * x * x;
    const double K = nx / (nx + 16.0 * x * x * x * x);
    T[(size_t)u * npw + j] = cmake(K * (b.x - e * a.x), K * (b.y - e * a.y));
  }
}

// column 2-norms of a block, then scaling to unit norm
__global__ void __launch_bounds__(RED_THREADS) k_col_norm2(int npw, const cplx* __restrict__ T, double* __restrict__ out) {
  __shared__ double sh[RED_THREADS / 32];
  const cplx* t = T + (size_t)blockIdx.x * npw;
  double s = 0;
  for (int j = threadIdx.x; j < npw; j += blockDim.x) { const cplx a = t[j]; s += a.x * a.x + a.y * a.y; }
  s = block_sum(s, sh);
  if (threadIdx.x == 0) out[blockIdx.x] = s;
}
__global__ void k_col_scale(int npw, cplx* __restrict__ T, const double* __restrict__ n2) {
  const double nn = n2[blockIdx.y];
  const double s = nn > 0.0 ? rsqrt(nn) : 0.0;
  const double sc = nn > 0.0 ? s * (1.5 - 0.5 * nn * s * s) : 0.0;   // one Newton step on rsqrt: full FP64 accuracy
  cplx* t = T + (size_t)blockIdx.y * npw;
  for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < npw; j += gridDim.x * blockDim.x) t[j] = cscale(sc, t[j]);
}

// Drop thresholds of the Cholesky (D7): the Gram matrix is built from columns scaled to unit norm AFTER the projection
// against V, so its remaining diagonal d_j measures the shrinkage against the earlier T columns only.  The listing's
// rule compares the norm after ALL projections with the norm before any: d_j n1_j^2 / n0_j^2 < thr2, i.e. a column is
// dropped when d_j <= thr2 n0_j^2 / n1_j^2 (n0, n1: squared norms before / after the projection against V; a column that
// the projection wiped out, n1 = 0, gets +inf).  n0 == nullptr: no projection happened, plain thr2.
__global__ void k_drop_thresholds(int nu, const double* __restrict__ n0, const double* __restrict__ n1, double thr2,
                                  double* __restrict__ thrv) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= nu) return;
  if (!n0) { thrv[j] = thr2; return; }
  thrv[j] = (n1[j] > 0.0) ? thr2 * n0[j] / n1[j] : __longlong_as_double(0x7ff0000000000000LL);
}

// small-matrix helpers (column-major)
__global__ void k_negate(long n, cplx* __restrict__ a) {
  const long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (i < n) a[i] = cmake(-a[i].x, -a[i].y);
}
__global__ void k_set_diag(int m, long ld, cplx* __restrict__ H, const double* __restrict__ d) {
  const long e = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (e >= (long)m * m) return;
  const int i = (int)(e % m), j = (int)(e / m);
  H[(long)j * ld + i] = cmake(i == j ? d[i] : 0.0, 0.0);
}
// after the new columns Hc[0:m1, m0:m1] were written: mirror them into the rows and symmetrise the corner
// upper_only: the corner holds its upper triangle only (ks_gemm_hn with herm_r0): the lower one is its mirror image
__global__ void k_mirror(int m0, int m1, long ld, cplx* __restrict__ H, int upper_only) {
  const long e = blockIdx.x * (long)blockDim.x + threadIdx.x;
  const int nn = m1 - m0;
  if (e >= (long)m1 * nn) return;
  const int i = (int)(e % m1), j = m0 + (int)(e / m1);
  if (i < m0) {
    const cplx a = H[(long)j * ld + i];
    H[(long)i * ld + j] = cconj(a);
  } else if (upper_only) {
    if (i <= j) {
      cplx a = H[(long)j * ld + i];          // row i, column j: the computed triangle
      if (i == j) a.y = 0.0;
      H[(long)j * ld + i] = a;
      H[(long)i * ld + j] = cconj(a);
    }
  } else if (i <= j) {
    const cplx a = H[(long)j * ld + i], b = H[(long)i * ld + j];
    const cplx s = cmake(0.5 * (a.x + b.x), (i == j) ? 0.0 : 0.5 * (a.y - b.y));
    H[(long)j * ld + i] = s;
    H[(long)i * ld + j] = cconj(s);
  }
}
// D3 warm start: the subspace matrix in the basis Q = diag(C_prev, I).  Fills the leading mp x mp block with
// diag(theta_prev) and copies the trailing (m-mp) x (m-mp) corner of Hc; the mp x (m-mp) border comes from a GEMM.
__global__ void k_build_hrot(int mp, int m, const cplx* __restrict__ Hc, long ldh, const double* __restrict__ thp,
                             cplx* __restrict__ Hr) {
  const long e = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (e >= (long)m * m) return;
  const int i = (int)(e % m), j = (int)(e / m);
  if (i < mp && j < mp) Hr[e] = cmake(i == j ? thp[i] : 0.0, 0.0);
  else if (i >= mp && j >= mp) Hr[e] = Hc[(long)j * ldh + i];
}
__global__ void k_mirror_border(int mp, int m, cplx* __restrict__ Hr) {   // Hr[j][i] = conj(Hr[i][j]), i < mp <= j
  const long e = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (e >= (long)mp * (m - mp)) return;
  const int i = (int)(e % mp), j = mp + (int)(e / mp);
  Hr[(long)i * m + j] = cconj(Hr[(long)j * m + i]);
}
// D3 with locking: converged Ritz pairs (rows L of the rotated matrix, coupling <= their residual <= tol) are taken
// out of the eigenproblem; the solver sees Hr[F, F] only.
__global__ void k_gather_sub(int mf, const int* __restrict__ F, const cplx* __restrict__ Hr, int m, cplx* __restrict__ Hs) {
  const long e = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (e >= (long)mf * mf) return;
  const int i = (int)(e % mf), j = (int)(e / mf);
  Hs[e] = Hr[(long)F[j] * m + F[i]];
}
// merge the locked values thp[L[.]] (ascending) and the solved ones thf[.] (ascending): position of every entry in
// the merged ascending list (ties: locked first), theta[pos] and src[pos] = (1, e) locked / (0, j) free
__global__ void k_merge_order(int nl, const int* __restrict__ L, const double* __restrict__ thp, int mf,
                              const double* __restrict__ thf, double* __restrict__ theta, int2* __restrict__ src) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= nl + mf) return;
  if (e < nl) {
    const double v = thp[L[e]];
    int lo = 0, hi = mf;                       // number of free values < v
    while (lo < hi) { const int mid = (lo + hi) >> 1; if (thf[mid] < v) lo = mid + 1; else hi = mid; }
    theta[e + lo] = v;
    src[e + lo] = make_int2(1, e);
  } else {
    const int j = e - nl;
    const double v = thf[j];
    int lo = 0, hi = nl;                       // number of locked values <= v
    while (lo < hi) { const int mid = (lo + hi) >> 1; if (thp[L[mid]] <= v) lo = mid + 1; else hi = mid; }
    theta[j + lo] = v;
    src[j + lo] = make_int2(0, j);
  }
}
// eigenvectors in the rotated basis: column pos = unit vector of a locked row, or the free solution scattered to rows F
__global__ void k_assemble_cprime(int m, const int2* __restrict__ src, const int* __restrict__ L, const int* __restrict__ rowF,
                                  const cplx* __restrict__ Cf, long ldf, cplx* __restrict__ Cpr) {
  const long e = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (e >= (long)m * m) return;
  const int row = (int)(e % m), pos = (int)(e / m);
  const int2 s = src[pos];
  cplx v = cmake(0.0, 0.0);
  if (s.x) { if (L[s.y] == row) v = cmake(1.0, 0.0); }
  else { const int r = rowF[row]; if (r >= 0) v = Cf[(long)s.y * ldf + r]; }
  Cpr[e] = v;
}
__global__ void k_set_identity(int m, long ld, cplx* __restrict__ C) {
  const long e = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (e >= (long)m * m) return;
  const int i = (int)(e % m), j = (int)(e / m);
  C[(long)j * ld + i] = cmake(i == j ? 1.0 : 0.0, 0.0);
}
// D4 on the unconverged bands only: Cg[:, j] = C[:, idx[j]]  and  X[idx[j]][:] = T[j][:]
__global__ void k_gather_cols_idx(int m, int nu, const cplx* __restrict__ C, long ldc, const int* __restrict__ idx,
                                  cplx* __restrict__ Cg) {
  const long e = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (e >= (long)m * nu) return;
  const int i = (int)(e % m), j = (int)(e / m);
  Cg[e] = C[(long)idx[j] * ldc + i];
}
__global__ void k_scatter_bands(int npw, int nu, const int* __restrict__ idx, const cplx* __restrict__ T, cplx* __restrict__ X) {
  const int j = blockIdx.y;
  cplx* dst = X + (size_t)idx[j] * npw;
  const cplx* src = T + (size_t)j * npw;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < npw; i += gridDim.x * blockDim.x) dst[i] = src[i];
}
__global__ void k_copy_mat(int m, int n, const cplx* __restrict__ a, long lda, cplx* __restrict__ b, long ldb) {
  const long e = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (e >= (long)m * n) return;
  const int i = (int)(e % m), j = (int)(e / m);
  b[(long)j * ldb + i] = a[(long)j * lda + i];
}
// ------------------------------------------------------------------------------------------------
// Orthonormalisation through the Gram matrix G = T^H T (unit diagonal): right-looking Cholesky
// G = R^H R in one CTA, DROPPING column j when its remaining diagonal d_j = ||t_j - proj||^2 / ||t_j||^2
// falls below thr (the Gram-Schmidt drop rule of the listing, in the same column order), then
// M = R_kept^{-1} embedded in nu x nk, so that T M is orthonormal.  G is column-major; its upper
// triangle is overwritten by R (R[j][k] at G[k*ld + j], k >= j).
// ------------------------------------------------------------------------------------------------
#define CHOL_THREADS 1024
__global__ void __launch_bounds__(CHOL_THREADS) k_chol_drop(int n, cplx* __restrict__ G, long ld, const double* __restrict__ thrv,
                                                          int* __restrict__ kept, int* __restrict__ nk_out) {
  extern __shared__ cplx rowj[];          // [n] current row of R
  __shared__ double s_inv;
  __shared__ int s_keep;
  const int tid = threadIdx.x, nt = blockDim.x;
  for (int j = 0; j < n; ++j) {
    if (tid == 0) {
      const double d = G[(long)j * ld + j].x;
      s_keep = (d > thrv[j]) ? 1 : 0;
      if (s_keep) {
        const double r = sqrt(d);
        G[(long)j * ld + j] = cmake(r, 0.0);
        s_inv = 1.0 / r;
      } else {
        G[(long)j * ld + j] = cmake(0.0, 0.0);   // marks the column as dropped
      }
    }
    __syncthreads();
    const int keep = s_keep;
    const double inv = s_inv;
    __syncthreads();                       // everyone has read s_keep / s_inv before thread 0 writes the next column's
    if (!keep) continue;
    for (int k = j + 1 + tid; k < n; k += nt) {
      const cplx v = cscale(inv, G[(long)k * ld + j]);
      G[(long)k * ld + j] = v;
      rowj[k] = v;
    }
    __syncthreads();
    // trailing update of the upper triangle: G[i][k] -= conj(R[j][i]) R[j][k],  j < i <= k
    const int m = n - j - 1;
    for (long e = tid; e < (long)m * m; e += nt) {
      const int i = j + 1 + (int)(e % m), k = j + 1 + (int)(e / m);
      if (i <= k) {
        const cplx a = rowj[i], b = rowj[k];
        cplx g = G[(long)k * ld + i];
        g.x -= a.x * b.x + a.y * b.y;
        g.y -= a.x * b.y - a.y * b.x;
        G[(long)k * ld + i] = g;
      }
    }
    __syncthreads();
  }
  if (tid == 0) {
    int nk = 0;
    for (int j = 0; j < n; ++j)
      if (G[(long)j * ld + j].x > 0.0) kept[nk++] = j;
    *nk_out = nk;
  }
}

// Blocked form of the same factorisation (same column order, same drop rule, sums in a different order): panels of
// CB columns; per panel one CTA factors the CB x CB diagonal block in shared memory, a row-panel kernel solves
// R11^H R12 = G12 (one thread per trailing column), and a tiled rank-CB update takes R12^H R12 off the trailing
// upper triangle.  A dropped column's row of R is zero, so the later panels skip it by arithmetic.  n = 520 (cfg 3):
// 17 ms in the single-CTA kernel above, 51 short launches here.
#define CB 32
__global__ void __launch_bounds__(CB * CB) k_chol_diag(int n, int j0, cplx* __restrict__ G, long ld, const double* __restrict__ thrv) {
  __shared__ cplx D[CB][CB + 1];
  __shared__ double s_inv;
  __shared__ int s_keep;
  const int i = threadIdx.x % CB, k = threadIdx.x / CB;     // D[i][k] = element (row j0+i, column j0+k), i <= k
  const int w = min(CB, n - j0);
  const bool in = (i <= k && k < w);
  if (in) D[i][k] = G[(long)(j0 + k) * ld + j0 + i];
  __syncthreads();
  for (int j = 0; j < w; ++j) {
    if (threadIdx.x == 0) {
      const double d = D[j][j].x;
      s_keep = (d > thrv[j0 + j]) ? 1 : 0;
      const double r = s_keep ? sqrt(d) : 0.0;
      D[j][j] = cmake(r, 0.0);                 // 0 marks the column as dropped
      s_inv = s_keep ? 1.0 / r : 0.0;          // a dropped column's row of R becomes zero
    }
    __syncthreads();
    if (i == j && k > j && k < w) D[j][k] = cscale(s_inv, D[j][k]);
    __syncthreads();
    if (in && i > j) {
      const cplx a = D[j][i], b = D[j][k];
      D[i][k].x -= a.x * b.x + a.y * b.y;
      D[i][k].y -= a.x * b.y - a.y * b.x;
    }
    __syncthreads();
  }
  if (in) G[(long)(j0 + k) * ld + j0 + i] = D[i][k];
}
// R12 = R11^{-H} G12: thread per trailing column k, forward substitution in registers (right-looking)
__global__ void __launch_bounds__(64) k_chol_trsm(int n, int j0, cplx* __restrict__ G, long ld) {
  __shared__ cplx R[CB][CB + 1];
  const int w = min(CB, n - j0);
  for (int e = threadIdx.x; e < CB * CB; e += blockDim.x) {
    const int i = e % CB, k = e / CB;
    R[i][k] = (i <= k && k < w) ? G[(long)(j0 + k) * ld + j0 + i] : cmake(0.0, 0.0);
  }
  __syncthreads();
  const int k = j0 + w + blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  cplx* col = G + (long)k * ld + j0;
  cplx x[CB];
#pragma unroll
  for (int j = 0; j < CB; ++j) x[j] = (j < w) ? col[j] : cmake(0.0, 0.0);
#pragma unroll
  for (int j = 0; j < CB; ++j) {
    const double d = R[j][j].x;
    const double inv = (d > 0.0) ? 1.0 / d : 0.0;
    x[j] = cscale(inv, x[j]);
#pragma unroll
    for (int q = j + 1; q < CB; ++q) {        // x_q -= conj(R[j][q]) x_j
      const cplx r = R[j][q];
      x[q].x -= r.x * x[j].x + r.y * x[j].y;
      x[q].y -= r.x * x[j].y - r.y * x[j].x;
    }
  }
#pragma unroll
  for (int j = 0; j < CB; ++j)
    if (j < w) col[j] = x[j];
}
// trailing update of the upper triangle: G[i][k] -= sum_j conj(R[j][i]) R[j][k], j in the panel, j0+w <= i <= k < n
__global__ void __launch_bounds__(256) k_chol_update(int n, int j0, cplx* __restrict__ G, long ld) {
  if (blockIdx.x > blockIdx.y) return;        // tiles below the diagonal
  __shared__ cplx Pi[CB][CB + 1], Pk[CB][CB + 1];          // [column in tile][panel row]
  const int w = min(CB, n - j0), t0 = j0 + w;
  const int i0 = t0 + blockIdx.x * CB, k0 = t0 + blockIdx.y * CB;
  for (int e = threadIdx.x; e < CB * CB; e += 256) {
    const int j = e % CB, cidx = e / CB;
    Pi[cidx][j] = (j < w && i0 + cidx < n) ? G[(long)(i0 + cidx) * ld + j0 + j] : cmake(0.0, 0.0);
    Pk[cidx][j] = (j < w && k0 + cidx < n) ? G[(long)(k0 + cidx) * ld + j0 + j] : cmake(0.0, 0.0);
  }
  __syncthreads();
  const int ii = threadIdx.x % CB;
  for (int kk = threadIdx.x / CB; kk < CB; kk += 256 / CB) {
    const int gi = i0 + ii, gk = k0 + kk;
    if (gi > gk || gk >= n) continue;
    double sr = 0.0, si = 0.0;
#pragma unroll
    for (int j = 0; j < CB; ++j) {
      const cplx a = Pi[ii][j], b = Pk[kk][j];
      sr += a.x * b.x + a.y * b.y;
      si += a.x * b.y - a.y * b.x;
    }
    cplx* g = G + (long)gk * ld + gi;
    g->x -= sr;
    g->y -= si;
  }
}
__global__ void __launch_bounds__(256) k_chol_kept(int n, const cplx* __restrict__ G, long ld, int* __restrict__ kept,
                                                  int* __restrict__ nk_out) {
  extern __shared__ int s_flag[];
  for (int j = threadIdx.x; j < n; j += blockDim.x) s_flag[j] = G[(long)j * ld + j].x > 0.0;
  __syncthreads();
  if (threadIdx.x == 0) {
    int nk = 0;
    for (int j = 0; j < n; ++j)
      if (s_flag[j]) kept[nk++] = j;
    *nk_out = nk;
  }
}
static void chol_drop_blocked(cudaStream_t st, int n, cplx* G, long ld, const double* thrv, int* kept, int* nk_out) {
  for (int j0 = 0; j0 < n; j0 += CB) {
    k_chol_diag<<<1, CB * CB, 0, st>>>(n, j0, G, ld, thrv);
    const int m = n - j0 - CB;                 // trailing columns
    if (m <= 0) break;
    k_chol_trsm<<<ceil_div(m, 64), 64, 0, st>>>(n, j0, G, ld);
    const int nt = ceil_div(m, CB);
    k_chol_update<<<dim3(nt, nt), 256, 0, st>>>(n, j0, G, ld);
  }
  k_chol_kept<<<1, 256, sizeof(int) * n, st>>>(n, G, ld, kept, nk_out);
}

#define TRINV_MAX 3584     // columns k_trinv can hold: 4 warps x TRINV_MAX x 16 B = 224 KB of shared memory
// one warp per kept column jj: x = R_kept^{-1} e_jj by back substitution; M[:, jj] (nu rows) = scatter(x)
__global__ void __launch_bounds__(128) k_trinv(int nu, const cplx* __restrict__ R, long ld, const int* __restrict__ kept, int nk,
                                               cplx* __restrict__ M, long ldm) {
  extern __shared__ cplx xs[];            // [4][nk]
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int jj = blockIdx.x * 4 + w;
  if (jj >= nk) return;
  cplx* x = xs + (size_t)w * nk;
  for (int i = lane; i < nu; i += 32) M[(long)jj * ldm + i] = cmake(0.0, 0.0);
  for (int ii = jj; ii >= 0; --ii) {
    const int i = kept[ii];
    double sr = 0, si = 0;
    for (int kk = ii + 1 + lane; kk <= jj; kk += 32) {
      const cplx r = R[(long)kept[kk] * ld + i], v = x[kk];
      sr += r.x * v.x - r.y * v.y;
      si += r.x * v.y + r.y * v.x;
    }
    for (int o = 16; o > 0; o >>= 1) {
      sr += __shfl_xor_sync(0xffffffffu, sr, o);
      si += __shfl_xor_sync(0xffffffffu, si, o);
    }
    if (lane == 0) {
      const double rii = R[(long)i * ld + i].x;
      x[ii] = cmake(((ii == jj ? 1.0 : 0.0) - sr) / rii, -si / rii);
    }
    __syncwarp();
  }
  __syncwarp();
  for (int ii = lane; ii <= jj; ii += 32) M[(long)jj * ldm + kept[ii]] = x[ii];
}

// ------------------------------------------------------------------------------------------------
void ks_davidson_free(DavidsonWs* w) {
  cudaFree(w->V); cudaFree(w->W); cudaFree(w->X); cudaFree(w->HX); cudaFree(w->T);
  cudaFree(w->Hc); cudaFree(w->Cm); cudaFree(w->Hwork); cudaFree(w->S); cudaFree(w->Us);
  cudaFree(w->SV); cudaFree(w->SX); cudaFree(w->ST);
  cudaFree(w->Cp); cudaFree(w->Cq); cudaFree(w->thp); cudaFree(w->act); cudaFree(w->thf); cudaFree(w->lst); cudaFree(w->src);
  cudaFree(w->theta); cudaFree(w->rho); cudaFree(w->ekin); cudaFree(w->lam); cudaFree(w->lam0); cudaFree(w->thr); cudaFree(w->idx);
  *w = DavidsonWs();
}

static int reserve(ks_ctx* c, int nb) {
  DavidsonWs& w = c->dws;
  if (nb <= w.nb_cap) return KS_OK;
  ks_davidson_free(&w);
  const size_t npw = c->P.npw, vb = sizeof(cplx) * npw;
  const size_t m = 2 * (size_t)nb;
  KS_CUDA_CHECK(cudaMalloc(&w.V, vb * m), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.W, vb * m), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.X, vb * nb), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.HX, vb * nb), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.T, vb * nb), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.Hc, sizeof(cplx) * m * m), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.Cm, sizeof(cplx) * m * m), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.Hwork, sizeof(cplx) * m * m), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.Cp, sizeof(cplx) * m * m), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.Cq, sizeof(cplx) * m * m), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.thp, sizeof(double) * m), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.thf, sizeof(double) * m), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.lst, sizeof(int) * 3 * m), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.src, sizeof(int2) * m), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.S, sizeof(cplx) * m * nb), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.Us, sizeof(cplx) * (size_t)nb * nb), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.theta, sizeof(double) * m), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.rho, sizeof(double) * nb), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.ekin, sizeof(double) * nb), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.lam, sizeof(double) * nb), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.lam0, sizeof(double) * nb), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.thr, sizeof(double) * nb), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.idx, sizeof(int) * (nb + 1)), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.act, sizeof(int) * nb), c->err);
  w.nb_cap = nb;
  return KS_OK;
}

struct Phase {   // optional per-phase timing (KSPW_PROFILE=1; 2 also prints one line per iteration): adds a stream sync per phase
  bool on = false;
  int level = 0;
  double mark[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  void iter_line(int it, int m, int nu, int nk, int nl, int sweeps) {     // per-iteration phase times since the last line
    if (level < 2) return;
    fprintf(stderr, "dav it %d m %d nu %d nk %d locked %d sweeps %d | hpsi %.3f proj %.3f eigh %.3f rot %.3f resid %.3f orth %.3f ms\n", it, m, nu, nk,
            nl, sweeps, acc[0] - mark[0], acc[1] - mark[1], acc[2] - mark[2], acc[3] - mark[3], acc[4] - mark[4], acc[5] - mark[5]);
    for (int i = 0; i < 8; ++i) mark[i] = acc[i];
  }
  cudaEvent_t a = nullptr, b = nullptr;
  cudaStream_t st = 0;
  double* acc = nullptr;
  void init(cudaStream_t s, double* ms) {
    const char* e = getenv("KSPW_PROFILE");
    on = e && atoi(e) > 0;
    level = e ? atoi(e) : 0;
    st = s; acc = ms;
    for (int i = 0; i < 8; ++i) ms[i] = 0;
    if (on) { cudaEventCreate(&a); cudaEventCreate(&b); }
  }
  void begin() { if (on) cudaEventRecord(a, st); }
  void end(int ph) {
    if (!on) return;
    cudaEventRecord(b, st);
    cudaEventSynchronize(b);
    float ms = 0;
    cudaEventElapsedTime(&ms, a, b);
    acc[ph] += ms;
  }
  void done() { if (on) { cudaEventDestroy(a); cudaEventDestroy(b); } }
};
enum { PH_HPSI = 0, PH_PROJ = 1, PH_EIGH = 2, PH_ROT = 3, PH_RESID = 4, PH_ORTH = 5, PH_TOTAL = 6 };

#define RC(x) do { int rc__ = (x); if (rc__ < 0) return rc__; } while (0)

// One pass of D7/D0:  src (npw x nu) -> dst (npw x nk): optional projection against V[0:m] (nproj times),
// unit column norms, Gram matrix G, Cholesky G = R^H R dropping columns whose remaining squared norm is
// below 1e-12 of the original (norm ratio 1e-6; the Gram form cannot resolve the listing's 1e-10),
// dst = src R_kept^{-1}.
// Generalised problem (c->d_Q set): inner products in the S metric -- coefficients (S V)^H src, Gram matrix
// src^H (S src) with S src from ks_spsi, and sdst = (S src) R_kept^{-1} = S dst comes out alongside dst.
static int orth_pass(ks_ctx* c, cplx* src, int nu, cplx* dst, int m, int nproj_pass, int* nk_out, Phase& ph,
                     cplx* sdst = nullptr) {
  const bool gen = c->d_Q != nullptr;
  DavidsonWs& w = c->dws;
  const int npw = c->P.npw;
  cudaStream_t st = c->stream;
  ph.begin();
  const bool projected = nproj_pass > 0 && m > 0;
  if (projected) k_col_norm2<<<nu, RED_THREADS, 0, st>>>(npw, src, w.lam0);
  for (int p = 0; p < nproj_pass && m > 0; ++p) {
    RC(ks_gemm_hn(st, m, nu, npw, gen ? w.SV : w.V, npw, src, npw, w.S, m, &c->gws, c->err));
    k_negate<<<ceil_div((long)m * nu, 256), 256, 0, st>>>((long)m * nu, w.S);
    RC(ks_gemm_nn(st, npw, nu, m, w.V, npw, w.S, m, src, npw, 1, c->err));
  }
  k_col_norm2<<<nu, RED_THREADS, 0, st>>>(npw, src, w.lam);
  k_drop_thresholds<<<ceil_div(nu, 128), 128, 0, st>>>(nu, projected ? w.lam0 : nullptr, w.lam, 1e-12, w.thr);
  k_col_scale<<<dim3(std::max(1, std::min(64, ceil_div(npw, 1024))), nu), 256, 0, st>>>(npw, src, w.lam);
  if (gen) RC(ks_spsi_impl(c, src, w.ST, nu));
  // the Cholesky kernels read the upper triangle of the Gram matrix only: the tiles below its diagonal are not computed
  static const bool herm_on = !(getenv("KSPW_HERM_SKIP") && atoi(getenv("KSPW_HERM_SKIP")) == 0);
  RC(ks_gemm_hn(st, nu, nu, npw, src, npw, gen ? w.ST : src, npw, w.Us, nu, &c->gws, c->err, herm_on ? 0 : -1));
  ph.end(PH_ORTH);
  ph.begin();
  static std::atomic<bool> opted{false};
  if (!opted.load()) {
    KS_CUDA_CHECK(cudaFuncSetAttribute(k_trinv, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(cplx) * 4 * TRINV_MAX)), c->err);
    opted.store(true);
  }
  if (nu > TRINV_MAX) { c->err = "ks_davidson: more than 3584 columns in one orthonormalisation block"; return KS_EINVAL; }
  static const bool chol_blocked = !(getenv("KSPW_CHOL_BLOCKED") && atoi(getenv("KSPW_CHOL_BLOCKED")) == 0);
  if (chol_blocked) chol_drop_blocked(st, nu, w.Us, nu, w.thr, w.idx, w.idx + nu);
  else k_chol_drop<<<1, CHOL_THREADS, sizeof(cplx) * nu, st>>>(nu, w.Us, nu, w.thr, w.idx, w.idx + nu);
  int nk = 0;
  KS_CUDA_CHECK(cudaMemcpyAsync(&nk, w.idx + nu, sizeof(int), cudaMemcpyDeviceToHost, st), c->err);
  KS_CUDA_CHECK(cudaStreamSynchronize(st), c->err);
  *nk_out = nk;
  if (nk == 0) { ph.end(PH_EIGH); return KS_OK; }
  k_trinv<<<ceil_div(nk, 4), 128, sizeof(cplx) * 4 * nk, st>>>(nu, w.Us, nu, w.idx, nk, w.S, nu);
  ph.end(PH_EIGH);
  ph.begin();
  // no column dropped: w.S = R^{-1} is upper triangular, column n ends at row n (with drops it ends at row kept[n] >= n,
  // known on the device only: the full product then)
  const int btri = (herm_on && nk == nu) ? 0 : -1;
  RC(ks_gemm_nn(st, npw, nk, nu, src, npw, w.S, nu, dst, npw, 0, c->err, btri));
  if (gen && sdst) RC(ks_gemm_nn(st, npw, nk, nu, w.ST, npw, w.S, nu, sdst, npw, 0, c->err, btri));
  ph.end(PH_ORTH);
  return KS_OK;
}

int ks_davidson_impl(ks_ctx* c, cplx* psi, double* eig, int nb, double tol, int max_iter, double* resid, int* iters_out,
                     long long* nhpsi_out) {
  if (!c) return KS_EINVAL;
  const int npw = c->P.npw;
  if (!psi || !eig || nb < 1 || nb > npw || !(tol > 0) || max_iter < 0) { c->err = "ks_davidson: bad argument"; return KS_EINVAL; }
  RC(reserve(c, nb));
  DavidsonWs& w = c->dws;
  cudaStream_t st = c->stream;
  const size_t vb = sizeof(cplx) * (size_t)npw;
  // generalised problem H x = eps S x (ks_set_overlap): S V, S X are carried next to H V, H X
  const bool gen = c->d_Q != nullptr;
  if (gen && w.s_cap < nb) {
    cudaFree(w.SV); cudaFree(w.SX); cudaFree(w.ST);
    w.SV = w.SX = w.ST = nullptr; w.s_cap = 0;
    KS_CUDA_CHECK(cudaMalloc(&w.SV, vb * 2 * nb), c->err);
    KS_CUDA_CHECK(cudaMalloc(&w.SX, vb * nb), c->err);
    KS_CUDA_CHECK(cudaMalloc(&w.ST, vb * nb), c->err);
    w.s_cap = nb;
  }
  const long ldh = 2L * nb;
  Phase ph, tot;
  ph.init(st, c->prof_ms);
  double dummy[8];
  tot.init(st, dummy);
  tot.acc = c->prof_ms;
  tot.begin();

  // D0: orthonormalise the start block (two canonical passes)
  int nk = 0;
  KS_CUDA_CHECK(cudaMemcpyAsync(w.T, psi, vb * nb, cudaMemcpyDeviceToDevice, st), c->err);
  RC(orth_pass(c, w.T, nb, w.X, 0, 0, &nk, ph));
  if (nk < nb) { c->err = "ks_davidson: start block is rank deficient"; return KS_EINVAL; }
  RC(orth_pass(c, w.X, nb, w.V, 0, 0, &nk, ph, gen ? w.SV : nullptr));
  if (nk < nb) { c->err = "ks_davidson: start block is rank deficient"; return KS_EINVAL; }
  // D1-D4: initial Rayleigh-Ritz
  ph.begin();
  RC(ks_hpsi_impl(c, w.V, w.W, nb));
  ph.end(PH_HPSI);
  long long nh = nb;
  ph.begin();
  RC(ks_gemm_hn(st, nb, nb, npw, w.V, npw, w.W, npw, w.Hwork, nb, &c->gws, c->err));
  ph.end(PH_PROJ);
  ph.begin();
  RC(ks_eigh_run(st, nb, w.Hwork, nb, w.theta, w.Cm, ldh, &c->ews, nullptr, c->err));
  ph.end(PH_EIGH);
  ph.begin();
  RC(ks_gemm_nn(st, npw, nb, nb, w.V, npw, w.Cm, ldh, w.X, npw, 0, c->err));
  RC(ks_gemm_nn(st, npw, nb, nb, w.W, npw, w.Cm, ldh, w.HX, npw, 0, c->err));
  if (gen) RC(ks_gemm_nn(st, npw, nb, nb, w.SV, npw, w.Cm, ldh, w.SX, npw, 0, c->err));
  KS_CUDA_CHECK(cudaMemcpyAsync(w.V, w.X, vb * nb, cudaMemcpyDeviceToDevice, st), c->err);
  KS_CUDA_CHECK(cudaMemcpyAsync(w.W, w.HX, vb * nb, cudaMemcpyDeviceToDevice, st), c->err);
  if (gen) KS_CUDA_CHECK(cudaMemcpyAsync(w.SV, w.SX, vb * nb, cudaMemcpyDeviceToDevice, st), c->err);
  k_set_diag<<<ceil_div((long)nb * nb, 256), 256, 0, st>>>(nb, ldh, w.Hc, w.theta);
  ph.end(PH_ROT);
  // warm start of the subspace eigensolver (KSPW_WARM=0 switches it off): V = X, so C_prev = I, theta_prev = eps
  static const bool warm = !(getenv("KSPW_WARM") && atoi(getenv("KSPW_WARM")) == 0);
  int mp = nb;
  if (warm) {
    k_set_identity<<<ceil_div((long)nb * nb, 256), 256, 0, st>>>(nb, ldh, w.Cp);
    KS_CUDA_CHECK(cudaMemcpyAsync(w.thp, w.theta, sizeof(double) * nb, cudaMemcpyDeviceToDevice, st), c->err);
  }
  int m = nb, it = 0, status = KS_NOTCONV;
  std::vector<double> rho(nb);
  std::vector<int> idx(nb);
  // D4 rotates only the bands that are still unconverged (KSPW_ACTIVE_ROT=0: all bands every iteration, as the
  // listing says); `stale` = some converged band's X, HX are older than the last eigensolve.
  // locking (KSPW_LOCK=0 switches it off; needs the warm start's rotated basis)
  static const bool lock_env = !(getenv("KSPW_LOCK") && atoi(getenv("KSPW_LOCK")) == 0);
  const bool lock_on = lock_env && warm;
  std::vector<int> lockL, lockF, rowF;
  static const bool active_rot = !(getenv("KSPW_ACTIVE_ROT") && atoi(getenv("KSPW_ACTIVE_ROT")) == 0);
  bool stale = false;
  int n_changed = -1;        // bands whose X, HX changed since the last residual evaluation (-1: all)
  int dbg_nl = 0, dbg_sw = 0;
  auto rotate_all = [&]() -> int {
    const cplx* Cl = warm ? w.Cp : w.Cm;      // eigenvectors of the last eigensolve (after the end-of-iteration swap)
    RC(ks_gemm_nn(st, npw, nb, m, w.V, npw, Cl, ldh, w.X, npw, 0, c->err));
    RC(ks_gemm_nn(st, npw, nb, m, w.W, npw, Cl, ldh, w.HX, npw, 0, c->err));
    if (gen) RC(ks_gemm_nn(st, npw, nb, m, w.SV, npw, Cl, ldh, w.SX, npw, 0, c->err));
    stale = false;
    n_changed = -1;
    return KS_OK;
  };
  // leaving the loop with no correction left (every one was dropped as dependent): D9 must return X, HX, rho that
  // belong to the last eigensolve, so the bands that were not rotated since they converged are brought up to date
  auto refresh_if_stale = [&]() -> int {
    if (!stale) return KS_OK;
    RC(rotate_all());
    k_resid_norms<<<nb, RED_THREADS, 0, st>>>(npw, w.X, gen ? w.SX : w.X, w.HX, w.theta, c->P.d_g2, w.rho, w.ekin, nullptr);
    return KS_OK;
  };
  for (;;) {
    // D5
    ph.begin();
    // a locked band keeps its Ritz value and its (not rotated) vectors, so its residual cannot have changed: after an
    // active-band rotation only the nu rotated bands (w.act) are re-evaluated
    if (n_changed >= 0 && lock_on)
      k_resid_norms<<<n_changed, RED_THREADS, 0, st>>>(npw, w.X, gen ? w.SX : w.X, w.HX, w.theta, c->P.d_g2, w.rho, w.ekin, w.act);
    else
      k_resid_norms<<<nb, RED_THREADS, 0, st>>>(npw, w.X, gen ? w.SX : w.X, w.HX, w.theta, c->P.d_g2, w.rho, w.ekin, nullptr);
    KS_CUDA_CHECK(cudaMemcpyAsync(rho.data(), w.rho, sizeof(double) * nb, cudaMemcpyDeviceToHost, st), c->err);
    KS_CUDA_CHECK(cudaStreamSynchronize(st), c->err);
    ph.end(PH_RESID);
    int nu = 0;
    for (int i = 0; i < nb; ++i)
      if (!(rho[i] <= tol)) idx[nu++] = i;
    if ((nu == 0 || it >= max_iter) && stale) {
      // the Ritz vectors of the bands that were already converged have not been rotated since they converged:
      // bring every band up to date and look at all the residuals again before stopping
      ph.begin();
      RC(rotate_all());
      ph.end(PH_ROT);
      continue;
    }
    if (nu == 0) { status = KS_OK; break; }
    if (it >= max_iter) break;
    // D8 (restart)
    if (m + nu > 2 * nb) {
      if (stale) { ph.begin(); RC(rotate_all()); ph.end(PH_ROT); }
      KS_CUDA_CHECK(cudaMemcpyAsync(w.V, w.X, vb * nb, cudaMemcpyDeviceToDevice, st), c->err);
      KS_CUDA_CHECK(cudaMemcpyAsync(w.W, w.HX, vb * nb, cudaMemcpyDeviceToDevice, st), c->err);
      if (gen) KS_CUDA_CHECK(cudaMemcpyAsync(w.SV, w.SX, vb * nb, cudaMemcpyDeviceToDevice, st), c->err);
      k_set_diag<<<ceil_div((long)nb * nb, 256), 256, 0, st>>>(nb, ldh, w.Hc, w.theta);
      m = nb;
      if (warm) {   // V = X again: C_prev = I; theta_prev[0:nb] already holds eps
        k_set_identity<<<ceil_div((long)nb * nb, 256), 256, 0, st>>>(nb, ldh, w.Cp);
        mp = nb;
      }
    }
    // D6
    ph.begin();
    KS_CUDA_CHECK(cudaMemcpyAsync(w.idx, idx.data(), sizeof(int) * nu, cudaMemcpyHostToDevice, st), c->err);
    k_precond<<<dim3(std::max(1, std::min(64, ceil_div(npw, 1024))), nu), 256, 0, st>>>(npw, nu, w.idx, gen ? w.SX : w.X, w.HX, w.theta, w.ekin,
                                                                                      c->P.d_g2, w.T);
    ph.end(PH_RESID);
    // D7: two passes; the result lands in V[m : m+nk]
    cplx* Vnew = w.V + (size_t)m * npw;
    static const int nproj_first = (getenv("KSPW_ORTH_PROJ") && atoi(getenv("KSPW_ORTH_PROJ")) > 0) ? atoi(getenv("KSPW_ORTH_PROJ")) : 1;   // + one projection in the second pass = the listing's "twice"
    RC(orth_pass(c, w.T, nu, Vnew, m, nproj_first, &nk, ph));
    if (nk == 0) { RC(refresh_if_stale()); break; }
    int nk2 = 0;
    RC(orth_pass(c, Vnew, nk, w.T, m, 1, &nk2, ph, gen ? w.SV + (size_t)m * npw : nullptr));   // S V_new comes out of the second pass
    if (nk2 == 0) { RC(refresh_if_stale()); break; }
    nk = nk2;
    KS_CUDA_CHECK(cudaMemcpyAsync(Vnew, w.T, vb * nk, cudaMemcpyDeviceToDevice, st), c->err);
    // D1
    cplx* Wnew = w.W + (size_t)m * npw;
    ph.begin();
    RC(ks_hpsi_impl(c, Vnew, Wnew, nk));
    ph.end(PH_HPSI);
    nh += nk;
    // D2
    ph.begin();
    const int m1 = m + nk;
    // the corner V_new^H (H V_new) is Hermitian: only the tiles that reach its upper triangle are computed, k_mirror fills the rest
    static const bool herm_hc = !(getenv("KSPW_HERM_SKIP") && atoi(getenv("KSPW_HERM_SKIP")) == 0);
    RC(ks_gemm_hn(st, m1, nk, npw, w.V, npw, Wnew, npw, w.Hc + (size_t)m * ldh, ldh, &c->gws, c->err, herm_hc ? m : -1));
    k_mirror<<<ceil_div((long)m1 * nk, 256), 256, 0, st>>>(m, m1, ldh, w.Hc, herm_hc ? 1 : 0);
    ph.end(PH_PROJ);
    m = m1;
    // D3
    ph.begin();
    if (!warm) {
      k_copy_mat<<<ceil_div((long)m * m, 256), 256, 0, st>>>(m, m, w.Hc, ldh, w.Hwork, m);
      RC(ks_eigh_run(st, m, w.Hwork, m, w.theta, w.Cm, ldh, &c->ews, nullptr, c->err));
    } else {
      // Q = diag(C_prev, I):  Q^H Hc Q = [diag(theta_prev), C_prev^H B; (.)^H, D] -- already diagonal except for the
      // border that couples the new directions, so the Jacobi sweeps start close to convergence.
      k_build_hrot<<<ceil_div((long)m * m, 256), 256, 0, st>>>(mp, m, w.Hc, ldh, w.thp, w.Hwork);
      RC(ks_gemm_hn(st, mp, m - mp, mp, w.Cp, ldh, w.Hc + (size_t)mp * ldh, ldh, w.Hwork + (size_t)mp * m, m, &c->gws, c->err));
      k_mirror_border<<<ceil_div((long)mp * (m - mp), 256), 256, 0, st>>>(mp, m, w.Hwork);
      // locking: bands whose residual passed the test at this iteration's step 2 keep their Ritz pair; their rows
      // (index < nb <= mp: the leading diagonal block) are deflated from the eigenproblem
      int nl = 0;
      if (lock_on) {
        lockL.clear(); lockF.clear(); rowF.assign(m, -1);
        for (int i = 0; i < m; ++i) {
          if (i < nb && rho[i] <= tol) lockL.push_back(i);
          else { rowF[i] = (int)lockF.size(); lockF.push_back(i); }
        }
        nl = (int)lockL.size();
      }
      int sw = 0;
      // the sweep count costs a blocking read: only when somebody looks at it
      static const bool dbg_sweeps = getenv("KSPW_DEBUG_SWEEPS") != nullptr;
      int* swp = (dbg_sweeps || ph.level >= 2) ? &sw : nullptr;
      dbg_nl = nl;
      if (nl == 0) {
        RC(ks_eigh_run(st, m, w.Hwork, m, w.theta, w.Cq, ldh, &c->ews, swp, c->err));
        if (dbg_sweeps) fprintf(stderr, "it %d m %d nk %d sweeps %d\n", it, m, nk, sw);
        // C = Q C'
        RC(ks_gemm_nn(st, mp, m, mp, w.Cp, ldh, w.Cq, ldh, w.Cm, ldh, 0, c->err));
        k_copy_mat<<<ceil_div((long)(m - mp) * m, 256), 256, 0, st>>>(m - mp, m, w.Cq + mp, ldh, w.Cm + mp, ldh);
      } else {
        const int mf = m - nl;
        int *dL = w.lst, *dF = w.lst + 2 * nb, *dR = w.lst + 4 * nb;
        KS_CUDA_CHECK(cudaMemcpyAsync(dL, lockL.data(), sizeof(int) * nl, cudaMemcpyHostToDevice, st), c->err);
        KS_CUDA_CHECK(cudaMemcpyAsync(dF, lockF.data(), sizeof(int) * mf, cudaMemcpyHostToDevice, st), c->err);
        KS_CUDA_CHECK(cudaMemcpyAsync(dR, rowF.data(), sizeof(int) * m, cudaMemcpyHostToDevice, st), c->err);
        // Hc is not needed again before the next D2, but it must survive: the gathered problem goes to Cm (free until D4)
        k_gather_sub<<<ceil_div((long)mf * mf, 256), 256, 0, st>>>(mf, dF, w.Hwork, m, w.Cm);
        RC(ks_eigh_run(st, mf, w.Cm, mf, w.thf, w.Cq, ldh, &c->ews, swp, c->err));
        if (dbg_sweeps) fprintf(stderr, "it %d m %d nk %d locked %d sweeps %d\n", it, m, nk, nl, sw);
        k_merge_order<<<ceil_div(m, 128), 128, 0, st>>>(nl, dL, w.thp, mf, w.thf, w.theta, w.src);
        k_assemble_cprime<<<ceil_div((long)m * m, 256), 256, 0, st>>>(m, w.src, dL, dR, w.Cq, ldh, w.Hwork);
        // C = Q C'  (C' in Hwork, leading dimension m)
        RC(ks_gemm_nn(st, mp, m, mp, w.Cp, ldh, w.Hwork, m, w.Cm, ldh, 0, c->err));
        k_copy_mat<<<ceil_div((long)(m - mp) * m, 256), 256, 0, st>>>(m - mp, m, w.Hwork + mp, m, w.Cm + mp, ldh);
      }
      KS_CUDA_CHECK(cudaMemcpyAsync(w.thp, w.theta, sizeof(double) * m, cudaMemcpyDeviceToDevice, st), c->err);
      dbg_sw = sw;
    }
    ph.end(PH_EIGH);
    // D4
    ph.begin();
    if (!active_rot || 2 * nu > nb) {
      RC(ks_gemm_nn(st, npw, nb, m, w.V, npw, w.Cm, ldh, w.X, npw, 0, c->err));
      RC(ks_gemm_nn(st, npw, nb, m, w.W, npw, w.Cm, ldh, w.HX, npw, 0, c->err));
      if (gen) RC(ks_gemm_nn(st, npw, nb, m, w.SV, npw, w.Cm, ldh, w.SX, npw, 0, c->err));
      stale = false;
      n_changed = -1;
    } else {
      // idx[0:nu] = the bands that were unconverged at this iteration's D5
      KS_CUDA_CHECK(cudaMemcpyAsync(w.act, idx.data(), sizeof(int) * nu, cudaMemcpyHostToDevice, st), c->err);
      k_gather_cols_idx<<<ceil_div((long)m * nu, 256), 256, 0, st>>>(m, nu, w.Cm, ldh, w.act, w.S);
      const dim3 gs(std::max(1, std::min(32, ceil_div(npw, 2048))), nu);
      RC(ks_gemm_nn(st, npw, nu, m, w.V, npw, w.S, m, w.T, npw, 0, c->err));
      k_scatter_bands<<<gs, 256, 0, st>>>(npw, nu, w.act, w.T, w.X);
      RC(ks_gemm_nn(st, npw, nu, m, w.W, npw, w.S, m, w.T, npw, 0, c->err));
      k_scatter_bands<<<gs, 256, 0, st>>>(npw, nu, w.act, w.T, w.HX);
      if (gen) {
        RC(ks_gemm_nn(st, npw, nu, m, w.SV, npw, w.S, m, w.T, npw, 0, c->err));
        k_scatter_bands<<<gs, 256, 0, st>>>(npw, nu, w.act, w.T, w.SX);
      }
      stale = true;
      n_changed = nu;
    }
    ph.end(PH_ROT);
    if (warm) { std::swap(w.Cm, w.Cp); mp = m; }   // C of this iteration is C_prev of the next
    ph.iter_line(it, m, nu, nk, dbg_nl, dbg_sw);
    ++it;
  }
  // D9
  KS_CUDA_CHECK(cudaMemcpyAsync(psi, w.X, vb * nb, cudaMemcpyDeviceToDevice, st), c->err);
  KS_CUDA_CHECK(cudaMemcpyAsync(eig, w.theta, sizeof(double) * nb, cudaMemcpyDeviceToDevice, st), c->err);
  if (resid) KS_CUDA_CHECK(cudaMemcpyAsync(resid, w.rho, sizeof(double) * nb, cudaMemcpyDeviceToDevice, st), c->err);
  KS_CUDA_CHECK(cudaStreamSynchronize(st), c->err);
  tot.end(PH_TOTAL);
  ph.done();
  tot.done();
  if (iters_out) *iters_out = it;
  if (nhpsi_out) *nhpsi_out = nh;
  return status;
}
