// fft.cuh -- register DFT codelets and the two-stage shared-memory line FFT used by the H*psi kernels.
//
// A line of length n = R1*R2 is transformed in place in shared memory by two passes of register
// codelets dft<R> (R in {1,2,3,4,5,6,8,9,12,16,18,...}, built recursively from radix 2/3/4/5
// butterflies with compile-time twiddle indices into a __constant__ table):
//
//   type A (natural -> transposed):  input  x[j],  j = j1*R2 + j2
//        stage 1, item j2:  v[j1] = x[j1*R2+j2];  dft<R1>;  v[k1] *= w_n^{j2 k1};  store at k1*R2+j2
//        stage 2, item k1:  v[j2] = x[k1*R2+j2];  dft<R2>;                         store at k1*R2+k2
//        position p = k1*R2 + k2 then holds X[k1 + R1*k2]            (perm(p) = p/R2 + R1*(p%R2))
//   type B (transposed -> natural):  input at position k1*R2+k2 holds x[k1 + R1*k2]
//        stage 1, item k1:  v[k2] = x[k1*R2+k2];  dft<R2>;  v[q2] *= w_n^{k1 q2};  store at k1*R2+q2
//        stage 2, item q2:  v[k1] = x[k1*R2+q2];  dft<R1>;                         store at q1*R2+q2
//        position q1*R2 + q2 = natural index q = q2 + R2*q1.
//
// A followed (after a pointwise multiply in the transposed order) by B needs no reordering pass;
// the H*psi kernels keep every intermediate in "position" order and V(r) is stored permuted once.
// Sign convention: SIGN=+1 is e^{+2 pi i jk/n} (G -> r, Eq. 31), SIGN=-1 is e^{-...}
// (r -> G, Eq. 36).  Twiddles are FP64 cos/sin evaluated once on the host (no fast-math).
#pragma once
#include "common.cuh"

#define KS_WTAB 720  // 2^4 * 3^2 * 5: every supported codelet radix divides it

__constant__ double2 c_wtab[KS_WTAB];  // e^{+2 pi i t/720}; filled by ks_fft_init_constants() (one TU includes this header)

// multiply by w_R^{SIGN*idx}; idx is a compile-time constant after unrolling, so the quarter-turn
// cases fold away and the table entry becomes a constant-bank operand.
template <int R, int SIGN>
__device__ __forceinline__ cplx mul_w(cplx a, int idx) {
  idx %= R;
  if (idx == 0) return a;
  if (4 * idx == R) return SIGN > 0 ? cmake(-a.y, a.x) : cmake(a.y, -a.x);      // * (+-i)
  if (2 * idx == R) return cmake(-a.x, -a.y);
  if (4 * idx == 3 * R) return SIGN > 0 ? cmake(a.y, -a.x) : cmake(-a.y, a.x);  // * (-+i)
  const double2 w = c_wtab[idx * (KS_WTAB / R)];
  const double wy = SIGN > 0 ? w.y : -w.y;
  return cmake(a.x * w.x - a.y * wy, a.x * wy + a.y * w.x);
}

template <int R>
struct radix_split {  // R = P * M, P the butterfly applied last
  static constexpr int P = (R % 4 == 0) ? 4 : (R % 2 == 0) ? 2 : (R % 3 == 0) ? 3 : (R % 5 == 0) ? 5 : R;
  static constexpr int M = R / P;
};

template <int R, int SIGN>
__device__ __forceinline__ void dft(cplx (&x)[R]) {
  if constexpr (R == 1) {
    return;
  } else if constexpr (R == 2) {
    const cplx a = x[0], b = x[1];
    x[0] = cadd(a, b);
    x[1] = csub(a, b);
  } else if constexpr (R == 3) {
    constexpr double S3 = 0.86602540378443864676372317075294;  // sin(2 pi/3)
    const cplx a = x[0], s = cadd(x[1], x[2]), d = csub(x[1], x[2]);
    const cplx m = cmake(a.x - 0.5 * s.x, a.y - 0.5 * s.y);
    const double tx = SIGN * S3 * d.y, ty = SIGN * S3 * d.x;  // (+-i) S3 d = (-+S3 d.y, +-S3 d.x)
    x[0] = cadd(a, s);
    x[1] = cmake(m.x - tx, m.y + ty);
    x[2] = cmake(m.x + tx, m.y - ty);
  } else if constexpr (R == 4) {
    const cplx a = cadd(x[0], x[2]), b = csub(x[0], x[2]);
    const cplx c = cadd(x[1], x[3]), d = csub(x[1], x[3]);
    const cplx id = SIGN > 0 ? cmake(-d.y, d.x) : cmake(d.y, -d.x);  // (+-i) d
    x[0] = cadd(a, c);
    x[1] = cadd(b, id);
    x[2] = csub(a, c);
    x[3] = csub(b, id);
  } else if constexpr (R == 5) {
    constexpr double C1 = 0.30901699437494742410229341718282, C2 = -0.80901699437494742410229341718282;
    constexpr double S1 = 0.95105651629515357211643933337938, S2 = 0.58778525229247312916870595463907;
    const cplx a = x[0];
    const cplx s1 = cadd(x[1], x[4]), d1 = csub(x[1], x[4]);
    const cplx s2 = cadd(x[2], x[3]), d2 = csub(x[2], x[3]);
    const cplx m1 = cmake(a.x + C1 * s1.x + C2 * s2.x, a.y + C1 * s1.y + C2 * s2.y);
    const cplx m2 = cmake(a.x + C2 * s1.x + C1 * s2.x, a.y + C2 * s1.y + C1 * s2.y);
    const cplx t1 = cmake(S1 * d1.x + S2 * d2.x, S1 * d1.y + S2 * d2.y);
    const cplx t2 = cmake(S2 * d1.x - S1 * d2.x, S2 * d1.y - S1 * d2.y);
    const cplx i1 = SIGN > 0 ? cmake(-t1.y, t1.x) : cmake(t1.y, -t1.x);
    const cplx i2 = SIGN > 0 ? cmake(-t2.y, t2.x) : cmake(t2.y, -t2.x);
    x[0] = cmake(a.x + s1.x + s2.x, a.y + s1.y + s2.y);
    x[1] = cadd(m1, i1);
    x[4] = csub(m1, i1);
    x[2] = cadd(m2, i2);
    x[3] = csub(m2, i2);
  } else {
    constexpr int P = radix_split<R>::P, M = radix_split<R>::M;
    static_assert(P < R, "unsupported prime radix");
    cplx y[P][M];
#pragma unroll
    for (int r = 0; r < P; ++r) {
      cplx sub[M];
#pragma unroll
      for (int j = 0; j < M; ++j) sub[j] = x[r + P * j];
      dft<M, SIGN>(sub);
#pragma unroll
      for (int k = 0; k < M; ++k) y[r][k] = sub[k];
    }
#pragma unroll
    for (int k = 0; k < M; ++k) {
      cplx t[P];
#pragma unroll
      for (int r = 0; r < P; ++r) t[r] = mul_w<R, SIGN>(y[r][k], r * k);
      dft<P, SIGN>(t);
#pragma unroll
      for (int q = 0; q < P; ++q) x[k + M * q] = t[q];
    }
  }
}

// n = R1 * R2 factorisation of every supported line length
template <int N> struct fac;
#define KS_FAC(N_, A_, B_) template <> struct fac<N_> { static constexpr int R1 = A_, R2 = B_; };
KS_FAC(16, 4, 4)   KS_FAC(18, 6, 3)   KS_FAC(24, 6, 4)   KS_FAC(32, 8, 4)   KS_FAC(36, 6, 6)
KS_FAC(48, 8, 6)   KS_FAC(54, 9, 6)   KS_FAC(64, 8, 8)   KS_FAC(72, 9, 8)   KS_FAC(96, 12, 8)
KS_FAC(128, 16, 8) KS_FAC(144, 12, 12) KS_FAC(192, 16, 12) KS_FAC(256, 16, 16) KS_FAC(288, 18, 16)
// lengths with a factor 5 (grids with factors 2, 3, 5 are what plane-wave codes pick)
KS_FAC(20, 5, 4)   KS_FAC(40, 8, 5)   KS_FAC(60, 10, 6)  KS_FAC(80, 10, 8)  KS_FAC(100, 10, 10) KS_FAC(120, 12, 10)
#undef KS_FAC

// twiddle w_n^{SIGN*t} from a shared-memory table tw[t] = e^{+2 pi i t/n}
template <int SIGN>
__device__ __forceinline__ cplx mul_tw(cplx a, const cplx* tw, int t) {
  const cplx w = tw[t];
  const double wy = SIGN > 0 ? w.y : -w.y;
  return cmake(a.x * w.x - a.y * wy, a.x * wy + a.y * w.x);
}

// ---- type A ------------------------------------------------------------------------------------
// line: pointer to element 0 of the line; es: element stride (in cplx); tw: n-entry table (smem).
template <int N, int SIGN, class F = fac<N>>
__device__ __forceinline__ void lineA_stage1(cplx* line, int es, int j2, const cplx* tw) {
  constexpr int R1 = F::R1, R2 = F::R2;
  cplx v[R1];
#pragma unroll
  for (int j1 = 0; j1 < R1; ++j1) v[j1] = line[(j1 * R2 + j2) * es];
  dft<R1, SIGN>(v);
#pragma unroll
  for (int k1 = 0; k1 < R1; ++k1) line[(k1 * R2 + j2) * es] = (k1 == 0) ? v[0] : mul_tw<SIGN>(v[k1], tw, j2 * k1);
}
template <int N, int SIGN, class F = fac<N>>
__device__ __forceinline__ void lineA_stage2(cplx* line, int es, int k1) {
  constexpr int R2 = F::R2;
  cplx v[R2];
#pragma unroll
  for (int j2 = 0; j2 < R2; ++j2) v[j2] = line[(k1 * R2 + j2) * es];
  dft<R2, SIGN>(v);
#pragma unroll
  for (int k2 = 0; k2 < R2; ++k2) line[(k1 * R2 + k2) * es] = v[k2];
}
// ---- type B ------------------------------------------------------------------------------------
template <int N, int SIGN, class F = fac<N>>
__device__ __forceinline__ void lineB_stage1(cplx* line, int es, int k1, const cplx* tw) {
  constexpr int R2 = F::R2;
  cplx v[R2];
#pragma unroll
  for (int k2 = 0; k2 < R2; ++k2) v[k2] = line[(k1 * R2 + k2) * es];
  dft<R2, SIGN>(v);
#pragma unroll
  for (int q2 = 0; q2 < R2; ++q2) line[(k1 * R2 + q2) * es] = (q2 == 0) ? v[0] : mul_tw<SIGN>(v[q2], tw, k1 * q2);
}
template <int N, int SIGN, class F = fac<N>>
__device__ __forceinline__ void lineB_stage2(cplx* line, int es, int q2) {
  constexpr int R1 = F::R1, R2 = F::R2;
  cplx v[R1];
#pragma unroll
  for (int k1 = 0; k1 < R1; ++k1) v[k1] = line[(k1 * R2 + q2) * es];
  dft<R1, SIGN>(v);
#pragma unroll
  for (int q1 = 0; q1 < R1; ++q1) line[(q1 * R2 + q2) * es] = v[q1];
}

// z axis of the yz kernels (sticks): the split whose line counts fill 256 threads best.  96 = 16 x 6: a plane of S <= 41
// sticks gives S*6 <= 246 DFT-16 lines (one round) and S*16 DFT-6 lines, instead of S*8 DFT-12 (two rounds, the second
// nearly empty) and S*12 DFT-8.
template <int N> struct facz : fac<N> {};
template <> struct facz<96> { static constexpr int R1 = 16, R2 = 6; };

// position -> natural index of a type-A output (host + device)
__host__ __device__ __forceinline__ int perm_index(int p, int R1, int R2) { return p / R2 + R1 * (p % R2); }
