// oracle/kso.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct CPU statement (FP64) of what the hot path computes:
// the plane-wave Kohn-Sham Hamiltonian apply and the block-Davidson iteration around it
// (arxiv 2501.08697 = /root/reference/PAPER.md, §III.A, §III.B, §II.A.1).
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// call it.  It shares no code, header, table or helper with the CUDA path under
// paper_2501_08697_b200/csrc/.  No BLAS / FFTW / LAPACK: own recursive mixed-radix FFT, explicit
// H(G,G'), cyclic Hermitian Jacobi, block Davidson.  OpenMP over bands / rows only.
//
// Units: Rydberg atomic units (reading C1): kinetic term |k+G|^2, no 1/2.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"):
//   kso_fft3d      direct O(n^2) DFT on tiny grids, delta <-> plane wave, Parseval, numpy.fft
//   kso_pw_list    counts vs Omega ecut^{3/2}/(6 pi^2), inversion symmetry, numpy enumeration
//   kso_hpsi       explicit H(G,G') (kso_explicit_h), V=1 identity, shift theorem, Hermiticity,
//                  single-projector closed form, p-triplet closed form
//   kso_explicit_h rebuilt entry by entry in numpy from Eq. 32 / Eq. 4 in the test
//   kso_jacobi     2x2 closed form, A C = C Theta, C^H C = I, numpy.linalg.eigvalsh
//   kso_density    numpy.fft.ifftn on the scattered grid, Parseval sum, one plane wave -> constant, two plane
//                  waves -> 2 + 2 cos((G1-G2).r) closed form, non-negativity
//   kso_chebyshev  U p(Lambda) U^H chi from numpy.linalg.eigh of the explicit H with p evaluated by
//                  numpy.polynomial.chebyshev.chebval; T_n = cos(n arccos x) on an eigenvector; sqrt(Fermi-Dirac)
//   kso_spsi / kso_explicit_s / kso_davidson_s   S rebuilt from its definition in numpy, scipy.linalg.eigh(H, S),
//                  X^H S X = I, Q = 0 reduces to kso_davidson
//   kso_cg         V=0: sorted |k+G|^2 exactly; numpy.linalg.eigvalsh of the explicit H; kso_davidson's eigenvalues;
//                  residuals, orthonormality, Ritz values above the exact ones
//   kso_davidson   V=0: sorted |k+G|^2 exactly; constant shift; brute-force Jacobi / eigvalsh of
//                  explicit H on cfg 0 and the shrunk variants; Ritz values monotone
//   Eigenvalues of cfg 1, 3, 4 at FULL size: parity unpinned by anything external.
#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdio>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cplx;
static const double PI = 3.14159265358979323846264338327950288;

// ------------------------------------------------------------------------------------------------
// FFT.  sign=+1:  X[k] = sum_j x[j] e^{+2 pi i jk/n}  (G -> r, unnormalised: Eq. 31)
//       sign=-1:  X[k] = sum_j x[j] e^{-2 pi i jk/n}  (r -> G, the caller divides by N: Eq. 36)
// Recursive decimation in time on the smallest prime factor; generic O(p^2) butterfly.
// ------------------------------------------------------------------------------------------------
static int smallest_factor(int n) {
  for (int p = 2; p * p <= n; ++p)
    if (n % p == 0) return p;
  return n;
}

// out[k] = sum_j in[j*stride] * w[(j*k mod n) * (N0/n)],  w[t] = e^{sign 2 pi i t/N0}
static void fft_rec(const cplx* in, long stride, cplx* out, int n, const cplx* w, int N0) {
  if (n == 1) { out[0] = in[0]; return; }
  const int p = smallest_factor(n), m = n / p, step = N0 / n;
  for (int r = 0; r < p; ++r) fft_rec(in + r * stride, stride * p, out + (long)r * m, m, w, N0);
  std::vector<cplx> t(p);
  for (int k = 0; k < m; ++k) {
    for (int r = 0; r < p; ++r) t[r] = out[(long)r * m + k];
    for (int q = 0; q < p; ++q) {
      const int kk = k + q * m;
      cplx s(0.0, 0.0);
      for (int r = 0; r < p; ++r) s += t[r] * w[(long)(((long)r * kk) % n) * step];
      out[kk] = s;
    }
  }
}

static std::vector<cplx> twiddles(int n, int sign) {
  std::vector<cplx> w(n);
  for (int t = 0; t < n; ++t) {
    const double a = 2.0 * PI * (double)t / (double)n;
    w[t] = cplx(std::cos(a), sign * std::sin(a));
  }
  return w;
}

// 3D transform of a[n1][n2][n3] (n3 fastest), axis by axis.
static void fft3d(int n1, int n2, int n3, cplx* a, int sign) {
  const int nn[3] = {n1, n2, n3};
  const long st[3] = {(long)n2 * n3, (long)n3, 1};
  for (int ax = 0; ax < 3; ++ax) {
    const int n = nn[ax];
    const std::vector<cplx> w = twiddles(n, sign);
    std::vector<cplx> line(n), res(n);
    const int o1 = (ax + 1) % 3, o2 = (ax + 2) % 3;
    for (int i = 0; i < nn[o1]; ++i)
      for (int j = 0; j < nn[o2]; ++j) {
        cplx* base = a + i * st[o1] + j * st[o2];
        for (int t = 0; t < n; ++t) line[t] = base[t * st[ax]];
        fft_rec(line.data(), 1, res.data(), n, w.data(), n);
        for (int t = 0; t < n; ++t) base[t * st[ax]] = res[t];
      }
  }
}

extern "C" int kso_fft3d(int n1, int n2, int n3, cplx* a, int sign) {
  if (n1 < 1 || n2 < 1 || n3 < 1 || (sign != 1 && sign != -1)) return -1;
  fft3d(n1, n2, n3, a, sign);
  return 0;
}

// ------------------------------------------------------------------------------------------------
// Plane-wave list: keep G = m1 b1 + m2 b2 + m3 b3 iff |k+G|^2 <= ecutwfc (inclusive; reading C2),
// order m1 slowest, m3 fastest, each ascending (reading C3).  Eq. 31, L500-505.
// ------------------------------------------------------------------------------------------------
static void recip(const double* cell, double b[9]) {
  const double* a1 = cell; const double* a2 = cell + 3; const double* a3 = cell + 6;
  double c23[3] = {a2[1] * a3[2] - a2[2] * a3[1], a2[2] * a3[0] - a2[0] * a3[2], a2[0] * a3[1] - a2[1] * a3[0]};
  double c31[3] = {a3[1] * a1[2] - a3[2] * a1[1], a3[2] * a1[0] - a3[0] * a1[2], a3[0] * a1[1] - a3[1] * a1[0]};
  double c12[3] = {a1[1] * a2[2] - a1[2] * a2[1], a1[2] * a2[0] - a1[0] * a2[2], a1[0] * a2[1] - a1[1] * a2[0]};
  const double vol = a1[0] * c23[0] + a1[1] * c23[1] + a1[2] * c23[2];
  for (int i = 0; i < 3; ++i) {
    b[i] = 2 * PI * c23[i] / vol; b[3 + i] = 2 * PI * c31[i] / vol; b[6 + i] = 2 * PI * c12[i] / vol;
  }
}

static int pw_enumerate(const double* cell, const double* kf, double ecut, std::vector<int>* mil,
                        std::vector<double>* g2out) {
  double b[9]; recip(cell, b);
  double kc[3];
  for (int i = 0; i < 3; ++i) kc[i] = kf[0] * b[i] + kf[1] * b[3 + i] + kf[2] * b[6 + i];
  const double rmax = std::sqrt(ecut) + std::sqrt(kc[0] * kc[0] + kc[1] * kc[1] + kc[2] * kc[2]);
  int M[3];
  for (int i = 0; i < 3; ++i) {
    const double* a = cell + 3 * i;
    M[i] = (int)std::floor(rmax * std::sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]) / (2 * PI)) + 1;
  }
  int count = 0;
  for (int m1 = -M[0]; m1 <= M[0]; ++m1)
    for (int m2 = -M[1]; m2 <= M[1]; ++m2)
      for (int m3 = -M[2]; m3 <= M[2]; ++m3) {
        const double f[3] = {m1 + kf[0], m2 + kf[1], m3 + kf[2]};
        double q[3];
        for (int i = 0; i < 3; ++i) q[i] = f[0] * b[i] + f[1] * b[3 + i] + f[2] * b[6 + i];
        const double g2 = q[0] * q[0] + q[1] * q[1] + q[2] * q[2];
        if (g2 <= ecut) {
          if (mil) { mil->push_back(m1); mil->push_back(m2); mil->push_back(m3); }
          if (g2out) g2out->push_back(g2);
          ++count;
        }
      }
  return count;
}

extern "C" int kso_pw_count(const double* cell, const double* kf, double ecut, int* npw) {
  *npw = pw_enumerate(cell, kf, ecut, nullptr, nullptr);
  return 0;
}
extern "C" int kso_pw_list(const double* cell, const double* kf, double ecut, int* miller, double* g2) {
  std::vector<int> m; std::vector<double> g;
  pw_enumerate(cell, kf, ecut, &m, &g);
  std::memcpy(miller, m.data(), m.size() * sizeof(int));
  if (g2) std::memcpy(g2, g.data(), g.size() * sizeof(double));
  return 0;
}

// ------------------------------------------------------------------------------------------------
// Context
// ------------------------------------------------------------------------------------------------
struct kso_ctx {
  int n1, n2, n3, npw, nproj, natom;
  long N;
  std::vector<int> miller;      // [npw][3]
  std::vector<long> idx;        // grid index of G_j : (m mod n), n3 fastest (reading C5)
  std::vector<double> g2;       // |k+G|^2 (Ry)
  std::vector<cplx> vhat;       // V_loc(G) as passed, [n1][n2][n3]
  std::vector<double> vr;       // V(r) = Re sum_m vhat[m] e^{+2 pi i m.j/n}
  std::vector<cplx> beta;       // [nproj][npw]
  std::vector<int> off;         // [natom+1]
  std::vector<double> D;        // concatenated per-atom blocks
  std::vector<long> doff;       // offset of each atom's block in D
  std::vector<double> Q;        // overlap blocks (same layout as D); empty: S = I
};

static inline int pmod(int a, int n) { int r = a % n; return r < 0 ? r + n : r; }

extern "C" int kso_create(kso_ctx** out, const double* cell, const double* kf, double ecut, const int* grid,
                          const cplx* vloc_g, int nproj, const cplx* beta, int natom, const int* proj_offset,
                          const double* D) {
  kso_ctx* c = new kso_ctx;
  c->n1 = grid[0]; c->n2 = grid[1]; c->n3 = grid[2];
  c->N = (long)c->n1 * c->n2 * c->n3;
  c->npw = pw_enumerate(cell, kf, ecut, &c->miller, &c->g2);
  c->idx.resize(c->npw);
  for (int j = 0; j < c->npw; ++j) {
    const int* m = &c->miller[3 * j];
    if (2 * std::abs(m[0]) >= c->n1 || 2 * std::abs(m[1]) >= c->n2 || 2 * std::abs(m[2]) >= c->n3) { delete c; return -2; }
    c->idx[j] = ((long)pmod(m[0], c->n1) * c->n2 + pmod(m[1], c->n2)) * c->n3 + pmod(m[2], c->n3);
  }
  c->vhat.assign(vloc_g, vloc_g + c->N);
  std::vector<cplx> v(c->vhat);
  fft3d(c->n1, c->n2, c->n3, v.data(), +1);
  double vmax = 0, imax = 0;
  for (long i = 0; i < c->N; ++i) { vmax = std::max(vmax, std::abs(v[i].real())); imax = std::max(imax, std::abs(v[i].imag())); }
  if (imax > 1e-12 * std::max(vmax, 1e-300) && imax > 0) { delete c; return -5; }
  c->vr.resize(c->N);
  for (long i = 0; i < c->N; ++i) c->vr[i] = v[i].real();
  c->nproj = nproj; c->natom = natom;
  if (nproj > 0) {
    c->beta.assign(beta, beta + (long)nproj * c->npw);
    c->off.assign(proj_offset, proj_offset + natom + 1);
    long o = 0;
    for (int a = 0; a < natom; ++a) { c->doff.push_back(o); const int np = c->off[a + 1] - c->off[a]; o += (long)np * np; }
    c->D.assign(D, D + o);
    if (c->off[natom] != nproj) { delete c; return -1; }
  }
  *out = c;
  return 0;
}
extern "C" void kso_destroy(kso_ctx* c) { delete c; }
extern "C" int kso_npw(const kso_ctx* c) { return c->npw; }
extern "C" int kso_get_vr(const kso_ctx* c, double* out) { std::memcpy(out, c->vr.data(), c->N * sizeof(double)); return 0; }
extern "C" int kso_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// ------------------------------------------------------------------------------------------------
// H psi, dual-space form:  Eq. 32 (L507) kinetic + local, Eq. 3-4 (L217-221) nonlocal.
//   per band: zero grid; scatter; unnormalised inverse DFT (+); times V(r); forward DFT (-);
//   hpsi(G_j) = g2_j psi(G_j) + grid[idx_j]/N ;  B = beta^H psi ; B <- D B ; hpsi += beta B.
// ------------------------------------------------------------------------------------------------
extern "C" int kso_hpsi(const kso_ctx* c, const cplx* psi, cplx* hpsi, int nb) {
  const int npw = c->npw;
#pragma omp parallel
  {
    std::vector<cplx> g(c->N);
#pragma omp for schedule(dynamic, 1)
    for (int b = 0; b < nb; ++b) {
      const cplx* p = psi + (long)b * npw;
      cplx* h = hpsi + (long)b * npw;
      std::fill(g.begin(), g.end(), cplx(0, 0));
      for (int j = 0; j < npw; ++j) g[c->idx[j]] = p[j];
      fft3d(c->n1, c->n2, c->n3, g.data(), +1);
      for (long i = 0; i < c->N; ++i) g[i] *= c->vr[i];
      fft3d(c->n1, c->n2, c->n3, g.data(), -1);
      const double inv = 1.0 / (double)c->N;
      for (int j = 0; j < npw; ++j) h[j] = c->g2[j] * p[j] + g[c->idx[j]] * inv;
    }
  }
  if (c->nproj == 0) return 0;
  const int P = c->nproj;
  std::vector<cplx> B((long)P * nb), DB((long)P * nb);
#pragma omp parallel for collapse(2) schedule(static)
  for (int p = 0; p < P; ++p)
    for (int b = 0; b < nb; ++b) {
      const cplx* be = &c->beta[(long)p * npw];
      const cplx* ps = psi + (long)b * npw;
      double sr = 0, si = 0;   // conj(beta) * psi
      for (int j = 0; j < npw; ++j) {
        sr += be[j].real() * ps[j].real() + be[j].imag() * ps[j].imag();
        si += be[j].real() * ps[j].imag() - be[j].imag() * ps[j].real();
      }
      B[(long)p * nb + b] = cplx(sr, si);
    }
  for (int a = 0; a < c->natom; ++a) {
    const int p0 = c->off[a], np = c->off[a + 1] - p0;
    const double* Da = &c->D[c->doff[a]];
    for (int p = 0; p < np; ++p)
      for (int b = 0; b < nb; ++b) {
        cplx s(0, 0);
        for (int q = 0; q < np; ++q) s += Da[p * np + q] * B[(long)(p0 + q) * nb + b];
        DB[(long)(p0 + p) * nb + b] = s;
      }
  }
#pragma omp parallel for schedule(static)
  for (int b = 0; b < nb; ++b) {
    cplx* h = hpsi + (long)b * npw;
    for (int p = 0; p < P; ++p) {
      const cplx* be = &c->beta[(long)p * npw];
      const double cr = DB[(long)p * nb + b].real(), ci = DB[(long)p * nb + b].imag();
      for (int j = 0; j < npw; ++j)
        h[j] += cplx(be[j].real() * cr - be[j].imag() * ci, be[j].real() * ci + be[j].imag() * cr);
    }
  }
  return 0;
}

// ------------------------------------------------------------------------------------------------
// Density build (the step after diagonalisation in the SCF loop, Fig. 3):
//   rho(r) = sum_b occ_b |psi_b(r)|^2,   psi_b(r) = sum_G c_b(G) e^{+i G.r}   (Eq. 31, unnormalised; the
// Bloch phase e^{ik.r} has modulus one and drops out; the same form as Eq. 55).  The caller owns the
// 1/Omega and k-weight factors.  rho: [n1][n2][n3], n3 fastest, natural grid order.  Band by band, in order.
// ------------------------------------------------------------------------------------------------
extern "C" int kso_density(const kso_ctx* c, const cplx* psi, const double* occ, int nb, double* rho) {
  std::vector<cplx> g(c->N);
  for (long i = 0; i < c->N; ++i) rho[i] = 0.0;
  for (int b = 0; b < nb; ++b) {
    const cplx* p = psi + (long)b * c->npw;
    std::fill(g.begin(), g.end(), cplx(0, 0));
    for (int j = 0; j < c->npw; ++j) g[c->idx[j]] = p[j];
    fft3d(c->n1, c->n2, c->n3, g.data(), +1);
    for (long i = 0; i < c->N; ++i) rho[i] += occ[b] * (g[i].real() * g[i].real() + g[i].imag() * g[i].imag());
  }
  return 0;
}

// ------------------------------------------------------------------------------------------------
// Chebyshev expansion of an operator function applied to a block (the inner loop of sDFT,
// PAPER.md L588 "Chebyshev expansion scheme", Eq. 54 L680 gamma = f_H^{1/2} chi, orders 25..1200 at L714):
//   out = sum_{n=0}^{ncoef-1} c_n T_n(Ht) chi,   Ht = (H - ebar)/de  (spectrum of Ht inside [-1, 1]),
//   T_0 = chi,  T_1 = Ht chi,  T_{n+1} = 2 Ht T_n - T_{n-1}   (the textbook three-term recurrence; the paper
//   does not print it).  Term by term, in order.
// ------------------------------------------------------------------------------------------------
extern "C" int kso_chebyshev(const kso_ctx* c, const cplx* chi, int nb, int ncoef, const double* coef, double ebar,
                             double de, cplx* out) {
  const long n = (long)nb * c->npw;
  std::vector<cplx> tp(chi, chi + n), tc(n), tn(n), h(n);
  for (long i = 0; i < n; ++i) out[i] = (ncoef > 0 ? coef[0] : 0.0) * chi[i];
  if (ncoef < 2) return 0;
  kso_hpsi(c, tp.data(), h.data(), nb);
  for (long i = 0; i < n; ++i) tc[i] = (h[i] - ebar * tp[i]) / de;
  for (long i = 0; i < n; ++i) out[i] += coef[1] * tc[i];
  for (int k = 2; k < ncoef; ++k) {
    kso_hpsi(c, tc.data(), h.data(), nb);
    for (long i = 0; i < n; ++i) tn[i] = 2.0 * (h[i] - ebar * tc[i]) / de - tp[i];
    for (long i = 0; i < n; ++i) out[i] += coef[k] * tn[i];
    tp.swap(tc);
    tc.swap(tn);
  }
  return 0;
}

// ------------------------------------------------------------------------------------------------
// Explicit H(G,G') -- the definition, row-major H[j][j']:
//   H = |k+G_j|^2 delta_jj' + vhat[(m_j - m_j') mod n] + sum_a sum_{p,p' in a} beta_p(j) D^a_pp' conj(beta_p'(j'))
// ------------------------------------------------------------------------------------------------
extern "C" int kso_explicit_h(const kso_ctx* c, cplx* H) {
  const int npw = c->npw;
#pragma omp parallel for schedule(static)
  for (int j = 0; j < npw; ++j) {
    const int* mj = &c->miller[3 * j];
    for (int l = 0; l < npw; ++l) {
      const int* ml = &c->miller[3 * l];
      const long id = ((long)pmod(mj[0] - ml[0], c->n1) * c->n2 + pmod(mj[1] - ml[1], c->n2)) * c->n3 + pmod(mj[2] - ml[2], c->n3);
      cplx h = c->vhat[id];
      if (j == l) h += c->g2[j];
      for (int a = 0; a < c->natom && c->nproj > 0; ++a) {
        const int p0 = c->off[a], np = c->off[a + 1] - p0;
        const double* Da = &c->D[c->doff[a]];
        for (int p = 0; p < np; ++p)
          for (int q = 0; q < np; ++q)
            if (Da[p * np + q] != 0.0)
              h += c->beta[(long)(p0 + p) * npw + j] * Da[p * np + q] * std::conj(c->beta[(long)(p0 + q) * npw + l]);
      }
      H[(long)j * npw + l] = h;
    }
  }
  return 0;
}

// ------------------------------------------------------------------------------------------------
// Cyclic-by-row two-sided Hermitian Jacobi.  A row-major n x n, destroyed.
// theta ascending; C row-major, COLUMN i is the unit eigenvector of theta[i].
// Rotation for pivot (p,q), a_pq = |a_pq| e^{i phi}:  J = diag(1, e^{-i phi}) * [[c, s], [-s, c]],
// tau = (a_qq - a_pp) / (2|a_pq|), t = sign(tau)/(|tau| + sqrt(1+tau^2)).
// Stop: off(A)_F <= 1e-15 ||A||_F or 60 sweeps.  Returns the number of sweeps.
// ------------------------------------------------------------------------------------------------
extern "C" int kso_jacobi(int n, cplx* A, double* theta, cplx* C) {
  std::vector<cplx> V((long)n * n, cplx(0, 0));
  for (int i = 0; i < n; ++i) V[(long)i * n + i] = 1.0;
  int sweep = 0;
  for (; sweep < 60; ++sweep) {
    double off = 0, tot = 0;
    for (int i = 0; i < n; ++i)
      for (int j = 0; j < n; ++j) { const double a = std::norm(A[(long)i * n + j]); tot += a; if (i != j) off += a; }
    if (off <= 1e-30 * tot) break;   // (1e-15)^2
    for (int p = 0; p < n - 1; ++p)
      for (int q = p + 1; q < n; ++q) {
        const cplx apq = A[(long)p * n + q];
        const double ab = std::abs(apq);
        if (ab == 0.0) continue;
        const double app = A[(long)p * n + p].real(), aqq = A[(long)q * n + q].real();
        const double tau = (aqq - app) / (2.0 * ab);
        const double t = (tau >= 0 ? 1.0 : -1.0) / (std::fabs(tau) + std::sqrt(1.0 + tau * tau));
        const double cs = 1.0 / std::sqrt(1.0 + t * t), sn = t * cs;
        const cplx e = apq / ab;               // e^{i phi}
        const cplx ec = std::conj(e);
        // columns: A <- A J
        for (int i = 0; i < n; ++i) {
          const cplx x = A[(long)i * n + p], y = A[(long)i * n + q];
          A[(long)i * n + p] = cs * x - sn * ec * y;
          A[(long)i * n + q] = sn * x + cs * ec * y;
        }
        // rows: A <- J^H A
        for (int j = 0; j < n; ++j) {
          const cplx x = A[(long)p * n + j], y = A[(long)q * n + j];
          A[(long)p * n + j] = cs * x - sn * e * y;
          A[(long)q * n + j] = sn * x + cs * e * y;
        }
        A[(long)p * n + q] = 0.0; A[(long)q * n + p] = 0.0;
        A[(long)p * n + p] = cplx(A[(long)p * n + p].real(), 0.0);
        A[(long)q * n + q] = cplx(A[(long)q * n + q].real(), 0.0);
        for (int i = 0; i < n; ++i) {
          const cplx x = V[(long)i * n + p], y = V[(long)i * n + q];
          V[(long)i * n + p] = cs * x - sn * ec * y;
          V[(long)i * n + q] = sn * x + cs * ec * y;
        }
      }
  }
  std::vector<int> ord(n);
  for (int i = 0; i < n; ++i) ord[i] = i;
  std::stable_sort(ord.begin(), ord.end(), [&](int a, int b) { return A[(long)a * n + a].real() < A[(long)b * n + b].real(); });
  for (int i = 0; i < n; ++i) {
    theta[i] = A[(long)ord[i] * n + ord[i]].real();
    double nr = 0;
    for (int r = 0; r < n; ++r) nr += std::norm(V[(long)r * n + ord[i]]);
    nr = 1.0 / std::sqrt(nr);
    for (int r = 0; r < n; ++r) C[(long)r * n + i] = V[(long)r * n + ord[i]] * nr;
  }
  return sweep;
}

// ------------------------------------------------------------------------------------------------
// Small dense helpers for Davidson (vectors are rows of length npw).
// ------------------------------------------------------------------------------------------------
static inline cplx cdot(const cplx* a, const cplx* b, int n) {  // a^H b
  double sr = 0, si = 0;
  for (int j = 0; j < n; ++j) {
    sr += a[j].real() * b[j].real() + a[j].imag() * b[j].imag();
    si += a[j].real() * b[j].imag() - a[j].imag() * b[j].real();
  }
  return cplx(sr, si);
}
static inline void caxpy(cplx al, const cplx* x, cplx* y, int n) {  // y += al x
  const double ar = al.real(), ai = al.imag();
  for (int j = 0; j < n; ++j)
    y[j] = cplx(y[j].real() + ar * x[j].real() - ai * x[j].imag(), y[j].imag() + ar * x[j].imag() + ai * x[j].real());
}
static inline double nrm2(const cplx* a, int n) {
  double s = 0;
  for (int j = 0; j < n; ++j) s += std::norm(a[j]);
  return std::sqrt(s);
}

// Hc = V^H W (m x m), symmetrised, Jacobi; X = V C[:, :nb], HX = W C[:, :nb].
static void rayleigh_ritz(int npw, int m, int nb, const std::vector<cplx>& V, const std::vector<cplx>& W,
                          std::vector<cplx>& X, std::vector<cplx>& HX, std::vector<double>& eps,
                          const std::vector<cplx>* SV = nullptr, std::vector<cplx>* SX = nullptr) {
  std::vector<cplx> Hc((long)m * m), C((long)m * m);
  std::vector<double> th(m);
#pragma omp parallel for collapse(2) schedule(static)
  for (int i = 0; i < m; ++i)
    for (int j = 0; j < m; ++j) Hc[(long)i * m + j] = cdot(&V[(long)i * npw], &W[(long)j * npw], npw);
  for (int i = 0; i < m; ++i)
    for (int j = i; j < m; ++j) {
      const cplx s = 0.5 * (Hc[(long)i * m + j] + std::conj(Hc[(long)j * m + i]));
      Hc[(long)i * m + j] = s; Hc[(long)j * m + i] = std::conj(s);
    }
  kso_jacobi(m, Hc.data(), th.data(), C.data());
  X.assign((long)nb * npw, cplx(0, 0)); HX.assign((long)nb * npw, cplx(0, 0));
  if (SX) SX->assign((long)nb * npw, cplx(0, 0));
#pragma omp parallel for schedule(static)
  for (int i = 0; i < nb; ++i)
    for (int r = 0; r < m; ++r) {
      caxpy(C[(long)r * m + i], &V[(long)r * npw], &X[(long)i * npw], npw);
      caxpy(C[(long)r * m + i], &W[(long)r * npw], &HX[(long)i * npw], npw);
      if (SX) caxpy(C[(long)r * m + i], &(*SV)[(long)r * npw], &(*SX)[(long)i * npw], npw);   // S X = (S V) C
    }
  eps.assign(th.begin(), th.begin() + nb);
}

// ------------------------------------------------------------------------------------------------
// Block Davidson, exactly the listing of SURVEY §8(c.2) / DESIGN.md (the paper names the method at
// L326, L547, L578 but prints no listing; reading C10).  Teter-Payne-Allan diagonal preconditioner
// (reading C11; the paper's ref 134, L1558), subspace <= max_sub_factor * nb (north_star: 2),
// convergence: all residual 2-norms <= tol (reading C12).
// ritz_hist (nullable): [max_iter+1][nb] Ritz values after the initial RR and after each expansion.
// returns 0 converged, 1 not converged (best X, eps, residuals still written), <0 error.
// ------------------------------------------------------------------------------------------------
extern "C" int kso_davidson(const kso_ctx* c, cplx* psi, double* eig, int nb, double tol, int max_iter,
                            double* resid, int* iters_out, long long* nhpsi_out, double* ritz_hist,
                            int max_sub_factor) {
  const int npw = c->npw;
  if (nb < 1 || nb > npw || max_sub_factor < 2) return -1;
  const int mmax = max_sub_factor * nb;
  std::vector<cplx> X(psi, psi + (long)nb * npw), HX, V, W, R((long)nb * npw), T;
  std::vector<double> eps(nb), rho(nb);
  // step 0: modified Gram-Schmidt, two passes
  for (int i = 0; i < nb; ++i) {
    cplx* x = &X[(long)i * npw];
    const double n0 = nrm2(x, npw);
    for (int pass = 0; pass < 2; ++pass)
      for (int j = 0; j < i; ++j) caxpy(-cdot(&X[(long)j * npw], x, npw), &X[(long)j * npw], x, npw);
    const double n1 = nrm2(x, npw);
    if (!(n1 > 1e-10 * n0) || n0 == 0.0) return -3;
    for (int j = 0; j < npw; ++j) x[j] /= n1;
  }
  // step 1: initial Rayleigh-Ritz
  W.resize((long)nb * npw);
  kso_hpsi(c, X.data(), W.data(), nb);
  long long nh = nb;
  V = X;
  { std::vector<cplx> X2, HX2; rayleigh_ritz(npw, nb, nb, V, W, X2, HX2, eps); X.swap(X2); HX.swap(HX2); }
  V = X; W = HX;
  int m = nb, it = 0, status = 1;
  if (ritz_hist) std::copy(eps.begin(), eps.end(), ritz_hist);
  for (;;) {
    // step 2: residuals
    int nu = 0;
    std::vector<int> U;
    for (int i = 0; i < nb; ++i) {
      for (int j = 0; j < npw; ++j) R[(long)i * npw + j] = HX[(long)i * npw + j] - eps[i] * X[(long)i * npw + j];
      rho[i] = nrm2(&R[(long)i * npw], npw);
      if (rho[i] > tol) U.push_back(i);
    }
    nu = (int)U.size();
    if (nu == 0) { status = 0; break; }
    if (it >= max_iter) break;
    // step 3: T_i = K_i R_i (Teter-Payne-Allan)
    T.assign((long)nu * npw, cplx(0, 0));
    std::vector<double> tn0(nu);
    for (int u = 0; u < nu; ++u) {
      const int i = U[u];
      double ekin = 0;
      for (int j = 0; j < npw; ++j) ekin += c->g2[j] * std::norm(X[(long)i * npw + j]);
      ekin = std::max(ekin, 1e-3);
      for (int j = 0; j < npw; ++j) {
        const double x = c->g2[j] / ekin;
        const double nx = 27.0 + 18.0 * x + 12.0 * x * x + 8.0 * x * x * x;
        const double K = nx / (nx + 16.0 * x * x * x * x);
        T[(long)u * npw + j] = K * R[(long)i * npw + j];
      }
      tn0[u] = nrm2(&T[(long)u * npw], npw);
    }
    // step 4: restart
    if (m + nu > mmax) { V = X; W = HX; m = nb; }
    // step 5: project out V (twice) and the kept T's (MGS, twice); drop rule
    int kept = 0;
    for (int u = 0; u < nu; ++u) {
      cplx* t = &T[(long)u * npw];
      for (int pass = 0; pass < 2; ++pass) {
        for (int r = 0; r < m; ++r) caxpy(-cdot(&V[(long)r * npw], t, npw), &V[(long)r * npw], t, npw);
        for (int r = 0; r < kept; ++r) caxpy(-cdot(&T[(long)r * npw], t, npw), &T[(long)r * npw], t, npw);
      }
      const double n1 = nrm2(t, npw);
      if (!(n1 >= 1e-10 * tn0[u]) || tn0[u] == 0.0) continue;   // dependent: drop
      cplx* dst = &T[(long)kept * npw];
      for (int j = 0; j < npw; ++j) dst[j] = t[j] / n1;
      ++kept;
    }
    nu = kept;
    if (nu == 0) break;   // KS_NOTCONV
    // step 6: expand
    std::vector<cplx> HT((long)nu * npw);
    kso_hpsi(c, T.data(), HT.data(), nu);
    nh += nu;
    V.insert(V.end(), T.begin(), T.begin() + (long)nu * npw);
    W.insert(W.end(), HT.begin(), HT.end());
    m += nu;
    // step 7: Rayleigh-Ritz
    rayleigh_ritz(npw, m, nb, V, W, X, HX, eps);
    ++it;
    if (ritz_hist) std::copy(eps.begin(), eps.end(), ritz_hist + (long)it * nb);
  }
  std::memcpy(psi, X.data(), (long)nb * npw * sizeof(cplx));
  std::copy(eps.begin(), eps.end(), eig);
  if (resid) std::copy(rho.begin(), rho.end(), resid);
  if (iters_out) *iters_out = it;
  if (nhpsi_out) *nhpsi_out = nh;
  return status;
}

// ------------------------------------------------------------------------------------------------
// Band-by-band preconditioned conjugate gradient, the only eigensolver the paper prints:
// PAPER.md Fig. 10 L549-570.  The listing is followed line by line; what it does not print is reading C19 of
// DESIGN.md (the caption's prose, L570, and its ref 134 Teter-Payne-Allan):
//   K      the Teter-Payne-Allan diagonal polynomial of the Davidson path (reading C11), x = |k+G|^2 / max(Ekin(psi_i), 1e-3)
//   gamma  Polak-Ribiere ("by Polak-Ribiere method"):  gamma = Re<g_k - g_{k-1} | r_k> / Re<g_{k-1} | r_{k-1}>,
//          r = (I - P)(p - lambda psi) the projected gradient, g = (I - P) K (p - lambda psi) as the listing has it
//   d      before the rotation d is made orthogonal to psi_i and normalised (the cos/sin update keeps ||psi|| = 1
//          only then); the un-normalised d_k = g_k + gamma d_{k-1} is what the next step conjugates against
//   theta  "optimal step size, ensuring maximal energy reduction": the minimiser of
//          E(theta) = <psi cos + d sin | H | psi cos + d sin>,  tan 2 theta = a / (lambda - b),
//          a = 2 Re<psi|H d>, b = Re<d|H d>, on the branch of the minimum: theta = atan2(-a, b - lambda) / 2
//   stop   "convergence not reached": ||r||_2 <= tol/2 (projected gradient), or k_maxiter steps
//   after the band loop one Rayleigh-Ritz step over the nb vectors orders the pairs and removes the O(tol) couplings
//   between bands that converged one after the other (the listing returns the psi_i as they are)
// ------------------------------------------------------------------------------------------------
extern "C" int kso_cg(const kso_ctx* c, cplx* psi, double* eig, int nb, double tol, int kmaxiter, double* resid,
                      int* steps_out, long long* nhpsi_out) {
  const int npw = c->npw;
  if (nb < 1 || nb > npw || kmaxiter < 1) return -1;
  std::vector<cplx> X(psi, psi + (long)nb * npw), HX((long)nb * npw);
  std::vector<cplx> p(npw), r(npw), g(npw), gp(npw), d(npw), dn(npw), h(npw);
  long long nh = 0;
  int steps = 0, status = 0;
  for (int i = 0; i < nb; ++i) {
    cplx* x = &X[(long)i * npw];
    // psi_i = (I - sum_{j<i} |psi_j><psi_j|) psi_i, normalised
    const double n0 = nrm2(x, npw);
    for (int pass = 0; pass < 2; ++pass)
      for (int j = 0; j < i; ++j) caxpy(-cdot(&X[(long)j * npw], x, npw), &X[(long)j * npw], x, npw);
    const double n1 = nrm2(x, npw);
    if (!(n1 > 1e-10 * n0) || n0 == 0.0) return -3;
    for (int j = 0; j < npw; ++j) x[j] /= n1;
    kso_hpsi(c, x, p.data(), 1);
    ++nh;
    double lambda = cdot(x, p.data(), npw).real();
    double zeta_prev = 0.0;
    bool conv = false;
    for (int k = 1; k <= kmaxiter; ++k) {
      // g_i = K (p_i - lambda psi_i)   (Fig. 10: K acts on the plain residual), then r = (I - P_{<=i}) (p - lambda psi)
      // for the stopping rule and the Polak-Ribiere products
      double ekin = 0;
      for (int j = 0; j < npw; ++j) ekin += c->g2[j] * std::norm(x[j]);
      ekin = std::max(ekin, 1e-3);
      for (int j = 0; j < npw; ++j) {
        r[j] = p[j] - lambda * x[j];
        const double xx = c->g2[j] / ekin;
        const double nx = 27.0 + 18.0 * xx + 12.0 * xx * xx + 8.0 * xx * xx * xx;
        g[j] = (nx / (nx + 16.0 * xx * xx * xx * xx)) * r[j];
      }
      for (int jj = 0; jj <= i; ++jj) caxpy(-cdot(&X[(long)jj * npw], r.data(), npw), &X[(long)jj * npw], r.data(), npw);
      if (nrm2(r.data(), npw) <= 0.5 * tol) { conv = true; break; }
      // g_i = (I - sum_{j<=i} |psi_j><psi_j|) g_i
      for (int jj = 0; jj <= i; ++jj) caxpy(-cdot(&X[(long)jj * npw], g.data(), npw), &X[(long)jj * npw], g.data(), npw);
      const double zeta = cdot(g.data(), r.data(), npw).real();
      if (k == 1) {
        d = g;
      } else {
        const double gamma = (zeta - cdot(gp.data(), r.data(), npw).real()) / zeta_prev;
        for (int j = 0; j < npw; ++j) d[j] = g[j] + gamma * d[j];
      }
      gp = g;
      zeta_prev = zeta;
      // d' = d - psi <psi|d>, normalised
      dn = d;
      caxpy(-cdot(x, dn.data(), npw), x, dn.data(), npw);
      const double nd = nrm2(dn.data(), npw);
      if (!(nd > 0.0)) { conv = true; break; }
      for (int j = 0; j < npw; ++j) dn[j] /= nd;
      kso_hpsi(c, dn.data(), h.data(), 1);
      ++nh; ++steps;
      const double a = 2.0 * cdot(x, h.data(), npw).real();
      const double b = cdot(dn.data(), h.data(), npw).real();
      const double theta = 0.5 * std::atan2(-a, b - lambda);
      const double ct = std::cos(theta), st = std::sin(theta);
      for (int j = 0; j < npw; ++j) {
        x[j] = x[j] * ct + dn[j] * st;
        p[j] = p[j] * ct + h[j] * st;
      }
      lambda = cdot(x, p.data(), npw).real();
    }
    if (!conv) status = 1;
    std::copy(p.begin(), p.end(), &HX[(long)i * npw]);
  }
  // one Rayleigh-Ritz step over the nb vectors (H psi_i are the p_i: no extra H application)
  std::vector<cplx> X2, HX2;
  std::vector<double> eps(nb);
  rayleigh_ritz(npw, nb, nb, X, HX, X2, HX2, eps);
  for (int i = 0; i < nb; ++i) {
    eig[i] = eps[i];
    if (resid) {
      for (int j = 0; j < npw; ++j) r[j] = HX2[(long)i * npw + j] - eps[i] * X2[(long)i * npw + j];
      resid[i] = nrm2(r.data(), npw);
    }
  }
  std::copy(X2.begin(), X2.end(), psi);
  if (steps_out) *steps_out = steps;
  if (nhpsi_out) *nhpsi_out = nh;
  return status;
}

// ------------------------------------------------------------------------------------------------
// Generalised problem H psi = eps S psi (ultrasoft pseudopotentials):
//   S = 1 + sum_a sum_{p,p' in a} |beta_p> q^a_pp' <beta_p'|,  q^a real symmetric per atom (same layout as D).
// kso_spsi applies S the way kso_hpsi applies the nonlocal term; kso_explicit_s is the definition; kso_davidson_s is
// the listing of kso_davidson with every inner product taken in the S metric:
//   X^H S X = I,  R_i = H X_i - eps_i S X_i,  T <- T - V ((S V)^H T),  T S-orthonormalised,  Hc = V^H H V (standard
//   subspace problem because V^H S V = I).  Residual test: ||R_i||_2 <= tol.
// ------------------------------------------------------------------------------------------------
extern "C" int kso_set_overlap(kso_ctx* c, const double* Q) {
  if (c->nproj == 0) return -1;
  long o = 0;
  for (int a = 0; a < c->natom; ++a) { const int np = c->off[a + 1] - c->off[a]; o += (long)np * np; }
  c->Q.assign(Q, Q + o);
  return 0;
}

extern "C" int kso_spsi(const kso_ctx* c, const cplx* psi, cplx* spsi, int nb) {
  const int npw = c->npw;
  std::copy(psi, psi + (long)nb * npw, spsi);
  if (c->Q.empty()) return 0;
  for (int b = 0; b < nb; ++b) {
    const cplx* ps = psi + (long)b * npw;
    cplx* out = spsi + (long)b * npw;
    for (int a = 0; a < c->natom; ++a) {
      const int p0 = c->off[a], np = c->off[a + 1] - p0;
      const double* Qa = &c->Q[c->doff[a]];
      std::vector<cplx> B(np), QB(np, cplx(0, 0));
      for (int p = 0; p < np; ++p) B[p] = cdot(&c->beta[(long)(p0 + p) * npw], ps, npw);
      for (int p = 0; p < np; ++p)
        for (int q = 0; q < np; ++q) QB[p] += Qa[p * np + q] * B[q];
      for (int p = 0; p < np; ++p) caxpy(QB[p], &c->beta[(long)(p0 + p) * npw], out, npw);
    }
  }
  return 0;
}

extern "C" int kso_explicit_s(const kso_ctx* c, cplx* S) {
  const int npw = c->npw;
  for (int j = 0; j < npw; ++j)
    for (int l = 0; l < npw; ++l) {
      cplx sv = (j == l) ? cplx(1, 0) : cplx(0, 0);
      for (int a = 0; a < c->natom && !c->Q.empty(); ++a) {
        const int p0 = c->off[a], np = c->off[a + 1] - p0;
        const double* Qa = &c->Q[c->doff[a]];
        for (int p = 0; p < np; ++p)
          for (int q = 0; q < np; ++q)
            if (Qa[p * np + q] != 0.0)
              sv += c->beta[(long)(p0 + p) * npw + j] * Qa[p * np + q] * std::conj(c->beta[(long)(p0 + q) * npw + l]);
      }
      S[(long)j * npw + l] = sv;
    }
  return 0;
}

// S-orthonormalise column t against basis vectors bv[0..nbv) (with their S images sb) by modified Gram-Schmidt, two
// passes; returns the S-norm after the projections (t is then scaled to S-norm one and st = S t is returned).
static double s_mgs(const kso_ctx* c, int npw, const std::vector<const cplx*>& bv, const std::vector<const cplx*>& sb, cplx* t,
                    cplx* st) {
  for (int pass = 0; pass < 2; ++pass)
    for (size_t r = 0; r < bv.size(); ++r) caxpy(-cdot(sb[r], t, npw), bv[r], t, npw);
  kso_spsi(c, t, st, 1);
  const double n2 = cdot(t, st, npw).real();
  const double n = std::sqrt(std::max(n2, 0.0));
  if (n > 0)
    for (int j = 0; j < npw; ++j) { t[j] /= n; st[j] /= n; }
  return n;
}

extern "C" int kso_davidson_s(const kso_ctx* c, cplx* psi, double* eig, int nb, double tol, int max_iter, double* resid,
                              int* iters_out, long long* nhpsi_out) {
  const int npw = c->npw;
  if (nb < 1 || nb > npw) return -1;
  const int mmax = 2 * nb;
  std::vector<cplx> X(psi, psi + (long)nb * npw), SX((long)nb * npw), HX, V, W, SV, R((long)nb * npw), T, ST;
  std::vector<double> eps(nb), rho(nb);
  // step 0: S-orthonormal start block
  for (int i = 0; i < nb; ++i) {
    std::vector<const cplx*> bv, sb;
    for (int j = 0; j < i; ++j) { bv.push_back(&X[(long)j * npw]); sb.push_back(&SX[(long)j * npw]); }
    const double n0 = nrm2(&X[(long)i * npw], npw);
    const double n1 = s_mgs(c, npw, bv, sb, &X[(long)i * npw], &SX[(long)i * npw]);
    if (!(n1 > 1e-10 * n0) || n0 == 0.0) return -3;
  }
  // step 1: Rayleigh-Ritz (V^H S V = I: standard subspace problem); S X rotates like H X
  W.resize((long)nb * npw);
  kso_hpsi(c, X.data(), W.data(), nb);
  long long nh = nb;
  V = X; SV = SX;
  auto ritz = [&](int m) {
    std::vector<cplx> X2, HX2, SX2;
    rayleigh_ritz(npw, m, nb, V, W, X2, HX2, eps, &SV, &SX2);
    X.swap(X2); HX.swap(HX2); SX.swap(SX2);
  };
  ritz(nb);
  V = X; W = HX; SV = SX;
  int m = nb, it = 0, status = 1;
  for (;;) {
    std::vector<int> U;
    for (int i = 0; i < nb; ++i) {
      for (int j = 0; j < npw; ++j) R[(long)i * npw + j] = HX[(long)i * npw + j] - eps[i] * SX[(long)i * npw + j];
      rho[i] = nrm2(&R[(long)i * npw], npw);
      if (rho[i] > tol) U.push_back(i);
    }
    int nu = (int)U.size();
    if (nu == 0) { status = 0; break; }
    if (it >= max_iter) break;
    T.assign((long)nu * npw, cplx(0, 0));
    ST.assign((long)nu * npw, cplx(0, 0));
    std::vector<double> tn0(nu);
    for (int u = 0; u < nu; ++u) {
      const int i = U[u];
      double ekin = 0;
      for (int j = 0; j < npw; ++j) ekin += c->g2[j] * std::norm(X[(long)i * npw + j]);
      ekin = std::max(ekin, 1e-3);
      for (int j = 0; j < npw; ++j) {
        const double x = c->g2[j] / ekin;
        const double nx = 27.0 + 18.0 * x + 12.0 * x * x + 8.0 * x * x * x;
        T[(long)u * npw + j] = (nx / (nx + 16.0 * x * x * x * x)) * R[(long)i * npw + j];
      }
      tn0[u] = nrm2(&T[(long)u * npw], npw);
    }
    if (m + nu > mmax) { V = X; W = HX; SV = SX; m = nb; }
    int kept = 0;
    for (int u = 0; u < nu; ++u) {
      std::vector<const cplx*> bv, sb;
      for (int r = 0; r < m; ++r) { bv.push_back(&V[(long)r * npw]); sb.push_back(&SV[(long)r * npw]); }
      for (int r = 0; r < kept; ++r) { bv.push_back(&T[(long)r * npw]); sb.push_back(&ST[(long)r * npw]); }
      std::vector<cplx> t(&T[(long)u * npw], &T[(long)u * npw] + npw), st(npw);
      const double n1 = s_mgs(c, npw, bv, sb, t.data(), st.data());
      if (!(n1 >= 1e-10 * tn0[u]) || tn0[u] == 0.0) continue;
      std::copy(t.begin(), t.end(), &T[(long)kept * npw]);
      std::copy(st.begin(), st.end(), &ST[(long)kept * npw]);
      ++kept;
    }
    nu = kept;
    if (nu == 0) break;
    std::vector<cplx> HT((long)nu * npw);
    kso_hpsi(c, T.data(), HT.data(), nu);
    nh += nu;
    V.insert(V.end(), T.begin(), T.begin() + (long)nu * npw);
    SV.insert(SV.end(), ST.begin(), ST.begin() + (long)nu * npw);
    W.insert(W.end(), HT.begin(), HT.end());
    m += nu;
    ritz(m);
    ++it;
  }
  std::copy(X.begin(), X.end(), psi);
  for (int i = 0; i < nb; ++i) { eig[i] = eps[i]; if (resid) resid[i] = rho[i]; }
  if (iters_out) *iters_out = it;
  if (nhpsi_out) *nhpsi_out = nh;
  return status;
}
