// cg.cu -- band-by-band preconditioned conjugate gradient, Fig. 10, with
// reading C19 of DESIGN.md for what the listing omits (K = Teter-Payne-Allan, gamma = Polak-Ribiere, theta = the
// minimiser of the Rayleigh quotient on the psi-d circle, stop at ||r|| <= tol/2, one closing Rayleigh-Ritz step).
//
// The method is sequential over bands and over CG steps, so the device work of a step is a chain of short kernels on
// ONE vector: fused elementwise updates that read their scalars (lambda, gamma, theta, ...) from a small device block
// and compute the step's scalar arithmetic redundantly per thread (no scalar kernels, no host round trip), block
// reductions with a fixed order, the projections against the bands found so far as (dot per band, then one fused
// subtraction), and ks_hpsi on a single vector.  One host read per step: ||r||^2 for the stopping rule.
#include "ctx.h"
#include <algorithm>
#include <cmath>
#include <vector>

#define CG_T 512
// scalar block (doubles)
enum { S_LAM = 0, S_EKIN, S_ZETA, S_ZETAP, S_GPR, S_XD_RE, S_XD_IM, S_DN2, S_XH, S_DH, S_R2, S_COUNT = 16 };

__device__ __forceinline__ double block_sum(double v) {
  __shared__ double sh[CG_T / 32];
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
  __syncthreads();
  double s = 0.0;
  for (int w = 0; w < CG_T / 32; ++w) s += sh[w];     // same order in every thread: deterministic
  return s;
}

// r = p - lambda x
__global__ void k_cg_resid(int n, const cplx* __restrict__ p, const cplx* __restrict__ x, const double* __restrict__ sc,
                           cplx* __restrict__ r) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double lam = sc[S_LAM];
  r[i] = cmake(p[i].x - lam * x[i].x, p[i].y - lam * x[i].y);
}
// s[j] = <X_j | v>, one CTA per band j
__global__ void __launch_bounds__(CG_T) k_cg_dots_x(int n, const cplx* __restrict__ X, const cplx* __restrict__ v, cplx* __restrict__ s) {
  const cplx* xj = X + (size_t)blockIdx.x * n;
  double re = 0, im = 0;
  for (int i = threadIdx.x; i < n; i += CG_T) {
    const cplx a = xj[i], b = v[i];
    re += a.x * b.x + a.y * b.y;
    im += a.x * b.y - a.y * b.x;
  }
  re = block_sum(re);
  im = block_sum(im);
  if (threadIdx.x == 0) s[blockIdx.x] = cmake(re, im);
}
// v -= sum_j s[j] X_j
__global__ void k_cg_sub_x(int n, int nvec, const cplx* __restrict__ X, const cplx* __restrict__ s, cplx* __restrict__ v) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double re = v[i].x, im = v[i].y;
  for (int j = 0; j < nvec; ++j) {
    const cplx c = s[j], a = X[(size_t)j * n + i];
    re -= c.x * a.x - c.y * a.y;
    im -= c.x * a.y + c.y * a.x;
  }
  v[i] = cmake(re, im);
}
// up to three real parts of dot products in one launch: out[k] = Re <a_k | b_k>, weighted by w if given.
// grid (CG_NB, count): CG_NB CTAs share one dot product, each writes its partial sum, and the CTA that arrives last adds
// the partials in index order -- many CTAs' worth of loads in flight, and still one fixed summation order.
#define CG_NB 32
struct Dot3 { const cplx* a[3]; const cplx* b[3]; const double* w[3]; int out[3]; int count; };
__global__ void __launch_bounds__(CG_T) k_cg_dot3(int n, Dot3 d, double* __restrict__ sc, double* __restrict__ part,
                                                  unsigned* __restrict__ ticket) {
  const int k = blockIdx.y;
  const cplx *a = d.a[k], *b = d.b[k];
  const double* w = d.w[k];
  double re = 0;
  for (int i = blockIdx.x * CG_T + threadIdx.x; i < n; i += CG_NB * CG_T) {
    const double t = a[i].x * b[i].x + a[i].y * b[i].y;
    re += w ? w[i] * t : t;
  }
  re = block_sum(re);
  __shared__ bool last;
  if (threadIdx.x == 0) {
    part[k * CG_NB + blockIdx.x] = re;
    __threadfence();
    last = (atomicAdd(&ticket[k], 1u) == CG_NB - 1);
  }
  __syncthreads();
  if (last && threadIdx.x == 0) {
    __threadfence();
    double s = 0;
    for (int j = 0; j < CG_NB; ++j) s += ((volatile double*)part)[k * CG_NB + j];
    sc[d.out[k]] = s;
    ticket[k] = 0;
  }
}
// complex <x|d> -> sc[S_XD_RE], sc[S_XD_IM]   (same scheme; partial slots 3 and 4)
__global__ void __launch_bounds__(CG_T) k_cg_cdot(int n, const cplx* __restrict__ x, const cplx* __restrict__ d, double* __restrict__ sc,
                                                  double* __restrict__ part, unsigned* __restrict__ ticket) {
  double re = 0, im = 0;
  for (int i = blockIdx.x * CG_T + threadIdx.x; i < n; i += CG_NB * CG_T) {
    re += x[i].x * d[i].x + x[i].y * d[i].y;
    im += x[i].x * d[i].y - x[i].y * d[i].x;
  }
  re = block_sum(re);
  im = block_sum(im);
  __shared__ bool last;
  if (threadIdx.x == 0) {
    part[3 * CG_NB + blockIdx.x] = re;
    part[4 * CG_NB + blockIdx.x] = im;
    __threadfence();
    last = (atomicAdd(&ticket[3], 1u) == CG_NB - 1);
  }
  __syncthreads();
  if (last && threadIdx.x == 0) {
    __threadfence();
    double sr = 0, si = 0;
    for (int j = 0; j < CG_NB; ++j) { sr += ((volatile double*)part)[3 * CG_NB + j]; si += ((volatile double*)part)[4 * CG_NB + j]; }
    sc[S_XD_RE] = sr; sc[S_XD_IM] = si;
    ticket[3] = 0;
  }
}
// g = K r, Teter-Payne-Allan with x = g2 / max(Ekin, 1e-3)
__global__ void k_cg_precond(int n, const cplx* __restrict__ r, const double* __restrict__ g2, const double* __restrict__ sc,
                             cplx* __restrict__ g) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double x = g2[i] / fmax(sc[S_EKIN], 1e-3);
  const double nx = 27.0 + 18.0 * x + 12.0 * x * x + 8.0 * x * x * x;
  const double K = nx / (nx + 16.0 * x * x * x * x);
  g[i] = cmake(K * r[i].x, K * r[i].y);
}
// d = g (first) or g + gamma d, gamma = (zeta - <g_prev|r>) / zeta_prev
__global__ void k_cg_dir(int n, const cplx* __restrict__ g, const double* __restrict__ sc, int first, cplx* __restrict__ d) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  if (first) { d[i] = g[i]; return; }
  const double gamma = (sc[S_ZETA] - sc[S_GPR]) / sc[S_ZETAP];
  d[i] = cmake(fma(gamma, d[i].x, g[i].x), fma(gamma, d[i].y, g[i].y));
}
// dn = d - x <x|d>
__global__ void k_cg_orth(int n, const cplx* __restrict__ d, const cplx* __restrict__ x, const double* __restrict__ sc,
                          cplx* __restrict__ dn) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double cr = sc[S_XD_RE], ci = sc[S_XD_IM];
  dn[i] = cmake(d[i].x - (cr * x[i].x - ci * x[i].y), d[i].y - (cr * x[i].y + ci * x[i].x));
}
__global__ void k_cg_scale(int n, const double* __restrict__ sc, cplx* __restrict__ dn) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double f = rsqrt(sc[S_DN2]);
  dn[i] = cmake(f * dn[i].x, f * dn[i].y);
}
// theta = atan2(-a, b - lambda)/2, a = 2 Re<x|h>, b = Re<dn|h>;  x <- x cos + dn sin,  p <- p cos + h sin
__global__ void k_cg_rotate(int n, const double* __restrict__ sc, cplx* __restrict__ x, cplx* __restrict__ p,
                            const cplx* __restrict__ dn, const cplx* __restrict__ h) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double theta = 0.5 * atan2(-2.0 * sc[S_XH], sc[S_DH] - sc[S_LAM]);
  double st, ct;
  sincos(theta, &st, &ct);
  x[i] = cmake(x[i].x * ct + dn[i].x * st, x[i].y * ct + dn[i].y * st);
  p[i] = cmake(p[i].x * ct + h[i].x * st, p[i].y * ct + h[i].y * st);
}
__global__ void k_cg_shift_scalar(double* sc) { sc[S_ZETAP] = sc[S_ZETA]; }
// closing residual norms: rho[b] = || HX_b - eps_b X_b ||
__global__ void __launch_bounds__(CG_T) k_cg_resnorm(int n, const cplx* __restrict__ X, const cplx* __restrict__ HX,
                                                     const double* __restrict__ eps, double* __restrict__ rho) {
  const cplx *x = X + (size_t)blockIdx.x * n, *h = HX + (size_t)blockIdx.x * n;
  const double e = eps[blockIdx.x];
  double s = 0;
  for (int i = threadIdx.x; i < n; i += CG_T) {
    const double a = h[i].x - e * x[i].x, b = h[i].y - e * x[i].y;
    s += a * a + b * b;
  }
  s = block_sum(s);
  if (threadIdx.x == 0) rho[blockIdx.x] = sqrt(s);
}

#define RC(x) do { int rc__ = (x); if (rc__ < 0) return rc__; } while (0)

struct CgBuf {     // freed on every exit path
  cplx *HX = nullptr, *X2 = nullptr, *HX2 = nullptr, *vec = nullptr, *s = nullptr, *Hc = nullptr, *Cm = nullptr;
  double *sc = nullptr, *theta = nullptr, *rho = nullptr, *part = nullptr;
  unsigned* ticket = nullptr;
  ~CgBuf() {
    cudaFree(part); cudaFree(ticket);
    cudaFree(HX); cudaFree(X2); cudaFree(HX2); cudaFree(vec); cudaFree(s); cudaFree(Hc); cudaFree(Cm);
    cudaFree(sc); cudaFree(theta); cudaFree(rho);
  }
};

int ks_cg_impl(ks_ctx* c, cplx* psi, double* eig, int nb, double tol, int kmaxiter, double* resid, int* steps_out,
               long long* nhpsi_out) {
  if (!c) return KS_EINVAL;
  const int npw = c->P.npw;
  if (!psi || !eig || nb < 1 || nb > npw || !(tol > 0) || kmaxiter < 1) { c->err = "ks_cg: bad argument"; return KS_EINVAL; }
  cudaStream_t st = c->stream;
  const size_t vb = sizeof(cplx) * (size_t)npw;
  CgBuf w;
  KS_CUDA_CHECK(cudaMalloc(&w.HX, vb * nb), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.X2, vb * nb), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.HX2, vb * nb), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.vec, vb * 6), c->err);             // r, g, g_prev, d, dn, h
  KS_CUDA_CHECK(cudaMalloc(&w.s, sizeof(cplx) * nb), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.Hc, sizeof(cplx) * (size_t)nb * nb), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.Cm, sizeof(cplx) * (size_t)nb * nb), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.sc, sizeof(double) * S_COUNT), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.part, sizeof(double) * 5 * CG_NB), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.ticket, sizeof(unsigned) * 4), c->err);
  KS_CUDA_CHECK(cudaMemsetAsync(w.ticket, 0, sizeof(unsigned) * 4, st), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.theta, sizeof(double) * nb), c->err);
  KS_CUDA_CHECK(cudaMalloc(&w.rho, sizeof(double) * nb), c->err);
  cplx *r = w.vec, *g = r + npw, *gp = g + npw, *d = gp + npw, *dn = d + npw, *h = dn + npw;
  cplx* X = psi;                                                  // the bands are refined in place
  const int nblk = ceil_div(npw, 256);
  long long nh = 0;
  int steps = 0, status = KS_OK;
  double hs[2];
  for (int i = 0; i < nb; ++i) {
    cplx* x = X + (size_t)i * npw;
    cplx* p = w.HX + (size_t)i * npw;
    // psi_i = (I - sum_{j<i} |psi_j><psi_j|) psi_i (twice), normalised
    Dot3 dq;
    dq.count = 1; dq.a[0] = x; dq.b[0] = x; dq.w[0] = nullptr; dq.out[0] = S_DN2;
    k_cg_dot3<<<dim3(CG_NB, 1), CG_T, 0, st>>>(npw, dq, w.sc, w.part, w.ticket);
    KS_CUDA_CHECK(cudaMemcpyAsync(&hs[0], w.sc + S_DN2, sizeof(double), cudaMemcpyDeviceToHost, st), c->err);
    for (int pass = 0; pass < 2 && i > 0; ++pass) {
      k_cg_dots_x<<<i, CG_T, 0, st>>>(npw, X, x, w.s);
      k_cg_sub_x<<<nblk, 256, 0, st>>>(npw, i, X, w.s, x);
    }
    k_cg_dot3<<<dim3(CG_NB, 1), CG_T, 0, st>>>(npw, dq, w.sc, w.part, w.ticket);
    KS_CUDA_CHECK(cudaMemcpyAsync(&hs[1], w.sc + S_DN2, sizeof(double), cudaMemcpyDeviceToHost, st), c->err);
    KS_CUDA_CHECK(cudaStreamSynchronize(st), c->err);
    if (!(hs[1] > 1e-20 * hs[0]) || hs[0] == 0.0) { c->err = "ks_cg: start block is rank deficient"; return KS_EINVAL; }
    k_cg_scale<<<nblk, 256, 0, st>>>(npw, w.sc, x);
    RC(ks_hpsi_impl(c, x, p, 1));
    ++nh;
    // lambda = Re<x|p>, Ekin = sum g2 |x|^2
    Dot3 dl;
    dl.count = 2; dl.a[0] = x; dl.b[0] = p; dl.w[0] = nullptr; dl.out[0] = S_LAM;
    dl.a[1] = x; dl.b[1] = x; dl.w[1] = c->P.d_g2; dl.out[1] = S_EKIN;
    k_cg_dot3<<<dim3(CG_NB, 2), CG_T, 0, st>>>(npw, dl, w.sc, w.part, w.ticket);
    bool conv = false;
    for (int k = 1; k <= kmaxiter; ++k) {
      // g = K (p - lambda psi) (Fig. 10: K acts on the plain residual); r = (I - P_{<=i}) (p - lambda psi)
      std::swap(g, gp);
      k_cg_resid<<<nblk, 256, 0, st>>>(npw, p, x, w.sc, r);
      k_cg_precond<<<nblk, 256, 0, st>>>(npw, r, c->P.d_g2, w.sc, g);
      k_cg_dots_x<<<i + 1, CG_T, 0, st>>>(npw, X, r, w.s);
      k_cg_sub_x<<<nblk, 256, 0, st>>>(npw, i + 1, X, w.s, r);
      Dot3 dr;
      dr.count = 1; dr.a[0] = r; dr.b[0] = r; dr.w[0] = nullptr; dr.out[0] = S_R2;
      k_cg_dot3<<<dim3(CG_NB, 1), CG_T, 0, st>>>(npw, dr, w.sc, w.part, w.ticket);
      KS_CUDA_CHECK(cudaMemcpyAsync(&hs[0], w.sc + S_R2, sizeof(double), cudaMemcpyDeviceToHost, st), c->err);
      KS_CUDA_CHECK(cudaStreamSynchronize(st), c->err);
      if (std::sqrt(hs[0]) <= 0.5 * tol) { conv = true; break; }
      // g = (I - P_{<=i}) g
      k_cg_dots_x<<<i + 1, CG_T, 0, st>>>(npw, X, g, w.s);
      k_cg_sub_x<<<nblk, 256, 0, st>>>(npw, i + 1, X, w.s, g);
      // zeta = Re<g|r>, <g_prev|r>; d = g + gamma d
      if (k > 1) k_cg_shift_scalar<<<1, 1, 0, st>>>(w.sc);
      Dot3 dz;
      dz.count = 2; dz.a[0] = g; dz.b[0] = r; dz.w[0] = nullptr; dz.out[0] = S_ZETA;
      dz.a[1] = gp; dz.b[1] = r; dz.w[1] = nullptr; dz.out[1] = S_GPR;
      k_cg_dot3<<<dim3(CG_NB, k > 1 ? 2 : 1), CG_T, 0, st>>>(npw, dz, w.sc, w.part, w.ticket);
      k_cg_dir<<<nblk, 256, 0, st>>>(npw, g, w.sc, k == 1, d);
      // dn = d - x <x|d>, normalised
      k_cg_cdot<<<CG_NB, CG_T, 0, st>>>(npw, x, d, w.sc, w.part, w.ticket);
      k_cg_orth<<<nblk, 256, 0, st>>>(npw, d, x, w.sc, dn);
      Dot3 dd;
      dd.count = 1; dd.a[0] = dn; dd.b[0] = dn; dd.w[0] = nullptr; dd.out[0] = S_DN2;
      k_cg_dot3<<<dim3(CG_NB, 1), CG_T, 0, st>>>(npw, dd, w.sc, w.part, w.ticket);
      k_cg_scale<<<nblk, 256, 0, st>>>(npw, w.sc, dn);
      RC(ks_hpsi_impl(c, dn, h, 1));
      ++nh; ++steps;
      // a/2 = Re<x|h>, b = Re<dn|h>; rotate; lambda, Ekin
      Dot3 da;
      da.count = 2; da.a[0] = x; da.b[0] = h; da.w[0] = nullptr; da.out[0] = S_XH;
      da.a[1] = dn; da.b[1] = h; da.w[1] = nullptr; da.out[1] = S_DH;
      k_cg_dot3<<<dim3(CG_NB, 2), CG_T, 0, st>>>(npw, da, w.sc, w.part, w.ticket);
      k_cg_rotate<<<nblk, 256, 0, st>>>(npw, w.sc, x, p, dn, h);
      k_cg_dot3<<<dim3(CG_NB, 2), CG_T, 0, st>>>(npw, dl, w.sc, w.part, w.ticket);
    }
    if (!conv) status = KS_NOTCONV;
  }
  // closing Rayleigh-Ritz step over the nb vectors (H psi_i = p_i: no extra H application)
  RC(ks_gemm_hn(st, nb, nb, npw, X, npw, w.HX, npw, w.Hc, nb, &c->gws, c->err));
  RC(ks_eigh_run(st, nb, w.Hc, nb, w.theta, w.Cm, nb, &c->ews, nullptr, c->err));
  RC(ks_gemm_nn(st, npw, nb, nb, X, npw, w.Cm, nb, w.X2, npw, 0, c->err));
  RC(ks_gemm_nn(st, npw, nb, nb, w.HX, npw, w.Cm, nb, w.HX2, npw, 0, c->err));
  k_cg_resnorm<<<nb, CG_T, 0, st>>>(npw, w.X2, w.HX2, w.theta, w.rho);
  KS_CUDA_CHECK(cudaMemcpyAsync(psi, w.X2, vb * nb, cudaMemcpyDeviceToDevice, st), c->err);
  KS_CUDA_CHECK(cudaMemcpyAsync(eig, w.theta, sizeof(double) * nb, cudaMemcpyDeviceToDevice, st), c->err);
  if (resid) KS_CUDA_CHECK(cudaMemcpyAsync(resid, w.rho, sizeof(double) * nb, cudaMemcpyDeviceToDevice, st), c->err);
  KS_CUDA_CHECK(cudaStreamSynchronize(st), c->err);
  KS_CUDA_CHECK(cudaGetLastError(), c->err);
  if (steps_out) *steps_out = steps;
  if (nhpsi_out) *nhpsi_out = nh;
  return status;
}
