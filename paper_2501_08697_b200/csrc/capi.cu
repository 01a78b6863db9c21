// capi.cu -- the C ABI of include/kspw.h: G-sphere helpers, context creation (host-side plan of the
// sticks / live planes / index maps), ks_hpsi and the exported building blocks.
#include "ctx.h"
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>

extern "C" {
typedef struct { double re, im; } ks_c128;
}

std::string& ks_global_error() {
  static thread_local std::string e;
  return e;
}

static const double KS_PI = 3.14159265358979323846264338327950288;

// ------------------------------------------------------------------------------------------------
// G sphere (Eq. 31; readings C2, C3): keep G iff |k+G|^2 <= ecutwfc, order m1 slowest.
// ------------------------------------------------------------------------------------------------
static void reciprocal_rows(const double* a, double* b) {
  const double c0[3] = {a[4] * a[8] - a[5] * a[7], a[5] * a[6] - a[3] * a[8], a[3] * a[7] - a[4] * a[6]};   // a2 x a3
  const double c1[3] = {a[7] * a[2] - a[8] * a[1], a[8] * a[0] - a[6] * a[2], a[6] * a[1] - a[7] * a[0]};   // a3 x a1
  const double c2[3] = {a[1] * a[5] - a[2] * a[4], a[2] * a[3] - a[0] * a[5], a[0] * a[4] - a[1] * a[3]};   // a1 x a2
  const double vol = a[0] * c0[0] + a[1] * c0[1] + a[2] * c0[2];
  for (int i = 0; i < 3; ++i) {
    b[i] = 2 * KS_PI * c0[i] / vol;
    b[3 + i] = 2 * KS_PI * c1[i] / vol;
    b[6 + i] = 2 * KS_PI * c2[i] / vol;
  }
}

static int sphere(const double* cell, const double* kf, double ecut, std::vector<int>* mil, std::vector<double>* g2) {
  double b[9];
  reciprocal_rows(cell, b);
  double kc[3], kn = 0;
  for (int i = 0; i < 3; ++i) {
    kc[i] = kf[0] * b[i] + kf[1] * b[3 + i] + kf[2] * b[6 + i];
    kn += kc[i] * kc[i];
  }
  const double rmax = std::sqrt(ecut) + std::sqrt(kn);
  int lim[3];
  for (int i = 0; i < 3; ++i) {
    const double* ai = cell + 3 * i;
    lim[i] = (int)std::floor(rmax * std::sqrt(ai[0] * ai[0] + ai[1] * ai[1] + ai[2] * ai[2]) / (2 * KS_PI)) + 1;
  }
  int n = 0;
  for (int m1 = -lim[0]; m1 <= lim[0]; ++m1)
    for (int m2 = -lim[1]; m2 <= lim[1]; ++m2)
      for (int m3 = -lim[2]; m3 <= lim[2]; ++m3) {
        const double f0 = m1 + kf[0], f1 = m2 + kf[1], f2 = m3 + kf[2];
        double q2 = 0;
        for (int i = 0; i < 3; ++i) {
          const double q = f0 * b[i] + f1 * b[3 + i] + f2 * b[6 + i];
          q2 += q * q;
        }
        if (q2 <= ecut) {
          ++n;
          if (mil) { mil->push_back(m1); mil->push_back(m2); mil->push_back(m3); }
          if (g2) g2->push_back(q2);
        }
      }
  return n;
}

extern "C" int ks_pw_count(const double cell[9], const double k_frac[3], double ecutwfc, int* npw) {
  if (!cell || !k_frac || !npw || !(ecutwfc > 0)) return KS_EINVAL;
  *npw = sphere(cell, k_frac, ecutwfc, nullptr, nullptr);
  return KS_OK;
}
extern "C" int ks_pw_list(const double cell[9], const double k_frac[3], double ecutwfc, int* miller, double* g2) {
  if (!cell || !k_frac || !miller || !(ecutwfc > 0)) return KS_EINVAL;
  std::vector<int> m;
  std::vector<double> g;
  sphere(cell, k_frac, ecutwfc, &m, &g);
  std::memcpy(miller, m.data(), m.size() * sizeof(int));
  if (g2) std::memcpy(g2, g.data(), g.size() * sizeof(double));
  return KS_OK;
}
extern "C" int ks_supported_sizes(int* sizes, int cap) { return ks_fft_sizes(sizes, sizes ? cap : 0); }

// ------------------------------------------------------------------------------------------------
// context
// ------------------------------------------------------------------------------------------------
static inline int pmod(int a, int n) { const int r = a % n; return r < 0 ? r + n : r; }

template <typename T>
static int upload(T** dst, const std::vector<T>& src, std::string& err) {
  *dst = nullptr;
  const size_t bytes = std::max<size_t>(src.size(), 1) * sizeof(T);
  KS_CUDA_CHECK(cudaMalloc(dst, bytes), err);
  if (!src.empty()) KS_CUDA_CHECK(cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice), err);
  return KS_OK;
}

// Live-plane workspace: c->fft_batch is the batch LIMIT (bands per launch of the three FFT kernels); the buffer itself is
// sized at first use to min(limit, bands actually applied) and grows when a larger block arrives, so a context that only
// ever sees 32 bands does not hold gigabytes.
static int auto_batch(const HpsiPlan& P) {
  const char* env = getenv("KSPW_FFT_BATCH");
  if (env && atoi(env) > 0) return atoi(env);
  const double per = 16.0 * P.L1 * P.n2 * P.n3;
  // as many bands per launch as 9 GB of live planes hold (cfg 1, cfg 4 and cfg 3: the whole block).  Measured, FFT path as a
  // fraction of HBM: cfg 1 80 -> 160 bands 51 -> 54 %; cfg 3 26 / 52 / 104 / 260 bands 52.1 / 53.8 / 55.0 / 55.7 %: the planes
  // stream through HBM and every launch ends with a partly filled wave, so fewer, larger launches win; L2 cannot hold a useful batch
  int b = (int)(9.0e9 / per);
  return std::max(2, std::min(b, 1024));
}

int ks_ensure_planes(ks_ctx* c, int nb, cudaStream_t sync_stream) {
  HpsiPlan& P = c->P;
  const int want = std::min(c->fft_batch, std::max(nb, 1));
  if (want <= P.batch_cap) return KS_OK;
  if (P.d_planes) {
    cudaStreamSynchronize(sync_stream);
    cudaFree(P.d_planes);
    P.d_planes = nullptr; P.batch_cap = 0;
  }
  const size_t per = sizeof(cplx) * (size_t)P.L1 * P.n2 * P.n3;
  KS_CUDA_CHECK(cudaMalloc(&P.d_planes, per * want), c->err);
  P.batch_cap = want;
  return ks_hpsi_make_tmap(P, c->err);
}

extern "C" void ks_destroy(ks_ctx* c);

static int create_impl(ks_ctx* c, const double* cell, const double* kf, double ecut, const int* grid, const cplx* vloc,
                       int nproj, const cplx* beta, int natom, const int* off, const double* D) {
  std::string& err = c->err;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { err = "no CUDA device (there is no CPU fallback)"; return KS_ECUDA; }
  KS_CUDA_CHECK(ks_fft_init_constants(), err);
  HpsiPlan& P = c->P;
  P.n1 = grid[0]; P.n2 = grid[1]; P.n3 = grid[2];
  P.N = (long)P.n1 * P.n2 * P.n3;
  std::vector<int> mil;
  std::vector<double> g2;
  P.npw = sphere(cell, kf, ecut, &mil, &g2);
  if (P.npw <= 0) { err = "empty G sphere"; return KS_EINVAL; }
  // alias rule (reading C6): n_i > 2 m_psi,i + m_V,i and n_i > 2 m_V,i, m_V,i = floor(2 sqrt(ecut) |a_i| / 2 pi)
  int mpsi[3] = {0, 0, 0};
  for (int j = 0; j < P.npw; ++j)
    for (int i = 0; i < 3; ++i) mpsi[i] = std::max(mpsi[i], std::abs(mil[3 * j + i]));
  for (int i = 0; i < 3; ++i) {
    const double* ai = cell + 3 * i;
    const int mv = (int)std::floor(2.0 * std::sqrt(ecut) * std::sqrt(ai[0] * ai[0] + ai[1] * ai[1] + ai[2] * ai[2]) / (2 * KS_PI));
    if (!(grid[i] > 2 * mpsi[i] + mv) || !(grid[i] > 2 * mv)) {
      char b[200];
      snprintf(b, sizeof b, "grid axis %d: n=%d violates n > 2*m_psi + m_V = %d (m_psi=%d, m_V=%d)", i, grid[i], 2 * mpsi[i] + mv, mpsi[i], mv);
      err = b;
      return KS_EGRID;
    }
  }
  // live planes, sticks, position maps (PW order is m1 slowest, so planes and sticks are contiguous runs)
  std::vector<int> plane_s0, plane_y0, plane_pw0;
  std::vector<int4> stick;
  int nst = 0, smax = 0, cur_m1 = 0, cur_m2 = 0, cur_m3 = 0, s_in_plane = 0;
  for (int j = 0; j < P.npw; ++j) {
    const int m1 = mil[3 * j], m2 = mil[3 * j + 1], m3 = mil[3 * j + 2];
    const bool new_plane = (j == 0) || (m1 != cur_m1);
    const bool new_stick = new_plane || (m2 != cur_m2);
    if (new_plane) {
      if (j && m1 != cur_m1 + 1) { err = "G sphere: live x-planes are not contiguous"; return KS_EINVAL; }
      plane_s0.push_back(nst);
      plane_y0.push_back(pmod(m2, P.n2));
      plane_pw0.push_back(j);
      smax = std::max(smax, s_in_plane);
      s_in_plane = 0;
    }
    if (new_stick) {
      if (!new_plane && m2 != cur_m2 + 1) { err = "G sphere: sticks of a plane are not contiguous in m2"; return KS_EINVAL; }
      ++nst; ++s_in_plane;
      stick.push_back(make_int4(j, pmod(m3, P.n3), 0, 0));
    } else if (m3 != cur_m3 + 1) { err = "G sphere: a stick is not contiguous in m3"; return KS_EINVAL; }
    ++stick.back().z;
    cur_m1 = m1; cur_m2 = m2; cur_m3 = m3;
  }
  smax = std::max(smax, s_in_plane);
  plane_s0.push_back(nst);
  plane_pw0.push_back(P.npw);
  P.L1 = (int)plane_y0.size();
  P.x0 = pmod(mil[0], P.n1);
  P.nsticks = nst;
  P.smax = smax;
  if (P.L1 > P.n1 || smax > P.n2) { err = "G sphere larger than the grid"; return KS_EGRID; }
  int rc;
  if ((rc = upload(&P.d_plane_s0, plane_s0, err))) return rc;
  if ((rc = upload(&P.d_plane_y0, plane_y0, err))) return rc;
  if ((rc = upload(&P.d_plane_pw0, plane_pw0, err))) return rc;
  if ((rc = upload(&P.d_stick, stick, err))) return rc;
  if ((rc = upload(&P.d_g2, g2, err))) return rc;
  for (int ax = 0; ax < 3; ++ax) {
    const int n = grid[ax];
    std::vector<cplx> tw(n);
    for (int t = 0; t < n; ++t) {
      const double a = 2.0 * KS_PI * (double)t / (double)n;
      tw[t] = cmake(std::cos(a), std::sin(a));
    }
    if ((rc = upload(&P.d_tw[ax], tw, err))) return rc;
  }
  if ((rc = ks_hpsi_configure(P, err))) return rc;
  KS_CUDA_CHECK(cudaMalloc(&P.d_vperm, sizeof(double) * P.N), err);
  if ((rc = ks_build_vperm(P, vloc, c->stream, err))) return rc;
  c->fft_batch = auto_batch(P);
  // nonlocal part (Eq. 4)
  c->nproj = nproj; c->natom = natom;
  if (nproj > 0) {
    if (!beta || !off || !D || natom <= 0 || off[0] != 0 || off[natom] != nproj) { err = "bad projector arguments"; return KS_EINVAL; }
    KS_CUDA_CHECK(cudaMalloc(&c->d_beta, sizeof(cplx) * (size_t)nproj * P.npw), err);
    KS_CUDA_CHECK(cudaMemcpy(c->d_beta, beta, sizeof(cplx) * (size_t)nproj * P.npw, cudaMemcpyHostToDevice), err);
    std::vector<int> pa(nproj), offv(off, off + natom + 1);
    std::vector<long> doff(natom);
    long o = 0;
    for (int a = 0; a < natom; ++a) {
      const int np = off[a + 1] - off[a];
      if (np < 0) { err = "proj_offset not ascending"; return KS_EINVAL; }
      doff[a] = o;
      for (int p = off[a]; p < off[a + 1]; ++p) pa[p] = a;
      o += (long)np * np;
    }
    std::vector<double> Dv(D, D + o);
    if ((rc = upload(&c->d_proj_atom, pa, err))) return rc;
    if ((rc = upload(&c->d_off, offv, err))) return rc;
    if ((rc = upload(&c->d_doff, doff, err))) return rc;
    if ((rc = upload(&c->d_D, Dv, err))) return rc;
  }
  return KS_OK;
}

extern "C" int ks_create(ks_ctx** out, const double cell[9], const double k_frac[3], double ecutwfc, const int grid[3],
                         const ks_c128* vloc_g, int nproj, const ks_c128* beta, int natom, const int* proj_offset,
                         const double* D) {
  if (!out) return KS_EINVAL;
  *out = nullptr;
  if (!cell || !k_frac || !grid || !vloc_g || !(ecutwfc > 0) || nproj < 0 || grid[0] < 1 || grid[1] < 1 || grid[2] < 1) {
    ks_global_error() = "ks_create: bad argument";
    return KS_EINVAL;
  }
  ks_ctx* c = new (std::nothrow) ks_ctx;
  if (!c) return KS_ENOMEM;
  const int rc = create_impl(c, cell, k_frac, ecutwfc, grid, (const cplx*)vloc_g, nproj, (const cplx*)beta, natom, proj_offset, D);
  if (rc != KS_OK) {
    ks_global_error() = c->err;
    ks_destroy(c);
    return rc;
  }
  *out = c;
  return KS_OK;
}

extern "C" void ks_destroy(ks_ctx* c) {
  if (!c) return;
  HpsiPlan& P = c->P;
  cudaFree(P.d_plane_s0); cudaFree(P.d_plane_y0); cudaFree(P.d_plane_pw0); cudaFree(P.d_stick);
  cudaFree(P.d_g2); cudaFree(P.d_vperm); cudaFree(P.d_planes); cudaFree(P.d_rho_part);
  for (int i = 0; i < 3; ++i) cudaFree(P.d_tw[i]);
  cudaFree(c->d_beta); cudaFree(c->d_D); cudaFree(c->d_Q); cudaFree(c->d_proj_atom); cudaFree(c->d_off); cudaFree(c->d_doff);
  cudaFree(c->d_B); cudaFree(c->d_DB); cudaFree(c->d_hin); cudaFree(c->d_hout);
  for (int i = 0; i < 3; ++i) cudaFree(c->d_cheb[i]);
  if (c->s_in) {
    cudaStreamDestroy(c->s_in); cudaStreamDestroy(c->s_out); cudaEventDestroy(c->ev_start);
    for (int i = 0; i < 8; ++i) { cudaEventDestroy(c->ev_in[i]); cudaEventDestroy(c->ev_done[i]); }
  }
  cudaFree(c->gws.part);
  ks_eigh_free(&c->ews);
  ks_davidson_free(&c->dws);
  ks_kbatch_free(&c->kb);
  for (auto& r : c->krecs) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
  for (auto e : c->kpool) cudaEventDestroy(e);
  delete c;
}

extern "C" int ks_npw(const ks_ctx* c) { return c ? c->P.npw : KS_EINVAL; }
extern "C" int ks_set_stream(ks_ctx* c, void* s) {
  if (!c) return KS_EINVAL;
  c->stream = (cudaStream_t)s;
  return KS_OK;
}
extern "C" int ks_set_fft_batch(ks_ctx* c, int nbatch) {
  if (!c || nbatch < 0) return KS_EINVAL;
  cudaStreamSynchronize(c->stream);
  c->fft_batch = nbatch > 0 ? nbatch : auto_batch(c->P);
  if (c->P.d_planes && c->P.batch_cap > c->fft_batch) {      // shrink on request
    cudaFree(c->P.d_planes);
    c->P.d_planes = nullptr; c->P.batch_cap = 0; c->P.tmap_ok = false;
  }
  return KS_OK;
}
extern "C" const char* ks_last_error(const ks_ctx* c) { return c ? c->err.c_str() : ks_global_error().c_str(); }

// ------------------------------------------------------------------------------------------------
// H psi = local + kinetic (three FFT kernels per band batch) + nonlocal  beta D (beta^H psi)
// ------------------------------------------------------------------------------------------------
// H7: DB[:, b] = D B[:, b], D block diagonal per atom (Eq. 4); B, DB column-major nproj x nb
__global__ void k_apply_D(int nproj, int nb, const cplx* __restrict__ B, cplx* __restrict__ DB, const int* __restrict__ proj_atom,
                          const int* __restrict__ off, const long* __restrict__ doff, const double* __restrict__ D) {
  const long e = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (e >= (long)nproj * nb) return;
  const int p = (int)(e % nproj), b = (int)(e / nproj);
  const int a = proj_atom[p], p0 = off[a], np = off[a + 1] - p0;
  const double* Da = D + doff[a] + (long)(p - p0) * np;
  double sr = 0, si = 0;
  for (int q = 0; q < np; ++q) {
    const cplx v = B[(long)b * nproj + p0 + q];
    sr = fma(Da[q], v.x, sr);
    si = fma(Da[q], v.y, si);
  }
  DB[e] = cmake(sr, si);
}

int ks_ensure_nl(ks_ctx* c, int nb, int nsplit) {
  if (c->nproj == 0 || nb <= 0) return KS_OK;
  if (nb > c->nl_cap) {
    cudaFree(c->d_B); cudaFree(c->d_DB);
    c->d_B = c->d_DB = nullptr; c->nl_cap = 0;
    KS_CUDA_CHECK(cudaMalloc(&c->d_B, sizeof(cplx) * (size_t)c->nproj * nb), c->err);
    KS_CUDA_CHECK(cudaMalloc(&c->d_DB, sizeof(cplx) * (size_t)c->nproj * nb), c->err);
    c->nl_cap = nb;
  }
  const size_t need = sizeof(cplx) * (size_t)nsplit * c->nproj * nb;
  if (c->gws.bytes < need) {
    cudaFree(c->gws.part);
    c->gws.part = nullptr; c->gws.bytes = 0;
    KS_CUDA_CHECK(cudaMalloc(&c->gws.part, need), c->err);
    c->gws.bytes = need;
  }
  return KS_OK;
}

int ks_hpsi_impl(ks_ctx* c, const cplx* psi, cplx* hpsi, int nb) {
  if (!c) return KS_EINVAL;
  if (nb == 0) return KS_OK;   // empty block: nothing to do (pointers may be NULL)
  if (!psi || !hpsi || nb < 0) { c->err = "ks_hpsi: bad argument"; return KS_EINVAL; }
  const HpsiPlan& P = c->P;
  {
    const char* a = (const char*)psi;
    const char* b = (const char*)hpsi;
    const size_t bytes = sizeof(cplx) * (size_t)nb * P.npw;
    if (a < b + bytes && b < a + bytes) { c->err = "ks_hpsi: psi and hpsi must not alias"; return KS_EINVAL; }
  }
  {
    const int rc = ks_ensure_planes(c, nb, c->stream);
    if (rc) return rc;
  }
  for (int b0 = 0; b0 < nb; b0 += c->fft_batch) {
    const int n = std::min(c->fft_batch, nb - b0);
    for (int stage = 0; stage < 3; ++stage) {
      ks_kprof_begin(c, KP_INV_YZ + stage, 1);
      const int rc = ks_hpsi_local_launch(P, psi + (size_t)b0 * P.npw, hpsi + (size_t)b0 * P.npw, n, c->stream, c->err, stage);
      ks_kprof_end(c);
      if (rc) return rc;
    }
  }
  if (c->nproj > 0) {
    if (nb > c->nl_cap) {
      cudaFree(c->d_B); cudaFree(c->d_DB);
      c->d_B = c->d_DB = nullptr; c->nl_cap = 0;
      KS_CUDA_CHECK(cudaMalloc(&c->d_B, sizeof(cplx) * (size_t)c->nproj * nb), c->err);
      KS_CUDA_CHECK(cudaMalloc(&c->d_DB, sizeof(cplx) * (size_t)c->nproj * nb), c->err);
      c->nl_cap = nb;
    }
    ks_kprof_begin(c, KP_GEMM_HN, 2);
    int rc = ks_gemm_hn(c->stream, c->nproj, nb, P.npw, c->d_beta, P.npw, psi, P.npw, c->d_B, c->nproj, &c->gws, c->err);
    ks_kprof_end(c);
    if (rc) return rc;
    ks_kprof_begin(c, KP_APPLY_D, 1);
    k_apply_D<<<ceil_div((long)c->nproj * nb, 256), 256, 0, c->stream>>>(c->nproj, nb, c->d_B, c->d_DB, c->d_proj_atom,
                                                                         c->d_off, c->d_doff, c->d_D);
    ks_kprof_end(c);
    ks_kprof_begin(c, KP_GEMM_NN, 1);
    rc = ks_gemm_nn(c->stream, P.npw, nb, c->nproj, c->d_beta, P.npw, c->d_DB, c->nproj, hpsi, P.npw, 1, c->err);
    ks_kprof_end(c);
    if (rc) return rc;
  }
  KS_CUDA_CHECK(cudaGetLastError(), c->err);
  return KS_OK;
}

// S psi = psi + beta q (beta^H psi); the same three kernels as the nonlocal term
int ks_spsi_impl(ks_ctx* c, const cplx* psi, cplx* spsi, int nb) {
  if (!c) return KS_EINVAL;
  if (nb == 0) return KS_OK;
  if (!psi || !spsi || nb < 0) { c->err = "ks_spsi: bad argument"; return KS_EINVAL; }
  const HpsiPlan& P = c->P;
  const size_t bytes = sizeof(cplx) * (size_t)nb * P.npw;
  {
    const char* a = (const char*)psi;
    const char* b = (const char*)spsi;
    if (a < b + bytes && b < a + bytes) { c->err = "ks_spsi: psi and spsi must not alias"; return KS_EINVAL; }
  }
  KS_CUDA_CHECK(cudaMemcpyAsync(spsi, psi, bytes, cudaMemcpyDeviceToDevice, c->stream), c->err);
  if (!c->d_Q) return KS_OK;
  if (nb > c->nl_cap) {
    cudaFree(c->d_B); cudaFree(c->d_DB);
    c->d_B = c->d_DB = nullptr; c->nl_cap = 0;
    KS_CUDA_CHECK(cudaMalloc(&c->d_B, sizeof(cplx) * (size_t)c->nproj * nb), c->err);
    KS_CUDA_CHECK(cudaMalloc(&c->d_DB, sizeof(cplx) * (size_t)c->nproj * nb), c->err);
    c->nl_cap = nb;
  }
  int rc = ks_gemm_hn(c->stream, c->nproj, nb, P.npw, c->d_beta, P.npw, psi, P.npw, c->d_B, c->nproj, &c->gws, c->err);
  if (rc) return rc;
  k_apply_D<<<ceil_div((long)c->nproj * nb, 256), 256, 0, c->stream>>>(c->nproj, nb, c->d_B, c->d_DB, c->d_proj_atom, c->d_off,
                                                                       c->d_doff, c->d_Q);
  rc = ks_gemm_nn(c->stream, P.npw, nb, c->nproj, c->d_beta, P.npw, c->d_DB, c->nproj, spsi, P.npw, 1, c->err);
  if (rc) return rc;
  KS_CUDA_CHECK(cudaGetLastError(), c->err);
  return KS_OK;
}

extern "C" int ks_set_overlap(ks_ctx* c, const double* Q) {
  if (!c) return KS_EINVAL;
  cudaStreamSynchronize(c->stream);
  cudaFree(c->d_Q);
  c->d_Q = nullptr;
  if (!Q) return KS_OK;                       // back to S = I
  if (c->nproj == 0) { c->err = "ks_set_overlap: the context has no projectors"; return KS_EINVAL; }
  std::vector<int> off(c->natom + 1);
  KS_CUDA_CHECK(cudaMemcpy(off.data(), c->d_off, sizeof(int) * (c->natom + 1), cudaMemcpyDeviceToHost), c->err);
  size_t n = 0;
  for (int a = 0; a < c->natom; ++a) n += (size_t)(off[a + 1] - off[a]) * (off[a + 1] - off[a]);
  KS_CUDA_CHECK(cudaMalloc(&c->d_Q, sizeof(double) * n), c->err);
  KS_CUDA_CHECK(cudaMemcpy(c->d_Q, Q, sizeof(double) * n, cudaMemcpyHostToDevice), c->err);
  return KS_OK;
}

extern "C" int ks_spsi(ks_ctx* c, const ks_c128* psi, ks_c128* spsi, int nbands) {
  return ks_spsi_impl(c, (const cplx*)psi, (cplx*)spsi, nbands);
}

// ---- per-kernel event timing (bench.py's roofline object) ----
void ks_kprof_begin(ks_ctx* c, int phase, int launches) {
  c->klaunch[phase] += launches;
  if (!c->kprof_on) return;
  ks_ctx::KRec r;
  r.phase = phase;
  for (cudaEvent_t* e : {&r.a, &r.b}) {
    if (c->kpool.empty()) cudaEventCreate(e);
    else { *e = c->kpool.back(); c->kpool.pop_back(); }
  }
  cudaEventRecord(r.a, c->stream);
  c->krecs.push_back(r);
}
void ks_kprof_end(ks_ctx* c) {
  if (!c->kprof_on || c->krecs.empty()) return;
  cudaEventRecord(c->krecs.back().b, c->stream);
}
extern "C" int ks_profile_begin(ks_ctx* c) {
  if (!c) return KS_EINVAL;
  for (auto& r : c->krecs) { c->kpool.push_back(r.a); c->kpool.push_back(r.b); }
  c->krecs.clear();
  for (int i = 0; i < 8; ++i) c->klaunch[i] = 0;
  c->kprof_on = true;
  return KS_OK;
}
extern "C" int ks_profile_end(ks_ctx* c, double* ms, long long* launches) {
  if (!c || !ms || !launches) return KS_EINVAL;
  KS_CUDA_CHECK(cudaStreamSynchronize(c->stream), c->err);
  for (int i = 0; i < 8; ++i) { ms[i] = 0; launches[i] = c->klaunch[i]; }
  for (auto& r : c->krecs) {
    float t = 0;
    cudaEventElapsedTime(&t, r.a, r.b);
    ms[r.phase] += t;
    c->kpool.push_back(r.a); c->kpool.push_back(r.b);
  }
  c->krecs.clear();
  c->kprof_on = false;
  return KS_OK;
}

extern "C" int ks_hpsi(ks_ctx* c, const ks_c128* psi, ks_c128* hpsi, int nbands) {
  return ks_hpsi_impl(c, (const cplx*)psi, (cplx*)hpsi, nbands);
}

static int stage(ks_ctx* c, size_t bytes) {
  if (c->host_stage_bytes >= bytes) return KS_OK;
  cudaFree(c->d_hin); cudaFree(c->d_hout);
  c->d_hin = c->d_hout = nullptr; c->host_stage_bytes = 0;
  KS_CUDA_CHECK(cudaMalloc(&c->d_hin, bytes), c->err);
  KS_CUDA_CHECK(cudaMalloc(&c->d_hout, bytes), c->err);
  c->host_stage_bytes = bytes;
  return KS_OK;
}

// Host-buffer entry point, pipelined: the block is cut into up to 8 chunks of bands; chunk i+1 is copied in and chunk
// i-1 copied out (two copy streams) while chunk i is applied on the context's stream, so with pinned host buffers the
// PCIe transfers in both directions overlap the kernels.  Bands are independent in H psi: chunking changes no bit.
extern "C" int ks_hpsi_host(ks_ctx* c, const ks_c128* psi_host, ks_c128* hpsi_host, int nbands) {
  if (!c) return KS_EINVAL;
  if (!psi_host || !hpsi_host || nbands < 0) { c->err = "ks_hpsi_host: bad argument"; return KS_EINVAL; }
  if (nbands == 0) return KS_OK;
  const size_t npw = c->P.npw, bytes = sizeof(cplx) * (size_t)nbands * npw;
  int rc = stage(c, bytes);
  if (rc) return rc;
  if (!c->s_in) {
    KS_CUDA_CHECK(cudaStreamCreateWithFlags(&c->s_in, cudaStreamNonBlocking), c->err);
    KS_CUDA_CHECK(cudaStreamCreateWithFlags(&c->s_out, cudaStreamNonBlocking), c->err);
    KS_CUDA_CHECK(cudaEventCreateWithFlags(&c->ev_start, cudaEventDisableTiming), c->err);
    for (int i = 0; i < 8; ++i) {
      KS_CUDA_CHECK(cudaEventCreateWithFlags(&c->ev_in[i], cudaEventDisableTiming), c->err);
      KS_CUDA_CHECK(cudaEventCreateWithFlags(&c->ev_done[i], cudaEventDisableTiming), c->err);
    }
  }
  // chunk = a multiple of 32 bands (the GEMM tile unit: no padded columns inside a chunk), about eight chunks per block.
  // Measured (band-applications/s through host buffers): cfg 1, 160 bands: 32 -> 39.2k, 64 -> 37.9k, 40 -> 33.7k;
  // cfg 3, 520 bands: 64 -> 6.78k, 96 -> 6.58k, 128 -> 6.56k, 160 -> 6.62k, 65 (the old nbands/8 rule) -> 5.41k.
  // Round 2: graded chunks (small head and tail, 1.5x growth up to 224 bands in between, so that only a short first H2D and
  // last D2H stay exposed) measured SLOWER than uniform ones -- cfg 3 7.25k vs 7.49k, cfg 1 41.5k vs 42.1k, cfg 4 14.37k vs
  // 14.47k: a long chunk's H2D does not hide behind the shorter chunks before it.
  static const int env_per = getenv("KSPW_HOST_CHUNK_BANDS") ? atoi(getenv("KSPW_HOST_CHUNK_BANDS")) : 0;
  const int per = env_per > 0 ? env_per : std::max(32, nbands / 8 / 32 * 32);
  KS_CUDA_CHECK(cudaEventRecord(c->ev_start, c->stream), c->err);          // order after earlier work on the stream
  KS_CUDA_CHECK(cudaStreamWaitEvent(c->s_in, c->ev_start, 0), c->err);
  // The first chunk is half as long as the others: its H2D is the one copy that nothing hides.  Measured (band-applications/s
  // through host buffers, first chunk = the full / half / quarter of the others): cfg 3 (64-band chunks) 7.47k / 7.60k / 7.56k,
  // cfg 1 (32) 41.6k / 44.3k / 43.0k, cfg 4 (32) 14.4k / 15.5k / 14.9k.  KSPW_HOST_HEAD=<n> sets it.
  static const int env_head = getenv("KSPW_HOST_HEAD") ? atoi(getenv("KSPW_HOST_HEAD")) : 0;
  const int head = (env_head > 0 && env_head <= per) ? env_head : std::max(8, per / 2);
  for (int i = 0, b0 = 0, n = 0; b0 < nbands; ++i, b0 += n) {
    n = std::min(i == 0 ? head : per, nbands - b0);
    const size_t off = (size_t)b0 * npw, cb = sizeof(cplx) * (size_t)n * npw;
    KS_CUDA_CHECK(cudaMemcpyAsync(c->d_hin + off, (const cplx*)psi_host + off, cb, cudaMemcpyHostToDevice, c->s_in), c->err);
    KS_CUDA_CHECK(cudaEventRecord(c->ev_in[i & 7], c->s_in), c->err);
    KS_CUDA_CHECK(cudaStreamWaitEvent(c->stream, c->ev_in[i & 7], 0), c->err);
    rc = ks_hpsi_impl(c, c->d_hin + off, c->d_hout + off, n);
    if (rc) return rc;
    KS_CUDA_CHECK(cudaEventRecord(c->ev_done[i & 7], c->stream), c->err);
    KS_CUDA_CHECK(cudaStreamWaitEvent(c->s_out, c->ev_done[i & 7], 0), c->err);
    KS_CUDA_CHECK(cudaMemcpyAsync((cplx*)hpsi_host + off, c->d_hout + off, cb, cudaMemcpyDeviceToHost, c->s_out), c->err);
  }
  KS_CUDA_CHECK(cudaStreamSynchronize(c->s_out), c->err);
  KS_CUDA_CHECK(cudaStreamSynchronize(c->stream), c->err);
  return KS_OK;
}

// ------------------------------------------------------------------------------------------------
// density build: rho(r) = sum_b occ_b |psi_b(r)|^2, Eq. 31 L502 / Fig. 3
// ------------------------------------------------------------------------------------------------
extern "C" int ks_density(ks_ctx* c, const ks_c128* psi, const double* occ, int nbands, double* rho) {
  if (!c) return KS_EINVAL;
  if (!rho || nbands < 0 || (nbands > 0 && (!psi || !occ))) { c->err = "ks_density: bad argument"; return KS_EINVAL; }
  HpsiPlan& P = c->P;
  if (nbands == 0) {
    KS_CUDA_CHECK(cudaMemsetAsync(rho, 0, sizeof(double) * P.N, c->stream), c->err);
    return KS_OK;
  }
  {
    const int rc = ks_ensure_planes(c, nbands, c->stream);
    if (rc) return rc;
  }
  for (int b0 = 0; b0 < nbands; b0 += c->fft_batch) {
    const int n = std::min(c->fft_batch, nbands - b0);
    ks_kprof_begin(c, KP_RHO, 2);
    const int rc = ks_density_batch(P, (const cplx*)psi + (size_t)b0 * P.npw, occ + b0, n, b0 == 0, c->stream, c->err);
    ks_kprof_end(c);
    if (rc) return rc;
  }
  return ks_density_finish(P, rho, c->stream, c->err);
}

extern "C" int ks_density_host(ks_ctx* c, const ks_c128* psi_host, const double* occ_host, int nbands, double* rho_host) {
  if (!c) return KS_EINVAL;
  if (!rho_host || nbands < 0 || (nbands > 0 && (!psi_host || !occ_host))) { c->err = "ks_density_host: bad argument"; return KS_EINVAL; }
  const size_t bytes = sizeof(cplx) * (size_t)nbands * c->P.npw;
  const size_t rbytes = sizeof(double) * (size_t)c->P.N;
  int rc = stage(c, std::max(bytes, rbytes + sizeof(double) * (size_t)nbands));
  if (rc) return rc;
  double* d_rho = (double*)c->d_hout;
  double* d_occ = d_rho + c->P.N;
  if (nbands > 0) {
    KS_CUDA_CHECK(cudaMemcpyAsync(c->d_hin, psi_host, bytes, cudaMemcpyHostToDevice, c->stream), c->err);
    KS_CUDA_CHECK(cudaMemcpyAsync(d_occ, occ_host, sizeof(double) * nbands, cudaMemcpyHostToDevice, c->stream), c->err);
  }
  rc = ks_density(c, (const ks_c128*)c->d_hin, d_occ, nbands, d_rho);
  if (rc) return rc;
  KS_CUDA_CHECK(cudaMemcpyAsync(rho_host, d_rho, rbytes, cudaMemcpyDeviceToHost, c->stream), c->err);
  KS_CUDA_CHECK(cudaStreamSynchronize(c->stream), c->err);
  return KS_OK;
}

// ------------------------------------------------------------------------------------------------
// Chebyshev expansion: out = sum_n coef[n] T_n((H - ebar)/de) chi, three-term recurrence on
// ks_hpsi; the recurrence step and the accumulation are one fused elementwise kernel (96 B per plane wave and band).
// ------------------------------------------------------------------------------------------------
// first != 0:  t1 = (h - ebar t0)/de ;            out = c0 t0 + c1 t1     (tp holds t0, result t1 goes to tc)
// first == 0:  tn = 2 (h - ebar tc)/de - tp ;     out += cn tn            (tn overwrites tp)
__global__ void k_cheb_step(long n, const cplx* __restrict__ h, cplx* __restrict__ tp, cplx* __restrict__ tc,
                            cplx* __restrict__ out, double ebar, double inv_de, double c0, double cn, int first) {
  const long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (i >= n) return;
  const cplx hv = h[i];
  if (first) {
    const cplx t0 = tp[i];
    const cplx t1 = cmake((hv.x - ebar * t0.x) * inv_de, (hv.y - ebar * t0.y) * inv_de);
    tc[i] = t1;
    out[i] = cmake(fma(cn, t1.x, c0 * t0.x), fma(cn, t1.y, c0 * t0.y));
  } else {
    const cplx t = tc[i], q = tp[i], o = out[i];
    const cplx tn = cmake(2.0 * (hv.x - ebar * t.x) * inv_de - q.x, 2.0 * (hv.y - ebar * t.y) * inv_de - q.y);
    tp[i] = tn;
    out[i] = cmake(fma(cn, tn.x, o.x), fma(cn, tn.y, o.y));
  }
}
__global__ void k_scale_copy(long n, const cplx* __restrict__ a, double s, cplx* __restrict__ b) {
  const long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (i < n) b[i] = cmake(s * a[i].x, s * a[i].y);
}

extern "C" int ks_chebyshev(ks_ctx* c, const ks_c128* chi_, ks_c128* out_, int nbands, int ncoef, const double* coef,
                            double ebar, double de) {
  if (!c) return KS_EINVAL;
  if (nbands == 0) return KS_OK;
  if (!chi_ || !out_ || nbands < 0 || ncoef < 0 || (ncoef > 0 && !coef) || !(de > 0)) { c->err = "ks_chebyshev: bad argument"; return KS_EINVAL; }
  const cplx* chi = (const cplx*)chi_;
  cplx* out = (cplx*)out_;
  const long n = (long)nbands * c->P.npw;
  const size_t bytes = sizeof(cplx) * (size_t)n;
  {
    const char* a = (const char*)chi;
    const char* b = (const char*)out;
    if (a < b + bytes && b < a + bytes) { c->err = "ks_chebyshev: chi and out must not alias"; return KS_EINVAL; }
  }
  const int nblk = ceil_div(n, 256);
  if (ncoef < 2) {
    k_scale_copy<<<nblk, 256, 0, c->stream>>>(n, chi, ncoef == 1 ? coef[0] : 0.0, out);
    KS_CUDA_CHECK(cudaGetLastError(), c->err);
    return KS_OK;
  }
  if (c->cheb_bytes < bytes) {
    for (int i = 0; i < 3; ++i) { cudaFree(c->d_cheb[i]); c->d_cheb[i] = nullptr; }
    c->cheb_bytes = 0;
    for (int i = 0; i < 3; ++i) KS_CUDA_CHECK(cudaMalloc(&c->d_cheb[i], bytes), c->err);
    c->cheb_bytes = bytes;
  }
  cplx *tp = c->d_cheb[0], *tc = c->d_cheb[1], *h = c->d_cheb[2];
  KS_CUDA_CHECK(cudaMemcpyAsync(tp, chi, bytes, cudaMemcpyDeviceToDevice, c->stream), c->err);
  int rc = ks_hpsi_impl(c, tp, h, nbands);
  if (rc) return rc;
  k_cheb_step<<<nblk, 256, 0, c->stream>>>(n, h, tp, tc, out, ebar, 1.0 / de, coef[0], coef[1], 1);
  for (int k = 2; k < ncoef; ++k) {
    rc = ks_hpsi_impl(c, tc, h, nbands);
    if (rc) return rc;
    k_cheb_step<<<nblk, 256, 0, c->stream>>>(n, h, tp, tc, out, ebar, 1.0 / de, 0.0, coef[k], 0);
    std::swap(tp, tc);      // the new term went into tp: it is the current one now
  }
  KS_CUDA_CHECK(cudaGetLastError(), c->err);
  return KS_OK;
}

extern "C" int ks_davidson(ks_ctx* c, ks_c128* psi, double* eig, int nbands, double tol, int max_iter, double* resid,
                           int* iters_out, long long* band_applications_out) {
  return ks_davidson_impl(c, (cplx*)psi, eig, nbands, tol, max_iter, resid, iters_out, band_applications_out);
}

extern "C" int ks_cg(ks_ctx* c, ks_c128* psi, double* eig, int nbands, double tol, int kmaxiter, double* resid,
                     int* steps_out, long long* band_applications_out) {
  return ks_cg_impl(c, (cplx*)psi, eig, nbands, tol, kmaxiter, resid, steps_out, band_applications_out);
}

extern "C" int ks_davidson_host(ks_ctx* c, ks_c128* psi_host, double* eig_host, int nbands, double tol, int max_iter,
                                double* resid_host, int* iters_out, long long* band_applications_out) {
  if (!c) return KS_EINVAL;
  if (!psi_host || !eig_host || nbands < 1) { c->err = "ks_davidson_host: bad argument"; return KS_EINVAL; }
  const size_t bytes = sizeof(cplx) * (size_t)nbands * c->P.npw;
  int rc = stage(c, bytes);
  if (rc) return rc;
  double* d_e = (double*)c->d_hout;   // eig [nb] then resid [nb]
  KS_CUDA_CHECK(cudaMemcpyAsync(c->d_hin, psi_host, bytes, cudaMemcpyHostToDevice, c->stream), c->err);
  const int st = ks_davidson_impl(c, c->d_hin, d_e, nbands, tol, max_iter, d_e + nbands, iters_out, band_applications_out);
  if (st < 0) return st;
  KS_CUDA_CHECK(cudaMemcpyAsync(psi_host, c->d_hin, bytes, cudaMemcpyDeviceToHost, c->stream), c->err);
  KS_CUDA_CHECK(cudaMemcpyAsync(eig_host, d_e, sizeof(double) * nbands, cudaMemcpyDeviceToHost, c->stream), c->err);
  if (resid_host)
    KS_CUDA_CHECK(cudaMemcpyAsync(resid_host, d_e + nbands, sizeof(double) * nbands, cudaMemcpyDeviceToHost, c->stream), c->err);
  KS_CUDA_CHECK(cudaStreamSynchronize(c->stream), c->err);
  return st;
}

extern "C" int ks_davidson_profile(const ks_ctx* c, double* ms) {
  if (!c || !ms) return KS_EINVAL;
  for (int i = 0; i < 8; ++i) ms[i] = c->prof_ms[i];
  return KS_OK;
}

// ------------------------------------------------------------------------------------------------
// building blocks (unit tests, microbenchmarks)
// ------------------------------------------------------------------------------------------------
// one process-wide workspace behind a lock: these exports have no context to keep it in
static GemmWs g_gws;
static EighWs g_ews;
static std::mutex g_ws_lock;

extern "C" int ks_zgemm_hn(void* stream, int M, int N, int K, const ks_c128* A, long lda, const ks_c128* B, long ldb,
                           ks_c128* C, long ldc) {
  std::lock_guard<std::mutex> lk(g_ws_lock);
  return ks_gemm_hn((cudaStream_t)stream, M, N, K, (const cplx*)A, lda, (const cplx*)B, ldb, (cplx*)C, ldc, &g_gws, ks_global_error());
}
extern "C" int ks_zgemm_nn(void* stream, int M, int N, int K, const ks_c128* A, long lda, const ks_c128* B, long ldb,
                           ks_c128* C, long ldc, int accumulate) {
  return ks_gemm_nn((cudaStream_t)stream, M, N, K, (const cplx*)A, lda, (const cplx*)B, ldb, (cplx*)C, ldc, accumulate, ks_global_error());
}
extern "C" int ks_eigh(void* stream, int n, ks_c128* A, long lda, double* theta, ks_c128* C, long ldc, int* sweeps_out) {
  std::lock_guard<std::mutex> lk(g_ws_lock);
  return ks_eigh_run((cudaStream_t)stream, n, (cplx*)A, lda, theta, (cplx*)C, ldc, &g_ews, sweeps_out, ks_global_error());
}
extern "C" int ks_dmma_latency(double* clk_per_dmma, double sm_ghz) {
  if (!clk_per_dmma || !(sm_ghz > 0)) return KS_EINVAL;
  return ks_dmma_latency_run(clk_per_dmma, sm_ghz, ks_global_error());
}
extern "C" int ks_fp64_mix_peak(double* tflops4) {
  if (!tflops4) return KS_EINVAL;
  return ks_fp64_mix_run(tflops4, ks_global_error());
}
extern "C" int ks_dmma_peak(double* tflops_out, double* dfma_tflops_out) {
  return ks_peak_run(tflops_out, dfma_tflops_out, ks_global_error());
}
