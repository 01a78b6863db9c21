// batch.cu -- the multi-k entry points of include/kspw.h: ks_hpsi_batch, ks_davidson_batch.
//
// The KS equation is solved independently for every k-point of the Monkhorst-Pack mesh (Eq. 32 L507 per k;
// "independently for each k point" L900).  One k-point of a small cell is a small problem (cfg 2: 32 bands x 8.5k plane
// waves on a 54^3 grid): launched k after k, every kernel is a fraction of a wave and the path is launch-bound.
// ks_hpsi_batch takes the contexts of all k-points and runs H psi as ONE grid per kernel over (plane | column chunk | tile,
// band, k-point) for a GROUP of k-points at a time: the three FFT kernels read a per-k descriptor (their own sticks, live
// planes, |k+G|^2, workspace), the projector products are grouped GEMMs (one launch for beta^H psi of every k of the group,
// a fused split-K reduction + D apply, one launch for hpsi += beta (D B)).  By default all k-points form one group.
#include "ctx.h"
#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <thread>
#include <vector>

extern "C" {
typedef struct { double re, im; } ks_c128;
}

// H6 reduce + H7 fused, grouped: DB[p][b] = sum_q D[p][q] sum_z part[z][b][p0 + q]   (fixed order: deterministic)
struct NlProb {
  const cplx* part; cplx* DB;
  const int* proj_atom; const int* off; const long* doff; const double* D;
  int nproj, nb;
};
__global__ void k_reduce_applyD_g(const NlProb* __restrict__ probs, int nsplit) {
  const NlProb P = probs[blockIdx.y];
  const long e = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (e >= (long)P.nproj * P.nb) return;
  const int p = (int)(e % P.nproj), b = (int)(e / P.nproj);
  const int a = P.proj_atom[p], p0 = P.off[a], np = P.off[a + 1] - p0;
  const double* Da = P.D + P.doff[a] + (long)(p - p0) * np;
  const size_t MN = (size_t)P.nproj * P.nb;
  double sr = 0, si = 0;
  for (int q = 0; q < np; ++q) {
    const cplx* src = P.part + (size_t)b * P.nproj + p0 + q;
    double vr = 0, vi = 0;
    for (int z = 0; z < nsplit; ++z) { const cplx v = src[(size_t)z * MN]; vr += v.x; vi += v.y; }
    sr = fma(Da[q], vr, sr);
    si = fma(Da[q], vi, si);
  }
  P.DB[e] = cmake(sr, si);
}

static int kb_reserve(KBatchWs& w, size_t bytes, std::string& err) {
  if (w.bytes >= bytes) return KS_OK;
  if (w.h) cudaFreeHost(w.h);
  cudaFree(w.d);
  w.h = nullptr; w.d = nullptr; w.bytes = 0;
  bytes = std::max<size_t>(bytes * 2, 1 << 16);
  KS_CUDA_CHECK(cudaMallocHost(&w.h, bytes), err);
  KS_CUDA_CHECK(cudaMalloc(&w.d, bytes), err);
  if (!w.ev) KS_CUDA_CHECK(cudaEventCreateWithFlags(&w.ev, cudaEventDisableTiming), err);
  w.bytes = bytes;
  w.ev_pending = false;
  return KS_OK;
}

void ks_kbatch_free(KBatchWs* w) {
  if (w->h) cudaFreeHost(w->h);
  cudaFree(w->d);
  if (w->ev) cudaEventDestroy(w->ev);
  for (auto s : w->pool) cudaStreamDestroy(s);
  for (auto e : w->pool_ev) cudaEventDestroy(e);
  *w = KBatchWs();
}

// k-points per group.  Measured on cfg 2 (64 k x 32 bands, 54^3; band-applications/s): groups sized to keep their live
// planes in L2 (2 k-points, 76 MB) 273k; 4 k 335k; 8 k 387k; all 64 k in one group 467k -- a group small enough for L2 is a
// fraction of a wave per kernel and pays the drain / fill between dependent launches 3 x 32 times, so the default is ONE
// group (the planes stream through HBM as in the single-k path).  KSPW_KBATCH_GROUP fixes the count, KSPW_KBATCH_L2_MB
// sizes groups by the planes they hold.
static int group_size(ks_ctx* const* ctxs, int nk, const int* nbands) {
  static const int env_g = getenv("KSPW_KBATCH_GROUP") ? atoi(getenv("KSPW_KBATCH_GROUP")) : 0;
  if (env_g > 0) return std::min(env_g, nk);
  static const double l2_mb = getenv("KSPW_KBATCH_L2_MB") ? atof(getenv("KSPW_KBATCH_L2_MB")) : 0.0;
  if (!(l2_mb > 0)) return std::min(nk, 4096);
  double per = 0;
  for (int i = 0; i < nk; ++i) {
    const HpsiPlan& P = ctxs[i]->P;
    per = std::max(per, 16.0 * P.L1 * P.n2 * P.n3 * std::max(nbands[i], 1));
  }
  return std::max(1, std::min(nk, (int)(l2_mb * 1e6 / per)));
}

extern "C" int ks_hpsi_batch(ks_ctx* const* ctxs, int nk, const ks_c128* const* psi_, ks_c128* const* hpsi_, const int* nbands) {
  if (nk == 0) return KS_OK;
  if (!ctxs || nk < 0 || !ctxs[0]) return KS_EINVAL;
  ks_ctx* c0 = ctxs[0];
  std::string& err = c0->err;
  if (!psi_ || !hpsi_ || !nbands) { err = "ks_hpsi_batch: bad argument"; return KS_EINVAL; }
  const HpsiPlan& P0 = c0->P;
  int slab = 1 << 30, nbmax = 0;
  for (int i = 0; i < nk; ++i) {
    ks_ctx* c = ctxs[i];
    if (!c) { err = "ks_hpsi_batch: NULL context"; return KS_EINVAL; }
    if (c->P.n1 != P0.n1 || c->P.n2 != P0.n2 || c->P.n3 != P0.n3) { err = "ks_hpsi_batch: the k-points of a batch must share the FFT grid"; return KS_EINVAL; }
    for (int j = 0; j < i; ++j)
      if (ctxs[j] == c) { err = "ks_hpsi_batch: a context appears twice (its workspace would be shared)"; return KS_EINVAL; }
    if (nbands[i] < 0 || (nbands[i] > 0 && (!psi_[i] || !hpsi_[i]))) { err = "ks_hpsi_batch: bad argument"; return KS_EINVAL; }
    const char* a = (const char*)psi_[i];
    const char* b = (const char*)hpsi_[i];
    const size_t bytes = sizeof(cplx) * (size_t)nbands[i] * c->P.npw;
    if (bytes && a < b + bytes && b < a + bytes) { err = "ks_hpsi_batch: psi and hpsi must not alias"; return KS_EINVAL; }
    slab = std::min(slab, c->fft_batch);
    nbmax = std::max(nbmax, nbands[i]);
  }
  if (nbmax == 0) return KS_OK;
  cudaStream_t st = c0->stream;
  for (int i = 0; i < nk; ++i) {
    int rc = ks_ensure_planes(ctxs[i], std::min(nbands[i], slab), st);
    if (rc) { if (ctxs[i] != c0) err = ctxs[i]->err; return rc; }
  }
  const int G = group_size(ctxs, nk, nbands);
  const int ngroups = ceil_div(nk, G);
  // split count of the grouped beta^H psi (one value for the whole call: the problems are alike)
  int Mmax = 0, Kmax = 0;
  for (int i = 0; i < nk; ++i) { Mmax = std::max(Mmax, ctxs[i]->nproj); Kmax = std::max(Kmax, ctxs[i]->P.npw); }
  const int nsplit = Mmax > 0 ? ks_gemm_hn_group_nsplit(std::min(G, nk), Mmax, std::min(nbmax, slab), Kmax) : 1;
  for (int i = 0; i < nk && Mmax > 0; ++i) {
    int rc = ks_ensure_nl(ctxs[i], std::min(nbands[i], slab), nsplit);
    if (rc) { if (ctxs[i] != c0) err = ctxs[i]->err; return rc; }
  }
  // descriptor block: per group [FFT descriptors][GemmProb hn][NlProb][GemmProb nn], per band slab
  const int nslab = ceil_div(nbmax, slab);
  const size_t per_k = ks_kdesc_bytes(1) + 2 * sizeof(GemmProb) + sizeof(NlProb);
  const size_t total = per_k * (size_t)nk * nslab + 256 * (size_t)(ngroups * nslab * 4 + 4);
  KBatchWs& w = c0->kb;
  { int rc = kb_reserve(w, total, err); if (rc) return rc; }
  if (w.ev_pending) { KS_CUDA_CHECK(cudaEventSynchronize(w.ev), err); w.ev_pending = false; }   // the previous call's copy has left the pinned block
  struct GroupOff { size_t fft, hn, nl, nn; int i0, n, nb, b0; };
  std::vector<GroupOff> go;
  size_t off = 0;
  auto take = [&](size_t bytes) { const size_t o = off; off = (off + bytes + 255) & ~(size_t)255; return o; };
  std::vector<KItem> items(G);
  for (int s = 0; s < nslab; ++s) {
    const int b0 = s * slab;
    for (int g = 0; g < ngroups; ++g) {
      const int i0 = g * G, n = std::min(G, nk - i0);
      GroupOff o;
      o.i0 = i0; o.n = n; o.b0 = b0; o.nb = 0;
      for (int j = 0; j < n; ++j) {
        ks_ctx* c = ctxs[i0 + j];
        const int nb = std::max(0, std::min(slab, nbands[i0 + j] - b0));
        items[j].P = &c->P; items[j].nb = nb;
        items[j].psi = (const cplx*)psi_[i0 + j] + (size_t)b0 * c->P.npw;
        items[j].hpsi = (cplx*)hpsi_[i0 + j] + (size_t)b0 * c->P.npw;
        o.nb = std::max(o.nb, nb);
      }
      if (o.nb == 0) continue;
      o.fft = take(ks_kdesc_bytes(n));
      ks_kdesc_fill(w.h + o.fft, items.data(), n);
      o.hn = take(sizeof(GemmProb) * n); o.nl = take(sizeof(NlProb) * n); o.nn = take(sizeof(GemmProb) * n);
      GemmProb* hn = (GemmProb*)(w.h + o.hn);
      NlProb* nl = (NlProb*)(w.h + o.nl);
      GemmProb* nn = (GemmProb*)(w.h + o.nn);
      for (int j = 0; j < n; ++j) {
        ks_ctx* c = ctxs[i0 + j];
        const int nb = items[j].nb, npw = c->P.npw;
        hn[j].A = c->d_beta; hn[j].B = items[j].psi; hn[j].C = c->gws.part;
        hn[j].M = c->nproj; hn[j].N = nb; hn[j].K = npw; hn[j].lda = npw; hn[j].ldb = npw; hn[j].ldc = c->nproj;
        nl[j].part = c->gws.part; nl[j].DB = c->d_DB; nl[j].proj_atom = c->d_proj_atom; nl[j].off = c->d_off;
        nl[j].doff = c->d_doff; nl[j].D = c->d_D; nl[j].nproj = c->nproj; nl[j].nb = nb;
        nn[j].A = c->d_beta; nn[j].B = c->d_DB; nn[j].C = items[j].hpsi;
        nn[j].M = npw; nn[j].N = nb; nn[j].K = c->nproj; nn[j].lda = npw; nn[j].ldb = c->nproj; nn[j].ldc = npw;
      }
      go.push_back(o);
    }
  }
  KS_CUDA_CHECK(cudaMemcpyAsync(w.d, w.h, off, cudaMemcpyHostToDevice, st), err);
  KS_CUDA_CHECK(cudaEventRecord(w.ev, st), err);
  w.ev_pending = true;
  for (const GroupOff& o : go) {
    for (int j = 0; j < o.n; ++j) {
      ks_ctx* c = ctxs[o.i0 + j];
      items[j].P = &c->P; items[j].nb = std::max(0, std::min(slab, nbands[o.i0 + j] - o.b0));
    }
    for (int stage = 0; stage < 3; ++stage) {
      ks_kprof_begin(c0, KP_INV_YZ + stage, 1);
      const int rc = ks_hpsi_local_launch_k(items.data(), o.n, w.d + o.fft, st, err, stage);
      ks_kprof_end(c0);
      if (rc) return rc;
    }
    int M = 0, npwmax = 0;
    for (int j = 0; j < o.n; ++j) { M = std::max(M, ctxs[o.i0 + j]->nproj); npwmax = std::max(npwmax, ctxs[o.i0 + j]->P.npw); }
    if (M > 0) {
      ks_kprof_begin(c0, KP_GEMM_HN, 1);
      int rc = ks_gemm_hn_group(st, (const GemmProb*)(w.d + o.hn), o.n, M, o.nb, nsplit, err);
      ks_kprof_end(c0);
      if (rc) return rc;
      ks_kprof_begin(c0, KP_APPLY_D, 1);
      k_reduce_applyD_g<<<dim3(ceil_div((long)M * o.nb, 256), o.n), 256, 0, st>>>((const NlProb*)(w.d + o.nl), nsplit);
      ks_kprof_end(c0);
      ks_kprof_begin(c0, KP_GEMM_NN, 1);
      rc = ks_gemm_nn_group(st, (const GemmProb*)(w.d + o.nn), o.n, npwmax, o.nb, 1, err);
      ks_kprof_end(c0);
      if (rc) return rc;
    }
  }
  KS_CUDA_CHECK(cudaGetLastError(), err);
  return KS_OK;
}

// Block Davidson on every k-point (independent solves).  Each solve is a host-driven iteration with a few
// blocking reads per step; the solves run on a pool of worker threads, one CUDA stream each, so the host waits of one
// k-point overlap the kernels of the others.  Results as ks_davidson, per k.
extern "C" int ks_davidson_batch(ks_ctx* const* ctxs, int nk, ks_c128* const* psi, double* const* eig, const int* nbands, double tol,
                                 int max_iter, double* const* resid, int* iters_out, long long* band_applications_out,
                                 int* status_out) {
  if (nk == 0) return KS_OK;
  if (!ctxs || nk < 0 || !ctxs[0]) return KS_EINVAL;
  ks_ctx* c0 = ctxs[0];
  if (!psi || !eig || !nbands) { c0->err = "ks_davidson_batch: bad argument"; return KS_EINVAL; }
  for (int i = 0; i < nk; ++i) {
    if (!ctxs[i] || !psi[i] || !eig[i]) { c0->err = "ks_davidson_batch: bad argument"; return KS_EINVAL; }
    for (int j = 0; j < i; ++j)
      if (ctxs[j] == ctxs[i]) { c0->err = "ks_davidson_batch: a context appears twice"; return KS_EINVAL; }
  }
  static const int env_t = getenv("KSPW_KBATCH_THREADS") ? atoi(getenv("KSPW_KBATCH_THREADS")) : 0;
  const int nt = std::max(1, std::min(nk, env_t > 0 ? env_t : 8));
  KBatchWs& w = c0->kb;
  while ((int)w.pool.size() < nt) {
    cudaStream_t s; cudaEvent_t e;
    KS_CUDA_CHECK(cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking), c0->err);
    KS_CUDA_CHECK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming), c0->err);
    w.pool.push_back(s); w.pool_ev.push_back(e);
  }
  if (!w.ev) KS_CUDA_CHECK(cudaEventCreateWithFlags(&w.ev, cudaEventDisableTiming), c0->err);
  int dev = 0;
  KS_CUDA_CHECK(cudaGetDevice(&dev), c0->err);
  // the solves start after the work already enqueued on the first context's stream
  cudaEvent_t start;
  KS_CUDA_CHECK(cudaEventCreateWithFlags(&start, cudaEventDisableTiming), c0->err);
  KS_CUDA_CHECK(cudaEventRecord(start, c0->stream), c0->err);
  for (int t = 0; t < nt; ++t) KS_CUDA_CHECK(cudaStreamWaitEvent(w.pool[t], start, 0), c0->err);
  std::vector<int> st(nk, KS_OK);
  std::vector<std::thread> th;
  for (int t = 0; t < nt; ++t)
    th.emplace_back([&, t]() {
      cudaSetDevice(dev);
      for (int i = t; i < nk; i += nt) {
        ks_ctx* c = ctxs[i];
        const cudaStream_t keep = c->stream;
        c->stream = w.pool[t];
        st[i] = ks_davidson_impl(c, (cplx*)psi[i], eig[i], nbands[i], tol, max_iter, resid ? resid[i] : nullptr,
                                 iters_out ? iters_out + i : nullptr, band_applications_out ? band_applications_out + i : nullptr);
        c->stream = keep;
      }
      cudaEventRecord(w.pool_ev[t], w.pool[t]);
    });
  for (auto& x : th) x.join();
  for (int t = 0; t < nt; ++t) cudaStreamWaitEvent(c0->stream, w.pool_ev[t], 0);
  cudaEventDestroy(start);
  int worst = KS_OK;
  for (int i = 0; i < nk; ++i) {
    if (status_out) status_out[i] = st[i];
    if (st[i] < 0) { if (worst >= 0) { worst = st[i]; if (ctxs[i] != c0) c0->err = ctxs[i]->err; } }
    else if (st[i] > 0 && worst == KS_OK) worst = st[i];
  }
  return worst;
}
