// hpsi_kernels.cu -- the dual-space local part of H*psi (DESIGN.md steps H1-H5) as three kernels, and the density
// build that reuses the first one and a half of them:
//
//   k_inv_yz  per (band, live x-plane): the first z codelet pass reads each stick's contiguous run of psi straight
//             from global memory (H1: no zero fill, no scatter pass), inverse FFT along z on the sticks only, then
//             along y for the plane (H2, pruned: PAPER.md Eq. 31, e^{+i}); the last y pass writes the live plane
//             [y'][z'] from registers.
//   k_x       per (32 (y',z') columns, group of bands): inverse FFT along x from the live planes (dead rows are zeros
//             in registers), multiply by V(r) (H3, Eq. 32), forward FFT along x, live planes written back in
//             place from registers; the next band's live rows are prefetched by cp.async into the tile rows the same
//             thread owns.  The full n1*n2*n3 cube never exists in HBM.
//   k_fwd_yz  per (band, live x-plane): forward FFT along y, keep the stick columns, forward FFT along z
//             (H4, Eq. 36, e^{-i} and 1/N); the last z pass writes hpsi = |k+G|^2 psi + (.)/N straight to the
//             stick's run of hpsi (H5: gather and kinetic term fused).
//   k_rho     the first half of k_x with occ |psi(r)|^2 accumulated over bands (ks_density).
//
// All intermediates are in "position" order (fft.cuh): type-A transforms leave their output transposed, type-B
// transforms consume exactly that order, and V(r) is stored permuted once at ks_create, so no reordering pass exists.
// A tile crosses shared memory only between codelet passes; thread t works on column t % ZC and codelet lines
// t / ZC, t / ZC + G, ... (stick passes: lines-first over (stick, line) with an odd stick stride), so every
// shared-memory offset is a compile-time multiple of the chunk width plus one per-thread base and the 16-byte accesses
// of a quarter-warp fall in distinct banks.
#include "fft.cuh"
#include "plan.h"
#include <cuda.h>          // CUtensorMap and its enums only; the driver entry point is looked up at run time
#include <algorithm>
#include <type_traits>
#include <cmath>
#include <cstdlib>
#include <vector>
#include <cooperative_groups.h>
namespace cg = cooperative_groups;


cudaError_t ks_fft_init_constants() {
  static bool done = false;
  if (done) return cudaSuccess;
  std::vector<double2> w(KS_WTAB);
  const double PI = 3.14159265358979323846264338327950288;
  for (int t = 0; t < KS_WTAB; ++t) {
    // exact quarter-turn symmetry: evaluate in the first octant
    const double a = 2.0 * PI * (double)t / (double)KS_WTAB;
    w[t] = make_double2(std::cos(a), std::sin(a));
  }
  cudaError_t e = cudaMemcpyToSymbol(c_wtab, w.data(), sizeof(double2) * KS_WTAB);
  if (e == cudaSuccess) done = true;
  return e;
}

// ------------------------------------------------------------------------------------------------
// supported sizes
// ------------------------------------------------------------------------------------------------
#define KS_X_SIZES(X) X(16) X(18) X(20) X(24) X(32) X(36) X(40) X(48) X(54) X(60) X(64) X(72) X(80) X(96) X(100) X(120) X(128)
#define KS_YZ_PAIRS(X) \
  X(16, 16) X(18, 18) X(24, 24) X(32, 32) X(36, 36) X(48, 48) X(54, 54) X(64, 64) X(72, 72) \
  X(96, 96) X(128, 128) X(18, 64) X(96, 288) X(20, 20) X(40, 40) X(60, 60) X(80, 80) X(100, 100) X(120, 120)

void ks_fft_factors(int n, int* R1, int* R2, int axis) {
  *R1 = 0; *R2 = 0;
  switch (n) {
#define C_(N_) case N_: *R1 = (axis == 2) ? facz<N_>::R1 : fac<N_>::R1; *R2 = (axis == 2) ? facz<N_>::R2 : fac<N_>::R2; break;
    C_(16) C_(18) C_(20) C_(24) C_(32) C_(36) C_(40) C_(48) C_(54) C_(60) C_(64) C_(72) C_(80) C_(96) C_(100) C_(120) C_(128) C_(144) C_(192) C_(256) C_(288)
#undef C_
    default: break;
  }
}
bool ks_fft_size_supported(int n) {
#define C_(N_) if (n == N_) return true;
  KS_X_SIZES(C_)
#undef C_
  return false;
}
bool ks_fft_yz_supported(int n2, int n3) {
#define C_(A_, B_) if (n2 == A_ && n3 == B_) return true;
  KS_YZ_PAIRS(C_)
#undef C_
  return false;
}
int ks_fft_sizes(int* out, int cap) {
  const int all[] = {
#define C_(N_) N_,
      KS_X_SIZES(C_)
#undef C_
  };
  const int n = (int)(sizeof(all) / sizeof(int));
  for (int i = 0; i < n && i < cap; ++i) out[i] = all[i];
  return n;
}

// ------------------------------------------------------------------------------------------------
// create-time kernels: plain DFT along one axis (O(N n)), permute + realness check
// ------------------------------------------------------------------------------------------------
__global__ void k_dft_axis(const cplx* __restrict__ in, cplx* __restrict__ out, long N, int n, long stride,
                           const cplx* __restrict__ tw) {
  const long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int k = (int)((i / stride) % n);
  const long base = i - (long)k * stride;
  double sr = 0, si = 0;
  for (int j = 0; j < n; ++j) {
    const cplx a = in[base + (long)j * stride];
    const cplx w = tw[(int)(((long)j * k) % n)];
    sr += a.x * w.x - a.y * w.y;
    si += a.x * w.y + a.y * w.x;
  }
  out[i] = cmake(sr, si);
}

__global__ void k_vperm(const cplx* __restrict__ v, double* __restrict__ vperm, int n1, int n2, int n3,
                        int a1, int b1, int a2, int b2, int a3, int b3, double* __restrict__ maxes) {
  const long N = (long)n1 * n2 * n3;
  const long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
  double re = 0, im = 0;
  if (i < N) {
    const int pz = (int)(i % n3), py = (int)((i / n3) % n2), px = (int)(i / ((long)n3 * n2));
    const int x = perm_index(px, a1, b1), y = perm_index(py, a2, b2), z = perm_index(pz, a3, b3);
    const cplx a = v[((long)x * n2 + y) * n3 + z];
    vperm[i] = a.x;
    re = fabs(a.x); im = fabs(a.y);
  }
  // block max -> atomicMax on the bit pattern (non-negative doubles order like unsigned integers)
  for (int o = 16; o > 0; o >>= 1) {
    re = fmax(re, __shfl_xor_sync(0xffffffffu, re, o));
    im = fmax(im, __shfl_xor_sync(0xffffffffu, im, o));
  }
  if ((threadIdx.x & 31) == 0) {
    atomicMax((unsigned long long*)&maxes[0], (unsigned long long)__double_as_longlong(re));
    atomicMax((unsigned long long*)&maxes[1], (unsigned long long)__double_as_longlong(im));
  }
}

struct VpermTmp {     // create-time temporaries, released on every return path
  cplx *a = nullptr, *b = nullptr;
  double* mx = nullptr;
  ~VpermTmp() { cudaFree(a); cudaFree(b); cudaFree(mx); }
};

int ks_build_vperm(HpsiPlan& P, const cplx* vhat_host, cudaStream_t st, std::string& err) {
  const long N = P.N;
  VpermTmp tmp;
  cplx *&a = tmp.a, *&b = tmp.b;
  double*& mx = tmp.mx;
  KS_CUDA_CHECK(cudaMalloc(&a, N * sizeof(cplx)), err);
  KS_CUDA_CHECK(cudaMalloc(&b, N * sizeof(cplx)), err);
  KS_CUDA_CHECK(cudaMalloc(&mx, 2 * sizeof(double)), err);
  KS_CUDA_CHECK(cudaMemsetAsync(mx, 0, 2 * sizeof(double), st), err);
  KS_CUDA_CHECK(cudaMemcpyAsync(a, vhat_host, N * sizeof(cplx), cudaMemcpyHostToDevice, st), err);
  const int nn[3] = {P.n1, P.n2, P.n3};
  const long stv[3] = {(long)P.n2 * P.n3, (long)P.n3, 1};
  const int nblk = ceil_div(N, 256);
  for (int ax = 0; ax < 3; ++ax) {
    k_dft_axis<<<nblk, 256, 0, st>>>(a, b, N, nn[ax], stv[ax], P.d_tw[ax]);
    std::swap(a, b);
  }
  int f[6];
  for (int ax = 0; ax < 3; ++ax) ks_fft_factors(nn[ax], &f[2 * ax], &f[2 * ax + 1], ax);
  k_vperm<<<nblk, 256, 0, st>>>(a, P.d_vperm, P.n1, P.n2, P.n3, f[0], f[1], f[2], f[3], f[4], f[5], mx);
  double h[2];
  KS_CUDA_CHECK(cudaMemcpyAsync(h, mx, sizeof h, cudaMemcpyDeviceToHost, st), err);
  KS_CUDA_CHECK(cudaStreamSynchronize(st), err);
  if (h[1] > 1e-12 * h[0] && h[1] > 0.0) {
    char buf[160];
    snprintf(buf, sizeof buf, "V(r) is not real: max|Im| = %.3e, max|Re| = %.3e", h[1], h[0]);
    err = buf;
    return KS_EVLOC;
  }
  return KS_OK;
}

// ------------------------------------------------------------------------------------------------
// yz kernels: one CTA per (band, live x-plane)
// ------------------------------------------------------------------------------------------------
// Shared memory: tw_y[NY], tw_z[NZ], stile[smax][NZ|1] (the plane's z-sticks), ytile[NY][ZC] (one chunk of
// z' positions during the y transform).  The first codelet pass of the inverse kernel reads psi straight
// from global memory (a stick's coefficients are a contiguous run of psi: no zero fill, no scatter pass,
// no index array), the last pass of the forward kernel writes hpsi straight from registers (gather,
// 1/N and the kinetic term fused).  Stick passes map threads lines-first over (stick, codelet line) with an
// odd stick stride; y passes map thread t to column t % ZC and lines t / ZC, t / ZC + G, ...
struct YzArgs {
  const cplx* psi;      // [nb][npw]
  cplx* hpsi;           // [nb][npw] (forward kernel only)
  cplx* planes;         // [nb][L1][NY][NZ]
  const int* plane_s0;  // [L1+1] first stick of each plane
  const int* plane_y0;  // [L1]   natural y index of the plane's first stick
  const int* plane_pw0; // [L1+1] first plane wave of each plane: a plane's coefficients are ONE contiguous run of psi
  const int4* stick;    // [nsticks] {first PW, natural z index of the first PW, number of PWs, 0}
  const double* g2;
  const cplx* tw_y;
  const cplx* tw_z;
  int npw, L1, smax;
  int nb;               // bands of this k-point (k-batched launches: CTAs beyond it leave at once)
  int pf_dist;          // L2 prefetch distance in CTAs (0 = off), see inv_yz_body / fwd_yz_body
  double invN;
};

constexpr int yz_pick_zc(int nz) {
  for (int zc = 32; zc >= 1; --zc)
    if (nz % zc == 0) return zc;
  return 1;
}
// DBF: the forward kernel splits the y tile into two half-width buffers filled by cp.async one chunk ahead (pays
// when two CTAs fit per SM; measured: 96x96 213 -> 201 us; 128x128 224 -> 254 us and 96x288 337 -> 376 us, where one CTA fills the SM: off there)
// ZS > 1: the z' positions of a plane are split over ZS CTAs (blockIdx.x = lx * ZS + h).  Position p = k1 * R2z + k2, so
// CTA h owns the codelet lines k1 in [h, h + 1) * R1z / ZS and holds only that part of every stick: the stick tile shrinks by
// ZS and two CTAs fit per SM where the whole plane's sticks filled it (128 x 128: 126 KB, 96 x 288: 190 KB of sticks).
// The inverse kernel repeats the first z codelet pass in every CTA of the plane (it needs no exchange); the forward kernel's
// last z pass needs all k1, so its ZS CTAs form a thread-block cluster and read each other's stick tiles through
// distributed shared memory.
// NG > 1: during the y transform the CTA's warps form NG independent groups of NT / NG threads; group q transforms the chunks
// q, q + NG, ... in its own y tile and synchronises with a named barrier of its own, so the groups drift apart and one
// group's global loads / stores overlap another's codelets (a single CTA per SM otherwise moves through load, compute and
// store phases in lockstep).  ZC is the chunk width of ONE group; the y tiles of all groups take NY * ZC * NG elements.
// TMA: the inverse kernel's last y pass runs in place in the y tile and the tile leaves for HBM as bulk asynchronous copies
// (one per plane row, issued by NY threads, SASS UBLKCP) instead of 16-byte stores from registers: the per-thread stores kept
// the CTA in a store phase for a third of its time (measured with clock64: 9.5k of 26.8k clocks per 128 x 128 plane) during
// which the LSU queue was full and nothing else progressed; the bulk copies drain while the next chunk is transformed.
template <int NY, int NZ> struct yzcfg { static constexpr int ZC = yz_pick_zc(NZ), NT = 256, ZS = 1, NG = 1; static constexpr bool DBF = (ZC % 2 == 0), TMA = false; };
#ifdef KSPW_ZSPLIT128   // measured on cfg 3 (104-band launches; unsplit: k_inv_yz 0.589 ms, k_fwd_yz 0.688 ms):
                        //   ZS = 2, ZC = 16, 256 threads: k_inv_yz 0.589 ms, k_fwd_yz 0.843 ms
                        //   ZS = 4, ZC = 32, 256 threads (both y passes fill the CTA): k_inv_yz 0.794 ms (the repeated first
                        //   z pass), k_fwd_yz 1.439 ms (clusters of 4 with two cluster barriers each)  -> off
template <> struct yzcfg<128, 128> { static constexpr int ZC = 32, NT = 256, ZS = 4, NG = 1; static constexpr bool DBF = false, TMA = false; };
#else
#ifdef KSPW_YZ128_NT256   // 8 warps, both y passes fill the CTA: k_inv_yz 0.605 ms (0.589 with 512 threads), k_fwd_yz 0.819 ms (0.688): off
template <> struct yzcfg<128, 128> { static constexpr int ZC = 32, NT = 256, ZS = 1, NG = 1; static constexpr bool DBF = false, TMA = false; };
#else
#ifndef KSPW_YZ128_NG
#define KSPW_YZ128_NG 4
#endif
#ifndef KSPW_NO_YHALF_INV
#define KSPW_YHALF_INV       // with four y groups the even/odd split of the DFT-16 pass pays in the inverse kernel too (0.628 -> 0.574 ms)
#endif
#ifndef KSPW_YZ128_TMA
#define KSPW_YZ128_TMA 0     // measured (cfg 3, k_inv_yz per 104 bands): register stores 0.574 ms; one tensor store per chunk 0.600-0.649 ms;
#endif                       // 128 row-wise cp.async.bulk per chunk 0.687-0.745 ms -- see DESIGN.md section 5
template <> struct yzcfg<128, 128> { static constexpr int NG = KSPW_YZ128_NG, ZC = 32 / NG, NT = 512, ZS = 1; static constexpr bool DBF = false, TMA = (KSPW_YZ128_TMA != 0); };
#endif
#endif
#ifndef KSPW_NO_ZSPLIT288
template <> struct yzcfg<96, 288> { static constexpr int ZC = 16, NT = 256, ZS = 3, NG = 1; static constexpr bool DBF = false, TMA = false; };
#else
template <> struct yzcfg<96, 288> { static constexpr int ZC = 16, NT = 256, ZS = 1, NG = 1; static constexpr bool DBF = false, TMA = false; };
#endif

// 16-byte global -> shared async copy (LDGSTS), ordered against the surrounding shared-memory accesses
__device__ __forceinline__ void cp16m(cplx* smem, const cplx* gmem) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_commit_m() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void cp_wait_n(int n) {   // n = groups allowed to stay in flight (uniform per thread)
  switch (n) {
    case 0: asm volatile("cp.async.wait_group 0;\n" ::: "memory"); break;
    case 1: asm volatile("cp.async.wait_group 1;\n" ::: "memory"); break;
    case 2: asm volatile("cp.async.wait_group 2;\n" ::: "memory"); break;
    default: asm volatile("cp.async.wait_group 3;\n" ::: "memory"); break;
  }
}

// plane elements are written once by k_inv_yz and read once by k_fwd_yz: streaming (evict-first) accesses
#ifdef KSPW_PLANE_CS
#define KS_ST_PLANE(p, v) __stcs((p), (v))
#define KS_LD_PLANE(p) __ldcs(p)
#else
#define KS_ST_PLANE(p, v) (*(p) = (v))
#define KS_LD_PLANE(p) (*(p))
#endif


#ifdef KSPW_PHASE_CLOCKS   // experiment: SM clocks per phase of the yz kernels, summed over CTAs (thread 0 of each CTA)
__device__ unsigned long long g_phase[16];
#define KS_PH_INIT() unsigned long long ph_t = clock64()
#define KS_PH(i_) do { if (threadIdx.x == 0) { const unsigned long long t_ = clock64(); atomicAdd(&g_phase[i_], t_ - ph_t); ph_t = t_; } } while (0)
extern "C" int ks_debug_phase_clocks(unsigned long long* out, int reset) {
  cudaMemcpyFromSymbol(out, g_phase, sizeof(g_phase));
  if (reset) { unsigned long long z[16] = {0}; cudaMemcpyToSymbol(g_phase, z, sizeof(z)); }
  return 0;
}
#else
#define KS_PH_INIT()
#define KS_PH(i_)
#endif

// ---- bulk asynchronous copies (TMA engine, SASS UBLKCP): shared -> global stores tracked by bulk async-groups ----
__device__ __forceinline__ void bulk_store(void* gmem, const void* smem, unsigned bytes) {     // 16-byte aligned, bytes % 16 == 0
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;\n" ::"l"(gmem), "r"(s), "r"(bytes) : "memory");
}
// one 2-D box [rows][cols] of a tensor map, shared -> global (SASS UTMASTG); x = column (fastest), y = row coordinate
__device__ __forceinline__ void tensor_store_2d(const void* tmap, const void* smem, int x, int y) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%2, %3}], [%1];\n" ::"l"(tmap), "r"(s), "r"(x), "r"(y) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;\n" ::: "memory"); }
// the issuing thread's bulk groups have finished READING their shared-memory source (the buffer may be overwritten)
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;\n" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;\n" ::: "memory"); }
// generic-proxy writes to shared memory made visible to the async proxy (before a barrier that precedes the bulk copy)
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }

// barrier of one y group (named barrier 1 + q over GT threads) or of the whole CTA when there is one group
template <int NG, int GT>
__device__ __forceinline__ void ygroup_sync(int q) {
  if constexpr (NG == 1) __syncthreads();
  else asm volatile("bar.sync %0, %1;" ::"r"(1 + q), "n"(GT) : "memory");
}

// lines-first walk over (stick s, line j) pairs: item it = j*S + s, it = tid, tid + NT, ...
struct StickWalk {
  int s, j, ds, dj, S;
  __device__ __forceinline__ StickWalk(int tid, int nt, int S_) : S(S_) {
    s = tid % S; j = tid / S; ds = nt % S; dj = nt / S;
  }
  __device__ __forceinline__ void next() {
    s += ds; j += dj;
    if (s >= S) { s -= S; ++j; }
  }
};

// line-first walk over (stick s, line j) pairs, j fastest: item it = s*L + j, it = start, start + step, ...  Used where a
// thread's line touches GLOBAL memory at psi[first + j1*L + j - z0]: the L lanes of one stick read or write consecutive
// plane waves (one or two 128-byte lines per stick instead of one line per lane)
template <int L>
struct JWalk {
  int s, j, it, step;
  __device__ __forceinline__ JWalk(int start, int step_) : it(start), step(step_) { s = it / L; j = it % L; }
  __device__ __forceinline__ void next() { it += step; s = it / L; j = it % L; }
};

template <bool JFAST, int L>
__device__ __forceinline__ typename std::conditional<JFAST, JWalk<L>, StickWalk>::type make_walk(int tid, int nt, int S) {
  if constexpr (JFAST) return JWalk<L>(tid, nt);
  else return StickWalk(tid, nt, S);
}

template <int NY, int NZ, bool USE_TMA>
__device__ __forceinline__ void inv_yz_body(const YzArgs& a, const int bx, const int b, const void* tmap) {
  constexpr int R1y = fac<NY>::R1, R2y = fac<NY>::R2, R1z = facz<NZ>::R1, R2z = facz<NZ>::R2;
  constexpr int ZS = yzcfg<NY, NZ>::ZS, NZH = NZ / ZS, K1H = R1z / ZS;   // this CTA's z' positions and codelet lines
  static_assert(R1z % ZS == 0 && NZH % yzcfg<NY, NZ>::ZC == 0, "z' split must cut between codelet lines and chunks");
  constexpr int SZ = NZH | 1, ZC = yzcfg<NY, NZ>::ZC, NT = yzcfg<NY, NZ>::NT, NG = yzcfg<NY, NZ>::NG, GT = NT / NG, G = GT / ZC;
  static_assert(NT % NG == 0 && GT % 32 == 0 && (NZH / ZC) % NG == 0, "y groups: whole warps, equal numbers of chunks");
#ifdef KSPW_YHALF_INV   // measured on cfg 3: k_inv_yz 0.589 -> 0.607 ms (twice the stick-tile reads in the pass, 128 registers): off
  constexpr bool YHALF = (G == 2 * R2y) && (R1y % 2 == 0) && (GT == G * ZC) && (ZC * NG == 32);
#else
  constexpr bool YHALF = false;
#endif
  extern __shared__ __align__(128) cplx sm[];
  cplx* ytile = sm;                               // first: the source of the tensor stores must be 128-byte aligned
  cplx* tw_y = ytile + NY * ZC * NG;
  cplx* tw_z = (NY == NZ) ? tw_y : tw_y + NY;     // equal lengths share one twiddle table
  cplx* stile = tw_z + NZ;
  const int tid = threadIdx.x;
  const int lx = bx / ZS, h = bx % ZS;
  const int s0 = a.plane_s0[lx], S = a.plane_s0[lx + 1] - s0;
  const int y0 = a.plane_y0[lx];
  const cplx* psi = a.psi + (size_t)b * a.npw;
  // H1 + H2 (z) pass 1: psi -> registers -> DFT-R1z -> twiddle -> stick tile (type A, inverse)
  KS_PH_INIT();
  {
    // walk over the (stick, line) items of the pass that touches psi: lines-first (StickWalk) or j-fastest (JWalk, the
    // lanes of a stick read consecutive plane waves).  Measured: 128 x 128 lines-first 0.592 / j-fastest 0.599 ms, 96 x 96
    // 0.272 / 0.276 ms -- but on the z'-split 96 x 288 planes, where the (stick, line) items of a plane are dealt over the
    // three CTAs of a cluster, j-fastest took the forward kernel from 33 to 42 % of HBM.  So: j-fastest iff ZS > 1.
    constexpr bool JFAST = (ZS > 1);
    typename std::conditional<JFAST, JWalk<R2z>, StickWalk>::type w = make_walk<JFAST, R2z>(tid, NT, S);
#define KS_W_OK(w_) (JFAST ? ((w_).s < S) : ((w_).j < R2z))
    // (Staging the plane's run of psi in the idle y tile by cp.async, as the forward kernel does, was measured here too:
    // 128 x 128 0.564 -> 0.570 ms, 96 x 96 0.266 -> 0.279 ms -- the opening phase is not bound by the scattered loads.)
    const cplx* pbase = psi;
    cplx v[R1z];
    auto load_in = [&]() {
      const int4 si = __ldg(a.stick + s0 + w.s);
      const cplx* src = pbase + si.x;
#pragma unroll
      for (int j1 = 0; j1 < R1z; ++j1) {
        int idx = j1 * R2z + w.j - si.y;
        if (idx < 0) idx += NZ;
        v[j1] = (idx < si.z) ? src[idx] : cmake(0.0, 0.0);
      }
    };
    if (KS_W_OK(w)) load_in();
    for (int i = tid; i < NY; i += NT) tw_y[i] = a.tw_y[i];
    if (NY != NZ)
      for (int i = tid; i < NZ; i += NT) tw_z[i] = a.tw_z[i];
    __syncthreads();
    while (KS_W_OK(w)) {
      dft<R1z, +1>(v);
      cplx* o = stile + w.s * SZ + w.j;
      const int j2 = w.j;
#pragma unroll
      for (int k1 = 0; k1 < R1z; ++k1) {
        if constexpr (ZS == 1) {
          o[k1 * R2z] = (k1 == 0) ? v[0] : mul_tw<+1>(v[k1], tw_z, j2 * k1);
        } else {
          if (k1 / K1H == h) o[(k1 % K1H) * R2z] = (k1 == 0) ? v[0] : mul_tw<+1>(v[k1], tw_z, j2 * k1);
        }
      }
      w.next();
      if (KS_W_OK(w)) load_in();
    }
  }
  __syncthreads();
  KS_PH(0);
  for (StickWalk w(tid, NT, S); w.j < K1H; w.next()) lineA_stage2<NZ, +1, facz<NZ>>(stile + w.s * SZ, 1, w.j);
  __syncthreads();
  KS_PH(1);
#ifndef KSPW_NO_PSI_PREFETCH
  // A CTA opens with a chain of dependent global loads that ends in the scattered reads of its plane's run of psi -- cold
  // DRAM reads queued behind the plane stores of the CTAs before it (clock64: 7.1 k of a 128 x 128 plane's 25.3 k clocks pass
  // before the first z pass is over, ~2 k of them arithmetic), with nothing else resident on the SM.  So every CTA asks L2
  // for the psi run of the CTA `pf_dist` places ahead in launch order (about one wave: it starts when this one ends,
  // on whichever SM) -- one prefetch per 128-byte line, one instruction per thread.
  {
    // (z'-split planes: the ZS CTAs of a plane read the same run; the first of them asks for the plane pf_dist CTAs ahead.
    //  Measured: 128 x 128 k_inv_yz 2.86 -> 2.71 ms per 520 bands at one wave (148), no gain at two; 96 x 288 1.00 -> 0.97 ms;
    //  96 x 96, two CTAs per SM: no change.)
    if (a.pf_dist > 0 && h == 0) {
      const long j = (long)b * gridDim.x + bx + a.pf_dist;
      const int lx2 = (int)(j % gridDim.x) / ZS;
      const long b2 = j / gridDim.x;
      if (b2 < a.nb) {
        const int p0 = a.plane_pw0[lx2], np2 = a.plane_pw0[lx2 + 1] - p0;
        const char* q = reinterpret_cast<const char*>(a.psi + (size_t)b2 * a.npw + p0);
        const char* q0 = reinterpret_cast<const char*>(reinterpret_cast<size_t>(q) & ~(size_t)127);
        const long bytes = (q + (size_t)np2 * sizeof(cplx)) - q0;
        for (long o = (long)tid * 128; o < bytes; o += (long)NT * 128) asm volatile("prefetch.global.L2 [%0];" ::"l"(q0 + o));
      }
    }
  }
#endif
  // H2 (y): for each chunk of z' positions, type-A inverse FFT along y; output straight to HBM
  cplx* plane = a.planes + ((size_t)b * a.L1 + lx) * ((size_t)NY * NZ) + h * NZH;
  const int grp = tid / GT, gt = tid % GT;
  const int pz = gt % ZC, g = gt / ZC;
  ytile += grp * (NY * ZC);
  if constexpr (USE_TMA) {
    static_assert(G >= R2y && G >= R1y, "TMA variant: at most one codelet line per thread and pass");
    static_assert(ZS == 1, "TMA variant: whole planes");
    for (int c = grp; c < NZH / ZC; c += NG) {
      // pass 1 in registers (reads the stick tile only)
      cplx v[R1y];
      const bool p1 = g < R2y;
      if (p1) {
        const cplx* src = stile + c * ZC + pz;
#pragma unroll
        for (int j1 = 0; j1 < R1y; ++j1) {
          int s = j1 * R2y + g - y0;
          if (s < 0) s += NY;
          v[j1] = (s < S) ? src[s * SZ] : cmake(0.0, 0.0);
        }
        dft<R1y, +1>(v);
#pragma unroll
        for (int k1 = 1; k1 < R1y; ++k1) v[k1] = mul_tw<+1>(v[k1], tw_y, g * k1);
      }
      // the bulk copies of the group's previous chunk have read the y tile (they drained during pass 1)
      if (gt == 0) bulk_wait_read();
      ygroup_sync<NG, GT>(grp);
      if (p1) {
        cplx* o = ytile + g * ZC + pz;
#pragma unroll
        for (int k1 = 0; k1 < R1y; ++k1) o[k1 * R2y * ZC] = v[k1];
      }
      ygroup_sync<NG, GT>(grp);
      KS_PH(2);
      if (g < R1y) {            // pass 2 in place: thread (g, pz) owns rows g*R2y .. g*R2y + R2y - 1 of column pz
        cplx u[R2y];
        cplx* t = ytile + g * R2y * ZC + pz;
#pragma unroll
        for (int j2 = 0; j2 < R2y; ++j2) u[j2] = t[j2 * ZC];
        dft<R2y, +1>(u);
#pragma unroll
        for (int k2 = 0; k2 < R2y; ++k2) t[k2 * ZC] = u[k2];
      }
      fence_proxy_async();
      ygroup_sync<NG, GT>(grp);
      // plane row r = k1*R2y + k2 is y-tile row r: the whole [NY][ZC] tile leaves as ONE tensor store (box = 2 ZC doubles x NY rows)
      if (gt == 0) {
        tensor_store_2d(tmap, ytile, 2 * (c * ZC), (b * a.L1 + lx) * NY);
        bulk_commit();
      }
      KS_PH(3);
    }
    if (gt == 0) bulk_wait_all();
    return;
  }
  for (int c = grp; c < NZH / ZC; c += NG) {
    if constexpr (YHALF) {
      // twice as many line groups as DFT-R1y lines: two groups share a line, one takes the even outputs (DFT-R1y/2 of
      // x[n] + x[n + R1y/2]), the other the odd ones (DFT-R1y/2 of (x[n] - x[n + R1y/2]) w^n): every warp works in this pass
      constexpr int H = R1y / 2;
      const int j2 = g % R2y, half = g / R2y;
      cplx v[R1y];
      const cplx* src = stile + c * ZC + pz;
#pragma unroll
      for (int j1 = 0; j1 < R1y; ++j1) {
        int s = j1 * R2y + j2 - y0;
        if (s < 0) s += NY;
        v[j1] = (s < S) ? src[s * SZ] : cmake(0.0, 0.0);
      }
      cplx u[H];
      if (half == 0) {
#pragma unroll
        for (int n = 0; n < H; ++n) u[n] = cmake(v[n].x + v[n + H].x, v[n].y + v[n + H].y);
      } else {
#pragma unroll
        for (int n = 0; n < H; ++n) {
          const cplx d = cmake(v[n].x - v[n + H].x, v[n].y - v[n + H].y);
          u[n] = (n == 0) ? d : mul_tw<+1>(d, tw_y, n * (NY / R1y));
        }
      }
      dft<H, +1>(u);
      cplx* o = ytile + j2 * ZC + pz + half * (R2y * ZC);
#pragma unroll
      for (int kh = 0; kh < H; ++kh)      // k1 = 2 kh + half
        o[2 * kh * R2y * ZC] = (kh == 0 && half == 0) ? u[0] : mul_tw<+1>(u[kh], tw_y, j2 * (2 * kh + half));
    } else if (g < G) {
      for (int j2 = g; j2 < R2y; j2 += G) {
        cplx v[R1y];
        const cplx* src = stile + c * ZC + pz;
#pragma unroll
        for (int j1 = 0; j1 < R1y; ++j1) {
          int s = j1 * R2y + j2 - y0;
          if (s < 0) s += NY;
          v[j1] = (s < S) ? src[s * SZ] : cmake(0.0, 0.0);
        }
        dft<R1y, +1>(v);
        cplx* o = ytile + j2 * ZC + pz;
#pragma unroll
        for (int k1 = 0; k1 < R1y; ++k1) o[k1 * R2y * ZC] = (k1 == 0) ? v[0] : mul_tw<+1>(v[k1], tw_y, j2 * k1);
      }
    }
    ygroup_sync<NG, GT>(grp);
    KS_PH(2);
    if (g < G) {
      for (int k1 = g; k1 < R1y; k1 += G) {
        cplx v[R2y];
        const cplx* t = ytile + k1 * R2y * ZC + pz;
#pragma unroll
        for (int j2 = 0; j2 < R2y; ++j2) v[j2] = t[j2 * ZC];
        dft<R2y, +1>(v);
        cplx* o = plane + (size_t)(k1 * R2y) * NZ + c * ZC + pz;
#pragma unroll
        for (int k2 = 0; k2 < R2y; ++k2) KS_ST_PLANE(o + k2 * NZ, v[k2]);
      }
    }
    ygroup_sync<NG, GT>(grp);
    KS_PH(3);
  }
}

template <int NY, int NZ>
__global__ void __launch_bounds__(yzcfg<NY, NZ>::NT, yzcfg<NY, NZ>::NT <= 256 ? 2 : 1) k_inv_yz(const __grid_constant__ YzArgs a) {
  inv_yz_body<NY, NZ, false>(a, blockIdx.x, blockIdx.y, nullptr);
}
// the same with the planes leaving through the tensor map `tm` of the live-plane workspace (yzcfg::TMA)
template <int NY, int NZ>
__global__ void __launch_bounds__(yzcfg<NY, NZ>::NT, yzcfg<NY, NZ>::NT <= 256 ? 2 : 1) k_inv_yz_tma(const __grid_constant__ YzArgs a,
                                                                                                const __grid_constant__ CUtensorMap tm) {
  inv_yz_body<NY, NZ, yzcfg<NY, NZ>::TMA>(a, blockIdx.x, blockIdx.y, &tm);
}
// k-batched form (ks_hpsi_batch): blockIdx.z picks the k-point's descriptor; the grid is sized for the largest k of the group
template <int NY, int NZ>
__global__ void __launch_bounds__(yzcfg<NY, NZ>::NT, yzcfg<NY, NZ>::NT <= 256 ? 2 : 1) k_inv_yz_k(const YzArgs* __restrict__ arr) {
  __shared__ YzArgs a;
  if (threadIdx.x == 0) a = arr[blockIdx.z];
  __syncthreads();
  if ((int)blockIdx.x >= a.L1 * yzcfg<NY, NZ>::ZS || (int)blockIdx.y >= a.nb) return;
  inv_yz_body<NY, NZ, false>(a, blockIdx.x, blockIdx.y, nullptr);
}

template <int NY, int NZ>
__device__ __forceinline__ void fwd_yz_body(const YzArgs& a, const int bx, const int b) {
  constexpr int R1y = fac<NY>::R1, R2y = fac<NY>::R2, R1z = facz<NZ>::R1, R2z = facz<NZ>::R2;
  constexpr int ZS = yzcfg<NY, NZ>::ZS, NZH = NZ / ZS, K1H = R1z / ZS;   // this CTA's z' positions and codelet lines
  static_assert(ZS == 1 || !yzcfg<NY, NZ>::DBF, "the z' split uses the single-buffer y transform");
  constexpr int SZ = NZH | 1, ZC = yzcfg<NY, NZ>::ZC, NT = yzcfg<NY, NZ>::NT, NG = yzcfg<NY, NZ>::NG, GT = NT / NG, G = GT / ZC;
  static_assert(NG == 1 || !yzcfg<NY, NZ>::DBF, "y groups use the single-buffer y transform");
#ifndef KSPW_NO_YHALF    // measured on cfg 3: k_fwd_yz 0.688 -> 0.665 ms
  constexpr bool YHALF = (G == 2 * R2y) && (R1y % 2 == 0) && (GT == G * ZC) && (ZC * NG == 32);   // 128 x 128: twice as many line groups as DFT-16 lines (on 96 x 288, ZC 16, it measured slower: 0.636 -> 0.688 ms)
#else
  constexpr bool YHALF = false;
#endif
  extern __shared__ __align__(128) cplx sm[];
  cplx* ytile = sm;                               // same layout as the inverse kernel
  cplx* const ytile0 = sm;                        // all groups' y tiles: NY * ZC * NG elements (reused for psi after the y phase)
  cplx* tw_y = ytile + NY * ZC * NG;
  cplx* tw_z = (NY == NZ) ? tw_y : tw_y + NY;     // equal lengths share one twiddle table
  cplx* stile = tw_z + NZ;
  const int tid = threadIdx.x;
  const int lx = bx / ZS, h = bx % ZS;   // h = rank in the cluster of ZS CTAs
  const int s0 = a.plane_s0[lx], S = a.plane_s0[lx + 1] - s0;
  const int y0 = a.plane_y0[lx];
  const cplx* plane = a.planes + ((size_t)b * a.L1 + lx) * ((size_t)NY * NZ) + h * NZH;
  const int grp = tid / GT, gt = tid % GT;
  const int pz = gt % ZC, g = gt / ZC;
  KS_PH_INIT();
#ifndef KSPW_NO_PSI_PREFETCH
  // z'-split planes: the last pass reads psi (for |k+G|^2 psi) straight from global memory, one dependent load per output,
  // long after k_inv_yz brought it in; the ZS CTAs of the plane ask L2 for the plane's run now, a y transform ahead of its use
#ifndef KSPW_FWD_PF_ALL
#define KSPW_FWD_PF_ALL 0     // unsplit planes stage the run by cp.async after the y transform; the same request ahead of it
#endif                        // measured slower: 128 x 128 2.839 -> 2.938 ms, 96 x 96 0.321 -> 0.324 ms
  if constexpr (ZS > 1 || KSPW_FWD_PF_ALL) {
    const int p0 = a.plane_pw0[lx], np2 = a.plane_pw0[lx + 1] - p0;
    const char* q = reinterpret_cast<const char*>(a.psi + (size_t)b * a.npw + p0);
    const char* q0 = reinterpret_cast<const char*>(reinterpret_cast<size_t>(q) & ~(size_t)127);
    const long bytes = (q + (size_t)np2 * sizeof(cplx)) - q0;
    for (long o = ((long)h * NT + tid) * 128; o < bytes; o += (long)ZS * NT * 128) asm volatile("prefetch.global.L2 [%0];" ::"l"(q0 + o));
  }
#endif
  // H4 (y), type B, forward.  The y tile is split into two half-width buffers: while chunk c (ZF = ZC/2 columns) is
  // transformed in place in one of them, chunk c+1 streams into the other by cp.async, so the plane loads are
  // in flight during both codelet passes.  (Odd ZC: single buffer, loads straight into registers.)
  if constexpr (yzcfg<NY, NZ>::DBF) {
    constexpr int ZF = ZC / 2, GF = NT / ZF, NCF = NZ / ZF;
    const int fz = tid % ZF, fg = tid / ZF;
    auto issue = [&](int c) {
      cplx* dst = ytile + (c & 1) * (NY * ZF);
      const cplx* src = plane + c * ZF;
      for (int e = tid; e < NY * ZF; e += NT) cp16m(dst + e, src + (size_t)(e / ZF) * NZ + (e % ZF));
      cp_commit_m();
    };
    issue(0);
    for (int i = tid; i < NY; i += NT) tw_y[i] = a.tw_y[i];
    if (NY != NZ)
      for (int i = tid; i < NZ; i += NT) tw_z[i] = a.tw_z[i];
    for (int c = 0; c < NCF; ++c) {
      cp_wait_n(0);
      __syncthreads();              // chunk c has landed; pass 2 of chunk c-1 is over, its buffer is free
      if (c + 1 < NCF) issue(c + 1);
      cplx* yb = ytile + (c & 1) * (NY * ZF) + fz;
      if (fg < GF) {
        for (int k1 = fg; k1 < R1y; k1 += GF) {
          cplx v[R2y];
          cplx* o = yb + k1 * R2y * ZF;
#pragma unroll
          for (int k2 = 0; k2 < R2y; ++k2) v[k2] = o[k2 * ZF];
          dft<R2y, -1>(v);
#pragma unroll
          for (int q2 = 0; q2 < R2y; ++q2) o[q2 * ZF] = (q2 == 0) ? v[0] : mul_tw<-1>(v[q2], tw_y, k1 * q2);
        }
      }
      __syncthreads();
      if (fg < GF) {
        for (int q2 = fg; q2 < R2y; q2 += GF) {
          cplx u[R1y];
          const cplx* t = yb + q2 * ZF;
#pragma unroll
          for (int k1 = 0; k1 < R1y; ++k1) u[k1] = t[k1 * R2y * ZF];
          dft<R1y, -1>(u);
          cplx* o = stile + c * ZF + fz;
#pragma unroll
          for (int q1 = 0; q1 < R1y; ++q1) {   // natural y = q1*R2y + q2; keep the stick columns only
            int s = q1 * R2y + q2 - y0;
            if (s < 0) s += NY;
            if (s < S) o[s * SZ] = u[q1];
          }
        }
      }
    }
    __syncthreads();
  } else {
  // H4 (y) pass 1 of a chunk: plane -> registers -> DFT-R2y -> twiddle -> ytile (type B, forward)
  auto load_in = [&](cplx (&v)[R2y], int c, int k1) {
    const cplx* src = plane + (size_t)(k1 * R2y) * NZ + c * ZC + pz;
#pragma unroll
    for (int k2 = 0; k2 < R2y; ++k2) v[k2] = KS_LD_PLANE(src + k2 * NZ);
  };
  {
    cplx v[R2y];
    ytile += grp * (NY * ZC);
    if (g < G && g < R1y) load_in(v, grp, g);
    for (int i = tid; i < NY; i += NT) tw_y[i] = a.tw_y[i];
    if (NY != NZ)
      for (int i = tid; i < NZ; i += NT) tw_z[i] = a.tw_z[i];
    __syncthreads();
    for (int c = grp; c < NZH / ZC; c += NG) {
      if (g < G) {
        for (int k1 = g; k1 < R1y; k1 += G) {
          if (k1 != g) load_in(v, c, k1);          // the thread's first line of a chunk is already in registers
          dft<R2y, -1>(v);
          cplx* o = ytile + k1 * R2y * ZC + pz;
#pragma unroll
          for (int q2 = 0; q2 < R2y; ++q2) o[q2 * ZC] = (q2 == 0) ? v[0] : mul_tw<-1>(v[q2], tw_y, k1 * q2);
        }
      }
      ygroup_sync<NG, GT>(grp);
      KS_PH(8);
      if (g < G && g < R1y && c + NG < NZH / ZC) load_in(v, c + NG, g);   // next chunk's loads fly during pass 2
      if constexpr (YHALF) {
        // two line groups per DFT-R1y line: even outputs from one, odd outputs from the other (see k_inv_yz)
        constexpr int H = R1y / 2;
        const int q2 = g % R2y, half = g / R2y;
        cplx u[R1y];
        const cplx* t = ytile + q2 * ZC + pz;
#pragma unroll
        for (int k1 = 0; k1 < R1y; ++k1) u[k1] = t[k1 * R2y * ZC];
        cplx w[H];
        if (half == 0) {
#pragma unroll
          for (int n = 0; n < H; ++n) w[n] = cmake(u[n].x + u[n + H].x, u[n].y + u[n + H].y);
        } else {
#pragma unroll
          for (int n = 0; n < H; ++n) {
            const cplx d = cmake(u[n].x - u[n + H].x, u[n].y - u[n + H].y);
            w[n] = (n == 0) ? d : mul_tw<-1>(d, tw_y, n * (NY / R1y));
          }
        }
        dft<H, -1>(w);
        cplx* o = stile + c * ZC + pz;
#pragma unroll
        for (int qh = 0; qh < H; ++qh) {     // q1 = 2 qh + half; natural y = q1*R2y + q2; keep the stick columns only
          int s = (2 * qh + half) * R2y + q2 - y0;
          if (s < 0) s += NY;
          if (s < S) o[s * SZ] = w[qh];
        }
      } else if (g < G) {
        for (int q2 = g; q2 < R2y; q2 += G) {
          cplx u[R1y];
          const cplx* t = ytile + q2 * ZC + pz;
#pragma unroll
          for (int k1 = 0; k1 < R1y; ++k1) u[k1] = t[k1 * R2y * ZC];
          dft<R1y, -1>(u);
          cplx* o = stile + c * ZC + pz;
#pragma unroll
          for (int q1 = 0; q1 < R1y; ++q1) {   // natural y = q1*R2y + q2; keep the stick columns only
            int s = q1 * R2y + q2 - y0;
            if (s < 0) s += NY;
            if (s < S) o[s * SZ] = u[q1];
          }
        }
      }
      ygroup_sync<NG, GT>(grp);
      KS_PH(9);
    }
    if constexpr (NG > 1) __syncthreads();      // every group's stick columns are in place before the z transform
    KS_PH(10);
  }
  }
#ifndef KSPW_NO_PLANE_PREFETCH
  // the same idea as in k_inv_yz: a CTA opens by waiting for the first chunk of its plane (cold DRAM reads, nothing else
  // resident on the SM), so every CTA asks L2 for the first chunk of every y group of the plane `pf_dist` CTAs ahead
  if constexpr (ZS == 1 && !yzcfg<NY, NZ>::DBF) {
    if (a.pf_dist > 0) {
      const long j = (long)b * gridDim.x + bx + a.pf_dist;
      const int lx2 = (int)(j % gridDim.x);
      const long b2 = j / gridDim.x;
      if (b2 < a.nb) {
        constexpr int LPR = (NG * ZC * (int)sizeof(cplx) + 127) / 128;      // 128-byte lines per plane row
        const char* q = reinterpret_cast<const char*>(a.planes + ((size_t)b2 * a.L1 + lx2) * ((size_t)NY * NZ));
        for (int i = tid; i < NY * LPR; i += NT)
          asm volatile("prefetch.global.L2 [%0];" ::"l"(q + (size_t)(i / LPR) * NZ * sizeof(cplx) + (size_t)(i % LPR) * 128));
      }
    }
  }
#endif
  // H4 (z): type-B forward FFT on each stick
  const cplx* psi = a.psi + (size_t)b * a.npw;
  cplx* hpsi = a.hpsi + (size_t)b * a.npw;
  if constexpr (ZS == 1) {
    // The plane waves of one x-plane are ONE contiguous run of psi (its sticks follow each other in the canonical order):
    // the run streams into the now idle y tile by cp.async while the first z pass runs, so the last pass finds psi in
    // shared memory instead of paying a dependent global load per output (clock64: 9.5k of 28.9k clocks per 128 x 128 plane
    // went to this pass).  Planes whose run does not fit the y tile read psi from global memory as before.
    const int pw0 = a.plane_pw0[lx], npl = a.plane_pw0[lx + 1] - pw0;
#ifdef KSPW_FWD_PSI_GLOBAL
    const bool staged = false;
#else
    const bool staged = npl <= NY * ZC * NG;
#endif
    if (staged) {
      for (int i = tid; i < npl; i += NT) cp16m(ytile0 + i, psi + pw0 + i);
      cp_commit_m();
    }
    for (StickWalk w(tid, NT, S); w.j < R1z; w.next()) lineB_stage1<NZ, -1, facz<NZ>>(stile + w.s * SZ, 1, w.j, tw_z);
    if (staged) cp_wait_n(0);
    __syncthreads();
    KS_PH(11);
    // last pass + H5: DFT-R1z, then hpsi = |k+G|^2 psi + (.)/N written straight to the stick's run of hpsi
    const cplx* psrc = staged ? (ytile0 - pw0) : psi;          // psrc[j] = psi[j] for the plane's run
    for (StickWalk w(tid, NT, S); w.j < R2z; w.next()) {
      const int4 si = __ldg(a.stick + s0 + w.s);
      // |k+G|^2 of the line's outputs first: the loads fly during the codelet
      double kk[R1z];
#pragma unroll
      for (int q1 = 0; q1 < R1z; ++q1) {
        int idx = q1 * R2z + w.j - si.y;
        if (idx < 0) idx += NZ;
        kk[q1] = (idx < si.z) ? __ldg(a.g2 + si.x + idx) : 0.0;
      }
      cplx v[R1z];
      const cplx* t = stile + w.s * SZ + w.j;
#pragma unroll
      for (int k1 = 0; k1 < R1z; ++k1) v[k1] = t[k1 * R2z];
      dft<R1z, -1>(v);
#pragma unroll
      for (int q1 = 0; q1 < R1z; ++q1) {       // natural z = q1*R2z + q2
        int idx = q1 * R2z + w.j - si.y;
        if (idx < 0) idx += NZ;
        if (idx < si.z) {
          const int j = si.x + idx;
          const cplx p = psrc[j];
          hpsi[j] = cmake(fma(kk[q1], p.x, v[q1].x * a.invN), fma(kk[q1], p.y, v[q1].y * a.invN));
        }
      }
    }
    KS_PH(12);
  } else {
    // first z pass on this CTA's lines k1 = h*K1H + k1l (local offset k1l, twiddle index from the global k1)
    for (StickWalk w(tid, NT, S); w.j < K1H; w.next()) {
      cplx* line = stile + w.s * SZ + w.j * R2z;
      const int k1 = h * K1H + w.j;
      cplx v[R2z];
#pragma unroll
      for (int k2 = 0; k2 < R2z; ++k2) v[k2] = line[k2];
      dft<R2z, -1>(v);
#pragma unroll
      for (int q2 = 0; q2 < R2z; ++q2) line[q2] = (q2 == 0) ? v[0] : mul_tw<-1>(v[q2], tw_z, k1 * q2);
    }
    cg::cluster_group cl = cg::this_cluster();
    cl.sync();                                   // every CTA of the plane has finished its part of the sticks
    const cplx* peer[ZS];
#pragma unroll
    for (int r = 0; r < ZS; ++r) peer[r] = (const cplx*)cl.map_shared_rank((void*)stile, r);
    // last pass + H5: the (stick, q2) items of the plane are dealt over the ZS CTAs; line k1 lives in CTA k1 / K1H
    for (JWalk<R2z> w(h * NT + tid, ZS * NT); w.s < S; w.next()) {   // j-fastest: see k_inv_yz
      const int4 si = __ldg(a.stick + s0 + w.s);
      cplx v[R1z];
      const int off = w.s * SZ + w.j;
#pragma unroll
      for (int k1 = 0; k1 < R1z; ++k1) v[k1] = peer[k1 / K1H][off + (k1 % K1H) * R2z];
      dft<R1z, -1>(v);
#pragma unroll
      for (int q1 = 0; q1 < R1z; ++q1) {       // natural z = q1*R2z + q2
        int idx = q1 * R2z + w.j - si.y;
        if (idx < 0) idx += NZ;
        if (idx < si.z) {
          const int j = si.x + idx;
          const cplx p = psi[j];
          const double k = __ldg(a.g2 + j);
          hpsi[j] = cmake(fma(k, p.x, v[q1].x * a.invN), fma(k, p.y, v[q1].y * a.invN));
        }
      }
    }
    cl.sync();                                   // no CTA leaves while its stick tile is still being read
  }
}

template <int NY, int NZ>
__global__ void __launch_bounds__(yzcfg<NY, NZ>::NT, yzcfg<NY, NZ>::NT <= 256 ? 2 : 1) k_fwd_yz(const __grid_constant__ YzArgs a) {
  fwd_yz_body<NY, NZ>(a, blockIdx.x, blockIdx.y);
}
template <int NY, int NZ>
__global__ void __launch_bounds__(yzcfg<NY, NZ>::NT, yzcfg<NY, NZ>::NT <= 256 ? 2 : 1) k_fwd_yz_k(const YzArgs* __restrict__ arr) {
  __shared__ YzArgs a;
  if (threadIdx.x == 0) a = arr[blockIdx.z];
  __syncthreads();
  // whole clusters leave together: lx = blockIdx.x / ZS is the same for the ZS CTAs of a cluster
  if ((int)blockIdx.x >= a.L1 * yzcfg<NY, NZ>::ZS || (int)blockIdx.y >= a.nb) return;
  fwd_yz_body<NY, NZ>(a, blockIdx.x, blockIdx.y);
}

// ------------------------------------------------------------------------------------------------
// x pass: inverse FFT, V(r) multiply, forward FFT in one kernel
// ------------------------------------------------------------------------------------------------
// A CTA owns ZC consecutive (y',z') columns of one band and all NX x-positions.  The first codelet
// pass reads the live planes straight from global memory into registers (rows that are not live are
// zeros and never touched), the last one writes the live planes back from registers, so the tile
// crosses shared memory only between the passes (two barriers per tile).  Thread t works on column
// t % ZC and on the codelet lines t / ZC, t / ZC + G, ... (G = NT / ZC); every shared-memory offset is
// a compile-time multiple of ZC plus one per-thread base.
struct XArgs {
  cplx* planes;         // [nb][L1][NY*NZ], in place
  const double* vperm;  // [NX][NY*NZ]
  const cplx* tw_x;
  int L1, x0, nb, bg;   // nb bands in the batch, bg bands per CTA (gridDim.y = ceil(nb / bg))
  long ncol;            // NY*NZ
};

// STAGE: the next band's live rows stream into a staging buffer [L1][ZC] instead of the tile rows (see x_body)
template <int NX> struct xcfg { static constexpr int ZC = 32, NT = 128, MINB = 4; static constexpr bool STAGE = false; };
template <> struct xcfg<18> { static constexpr int ZC = 32, NT = 96, MINB = 4; static constexpr bool STAGE = false; };
template <> struct xcfg<36> { static constexpr int ZC = 32, NT = 96, MINB = 4; static constexpr bool STAGE = false; };
template <> struct xcfg<54> { static constexpr int ZC = 32, NT = 96, MINB = 4; static constexpr bool STAGE = false; };
// 128: 16-column tiles and 4-warp CTAs (five per SM) beat 32-column tiles and two 8-warp CTAs (301 -> 283 us per 30-band launch);
// the same halving for 96 (64-thread CTAs, eight per SM) is slightly slower (283 -> 289 us)
#ifndef KSPW_X128_STAGE
#define KSPW_X128_STAGE 0   // measured (cfg 3, 520 bands): refill of the tile rows after pass 3 4.41 ms, staging buffer 4.70 ms: off
#endif
#ifndef KSPW_X128_MINB
#define KSPW_X128_MINB 5    // CTAs per SM asked of ptxas: 4 -> 128 registers, 5 -> 96 (12 bytes of spills), 6 -> 80 (148 bytes).
#endif                      // Measured (cfg 3, 520 bands): 4.424 / 4.348 / 4.992 ms
#ifndef KSPW_X_VPRE
#define KSPW_X_VPRE 0
#endif
template <> struct xcfg<128> { static constexpr int ZC = 16, NT = 128, MINB = KSPW_X128_MINB; static constexpr bool STAGE = (KSPW_X128_STAGE != 0); };

// The CTA walks over bg bands with the same columns.  Thread (pz, g) owns the codelet lines j2 = g, g+G, ...
// in the first AND the last pass, i.e. the tile rows {j1*R2 + j2}: once the last pass of band b has read a
// line into registers, the same thread refills the live rows of that line with band b+1 by cp.async, and the
// first pass of band b+1 picks them up with no barrier in between (only its own cp.async group to wait for).
// The global-load latency of a band is hidden behind the last pass of the band before it.
template <int NX>
__device__ __forceinline__ void x_body(const XArgs& a, const int bx, const int by) {
  constexpr int R1 = fac<NX>::R1, R2 = fac<NX>::R2;
  constexpr int ZC = xcfg<NX>::ZC, NT = xcfg<NX>::NT, G = NT / ZC;
  constexpr int ITEMS = (R2 + G - 1) / G;     // first/last-pass lines per thread
  constexpr int R1P = (R1 + 3) & ~3;          // row-offset table: R2+1 lines of R1P entries (line R2 is all dead)
  constexpr unsigned DEAD = 0xffffffffu;
  // STG: the live rows of the NEXT band stream into a staging buffer [L1][ZC] right after pass 1 has taken the current
  // band's rows out of it, so a band's global loads have all three passes of the band before it to land.  (Refilling the tile
  // rows themselves is only possible after pass 3 has read them, i.e. a few store instructions before pass 1 of the next band
  // wants them: ncu attributed 15 % of k_x<128>'s stall samples to that first shared-memory read, waiting on the cp.async.)
  constexpr bool STG = xcfg<NX>::STAGE;
  static_assert(NT % ZC == 0, "thread count must be a multiple of the column chunk");
  static_assert(ITEMS <= 4, "cp_wait_n covers up to 4 groups in flight");
  extern __shared__ cplx sm[];
  cplx* tw = sm;
  cplx* tile = sm + NX;
  unsigned* rofs = reinterpret_cast<unsigned*>(tile + NX * ZC);   // [R2+1][R1P]: element offset of row j1*R2+j2 (STG: its live-plane index), or DEAD
  cplx* stage = reinterpret_cast<cplx*>(rofs + (R2 + 1) * R1P);    // STG only: [L1][ZC]  (the table is a multiple of 16 bytes)
  const int tid = threadIdx.x, pz = tid % ZC, g = tid / ZC;
  const unsigned ncol = (unsigned)a.ncol;      // one band's live planes (L1*ncol elements) fit 32-bit offsets
  const unsigned col = bx * ZC + pz;
  const bool colok = col < ncol;              // ragged last chunk: such threads use the all-dead table line
  const int b0 = by * a.bg, b1 = min(b0 + a.bg, a.nb);
  const size_t bstride = (size_t)a.L1 * a.ncol;
  cplx* base = a.planes + (size_t)b0 * bstride + (colok ? col : 0);
  const double* vbase = a.vperm + (colok ? col : 0);
  cplx* tcol = tile + pz;

  for (int i = tid; i < (R2 + 1) * R1P; i += NT) {
    const int j2 = i / R1P, j1 = i % R1P;
    unsigned o = DEAD;
    if (j2 < R2 && j1 < R1) {
      int lx = j1 * R2 + j2 - a.x0;
      if (lx < 0) lx += NX;
      if (lx < a.L1) o = STG ? (unsigned)lx : (unsigned)lx * ncol;
    }
    rofs[i] = o;
  }
  for (int i = tid; i < NX; i += NT) tw[i] = a.tw_x[i];
  __syncthreads();

  // row offsets of line j2 (warp-uniform address: broadcast loads)
  auto line_offsets = [&](unsigned (&o)[R1P], int j2) {
    const uint4* t = reinterpret_cast<const uint4*>(rofs + ((colok && j2 < R2) ? j2 : R2) * R1P);
#pragma unroll
    for (int q = 0; q < R1P / 4; ++q) {
      const uint4 u = t[q];
      o[4 * q] = u.x; o[4 * q + 1] = u.y; o[4 * q + 2] = u.z; o[4 * q + 3] = u.w;
    }
  };
  // refill the live rows of line j2 from band `src` (one cp.async group per line, committed by every thread)
  auto prefetch_line = [&](const cplx* src, int j2) {
    unsigned o[R1P];
    line_offsets(o, j2);
#pragma unroll
    for (int j1 = 0; j1 < R1; ++j1)
      if (o[j1] != DEAD) {
        if constexpr (STG) cp16m(stage + o[j1] * ZC + pz, src + o[j1] * ncol);
        else cp16m(tcol + (j1 * R2 + j2) * ZC, src + o[j1]);
      }
    cp_commit_m();
  };
#pragma unroll
  for (int i = 0; i < ITEMS; ++i) prefetch_line(base, g + i * G);

  // (An L2 prefetch of the first band of the CTA one wave ahead -- what k_inv_yz / k_fwd_yz do for their opening loads -- was
  // measured here too: 128: 4.344 -> 4.414 ms, 96: 0.573 -> 0.601 ms, and 4.382 / 0.598 ms with the distance set to 0: the extra
  // live registers cost more than the cold first band.)
  for (int b = b0; b < b1; ++b, base += bstride) {
    const bool more = b + 1 < b1;
    // pass 1 (type-A stage 1): own prefetched rows -> registers -> DFT-R1 -> twiddle -> tile
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
      const int j2 = g + i * G;
      // STG: every line's turn leaves ITEMS - 1 younger groups in flight (the refills issued below included)
      cp_wait_n(STG ? ITEMS - 1 : ITEMS - 1 - i);
      if (R2 % G == 0 || j2 < R2) {
        unsigned o[R1P];
        line_offsets(o, j2);
        cplx v[R1];
#pragma unroll
        for (int j1 = 0; j1 < R1; ++j1) {
          if constexpr (STG) v[j1] = (o[j1] != DEAD) ? stage[o[j1] * ZC + pz] : cmake(0.0, 0.0);
          else v[j1] = (o[j1] != DEAD) ? tcol[(j1 * R2 + j2) * ZC] : cmake(0.0, 0.0);
        }
        dft<R1, +1>(v);
        if constexpr (STG) {                 // v is consumed: the line's staging rows are free for the next band
          if (more) {
#pragma unroll
            for (int j1 = 0; j1 < R1; ++j1)
              if (o[j1] != DEAD) cp16m(stage + o[j1] * ZC + pz, base + bstride + o[j1] * ncol);
          }
        }
        cplx* out = tcol + j2 * ZC;
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) out[k1 * R2 * ZC] = (k1 == 0) ? v[0] : mul_tw<+1>(v[k1], tw, j2 * k1);
      }
      if constexpr (STG) cp_commit_m();      // one group per line and band, empty or not: uniform accounting
    }
#if KSPW_X_VPRE
    // V(r) of the thread's first pass-2 line is requested BEFORE the barrier and each later line's one line ahead, so the
    // (mostly L2) latency of these loads runs under the barrier wait and the previous line's codelets (ncu: 6 % of
    // k_x<128>'s stall samples sat on the first use of vr)
    double vr[R2];
    if (g < R1) {
      const double* vp = vbase + (size_t)g * R2 * a.ncol;
#pragma unroll
      for (int k2 = 0; k2 < R2; ++k2) vr[k2] = __ldg(vp + (unsigned)k2 * ncol);
    }
    __syncthreads();
    // pass 2: type-A stage 2, V(r), type-B stage 1 on the same R2 elements, in registers
    for (int k1 = g; k1 < R1; k1 += G) {
      cplx v[R2];
      cplx* t = tcol + k1 * R2 * ZC;
#pragma unroll
      for (int j2 = 0; j2 < R2; ++j2) v[j2] = t[j2 * ZC];
      dft<R2, +1>(v);
#pragma unroll
      for (int k2 = 0; k2 < R2; ++k2) v[k2] = cmake(v[k2].x * vr[k2], v[k2].y * vr[k2]);
      if (k1 + G < R1) {
        const double* vp = vbase + (size_t)(k1 + G) * R2 * a.ncol;
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) vr[k2] = __ldg(vp + (unsigned)k2 * ncol);
      }
      dft<R2, -1>(v);
#pragma unroll
      for (int q2 = 0; q2 < R2; ++q2) t[q2 * ZC] = (q2 == 0) ? v[0] : mul_tw<-1>(v[q2], tw, k1 * q2);
    }
    __syncthreads();
#else
    __syncthreads();
    // pass 2: type-A stage 2, V(r), type-B stage 1 on the same R2 elements, in registers
    for (int k1 = g; k1 < R1; k1 += G) {
      double vr[R2];
      const double* vp = vbase + (size_t)k1 * R2 * a.ncol;
#pragma unroll
      for (int k2 = 0; k2 < R2; ++k2) vr[k2] = __ldg(vp + (unsigned)k2 * ncol);
      cplx v[R2];
      cplx* t = tcol + k1 * R2 * ZC;
#pragma unroll
      for (int j2 = 0; j2 < R2; ++j2) v[j2] = t[j2 * ZC];
      dft<R2, +1>(v);
#pragma unroll
      for (int k2 = 0; k2 < R2; ++k2) v[k2] = cmake(v[k2].x * vr[k2], v[k2].y * vr[k2]);
      dft<R2, -1>(v);
#pragma unroll
      for (int q2 = 0; q2 < R2; ++q2) t[q2 * ZC] = (q2 == 0) ? v[0] : mul_tw<-1>(v[q2], tw, k1 * q2);
    }
    __syncthreads();
#endif
    // pass 3 (type-B stage 2): tile -> DFT-R1 -> live planes (natural x = q1*R2 + q2); refill the line (tile-row variant)
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
      const int q2 = g + i * G;
      unsigned o[R1P];
      line_offsets(o, q2);
      cplx v[R1];
      if (R2 % G == 0 || q2 < R2) {
        const cplx* t = tcol + q2 * ZC;
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) v[k1] = t[k1 * R2 * ZC];
        dft<R1, -1>(v);
      }
      if constexpr (!STG) {
        if (more) {                                    // v is consumed: the line's rows are free
#pragma unroll
          for (int j1 = 0; j1 < R1; ++j1)
            if (o[j1] != DEAD) cp16m(tcol + (j1 * R2 + q2) * ZC, base + bstride + o[j1]);
          cp_commit_m();
        }
      }
#pragma unroll
      for (int q1 = 0; q1 < R1; ++q1)
        if (o[q1] != DEAD) base[STG ? o[q1] * ncol : o[q1]] = v[q1];
    }
    // no barrier here: pass 1 of the next band writes the tile rows {k1*R2 + j2} that this same thread read in pass 3
  }
}

template <int NX>
__global__ void __launch_bounds__(xcfg<NX>::NT, xcfg<NX>::MINB) k_x(const __grid_constant__ XArgs a) {
  x_body<NX>(a, blockIdx.x, blockIdx.y);
}
template <int NX>
__global__ void __launch_bounds__(xcfg<NX>::NT, xcfg<NX>::MINB) k_x_k(const XArgs* __restrict__ arr) {
  __shared__ XArgs a;
  if (threadIdx.x == 0) a = arr[blockIdx.z];
  __syncthreads();
  if ((int)blockIdx.y * a.bg >= a.nb) return;
  x_body<NX>(a, blockIdx.x, blockIdx.y);
}

// ------------------------------------------------------------------------------------------------
// density build: rho(r) += occ_b |psi_b(r)|^2 from the live planes k_inv_yz wrote
// ------------------------------------------------------------------------------------------------
// The first half of k_x: pass 1 (DFT-R1 on the live rows) and the inverse half of pass 2 (DFT-R2); instead of
// V(r) and the way back, |psi(r)|^2 is accumulated in registers over the bands the CTA walks through.  A CTA owns
// 32 columns and one of `ng` band groups and is the only writer of its slice part[group][x'][column], so the sum
// over bands has a fixed order (no atomics); k_rho_finish adds the groups in order and undoes the position order.
// The next band's live rows stream into a staging buffer by cp.async while the current band is transformed.
struct RhoArgs {
  const cplx* planes;   // [nb][L1][NY*NZ]
  const double* occ;    // [nb] occupations of this batch
  double* part;         // [ng][NX][NY*NZ] partial densities, x in position order
  const cplx* tw_x;
  int L1, x0, nb, ng, accumulate;
  long ncol;
};

// tile geometry of k_rho: it has one staging buffer and waits for it once per band, so it wants more (smaller) CTAs per SM
// than k_x: 16 columns x 64 threads, five CTAs per SM for 96 (cfg 1 density 217k -> 238k bands/s); k_x's geometry otherwise
template <int NX> struct rcfg { static constexpr int ZC = xcfg<NX>::ZC, NT = xcfg<NX>::NT, MINB = xcfg<NX>::MINB > 3 ? 3 : xcfg<NX>::MINB; };
template <> struct rcfg<96> { static constexpr int ZC = 16, NT = 64, MINB = 5; };

template <int NX>
__global__ void __launch_bounds__(rcfg<NX>::NT, rcfg<NX>::MINB) k_rho(RhoArgs a) {
  constexpr int R1 = fac<NX>::R1, R2 = fac<NX>::R2;
  constexpr int ZC = rcfg<NX>::ZC, NT = rcfg<NX>::NT, G = NT / ZC;
  constexpr int IT2 = (R1 + G - 1) / G;       // pass-2 lines per thread
  constexpr int R1P = (R1 + 3) & ~3;
  extern __shared__ cplx sm[];
  cplx* tw = sm;
  cplx* tile = sm + NX;
  int* rlx = reinterpret_cast<int*>(tile + NX * ZC);            // [R2+1][R1P]: live-plane index of row j1*R2+j2, or -1
  cplx* stage = reinterpret_cast<cplx*>(rlx + (R2 + 1) * R1P);   // [L1][ZC]  ((R2+1)*R1P ints = a multiple of 16 bytes)
  const int tid = threadIdx.x, pz = tid % ZC, g = tid / ZC;
  const unsigned ncol = (unsigned)a.ncol;
  const unsigned col = blockIdx.x * ZC + pz;
  const bool colok = col < ncol;
  // bands of this group: b = blockIdx.y, blockIdx.y + ng, ...
  const size_t bstride = (size_t)a.L1 * a.ncol;
  const cplx* base = a.planes + (colok ? col : 0);
  for (int i = tid; i < (R2 + 1) * R1P; i += NT) {
    const int j2 = i / R1P, j1 = i % R1P;
    int lx = -1;
    if (j2 < R2 && j1 < R1) {
      lx = j1 * R2 + j2 - a.x0;
      if (lx < 0) lx += NX;
      if (lx >= a.L1) lx = -1;
    }
    rlx[i] = lx;
  }
  for (int i = tid; i < NX; i += NT) tw[i] = a.tw_x[i];
  auto prefetch = [&](int b) {          // rows lx = g, g+G, ... of band b, column pz
    if (colok)
      for (int lx = g; lx < a.L1; lx += G) cp16m(stage + lx * ZC + pz, base + (size_t)b * bstride + (unsigned)lx * ncol);
    cp_commit_m();
  };
  int b = blockIdx.y;
  if (b < a.nb) prefetch(b);
  double acc[IT2][R2];
#pragma unroll
  for (int i = 0; i < IT2; ++i)
#pragma unroll
    for (int k = 0; k < R2; ++k) acc[i][k] = 0.0;
  for (; b < a.nb; b += a.ng) {
    cp_wait_n(0);
    __syncthreads();                    // band b staged (and, first time, the tables); the tile is free
    for (int j2 = g; j2 < R2; j2 += G) {
      const int* t = rlx + ((colok) ? j2 : R2) * R1P;
      cplx v[R1];
#pragma unroll
      for (int j1 = 0; j1 < R1; ++j1) {
        const int lx = t[j1];
        v[j1] = (lx >= 0) ? stage[lx * ZC + pz] : cmake(0.0, 0.0);
      }
      dft<R1, +1>(v);
      cplx* o = tile + j2 * ZC + pz;
#pragma unroll
      for (int k1 = 0; k1 < R1; ++k1) o[k1 * R2 * ZC] = (k1 == 0) ? v[0] : mul_tw<+1>(v[k1], tw, j2 * k1);
    }
    __syncthreads();                    // tile complete; the staging buffer is free
    if (b + a.ng < a.nb) prefetch(b + a.ng);
    const double f = __ldg(a.occ + b);
#pragma unroll
    for (int i = 0; i < IT2; ++i) {
      const int k1 = g + i * G;
      if (R1 % G == 0 || k1 < R1) {
        cplx v[R2];
        const cplx* t = tile + k1 * R2 * ZC + pz;
#pragma unroll
        for (int j2 = 0; j2 < R2; ++j2) v[j2] = t[j2 * ZC];
        dft<R2, +1>(v);
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) acc[i][k2] = fma(f, fma(v[k2].x, v[k2].x, v[k2].y * v[k2].y), acc[i][k2]);
      }
    }
  }
  if (!colok) return;
  double* out = a.part + (size_t)blockIdx.y * NX * a.ncol + col;
#pragma unroll
  for (int i = 0; i < IT2; ++i) {
    const int k1 = g + i * G;
    if (R1 % G == 0 || k1 < R1) {
#pragma unroll
      for (int k2 = 0; k2 < R2; ++k2) {
        double* q = out + (size_t)(k1 * R2 + k2) * a.ncol;
        *q = a.accumulate ? *q + acc[i][k2] : acc[i][k2];
      }
    }
  }
}

// rho[x][y][z] (natural order) = sum over groups, in order, of part[g][px][py][pz]
__global__ void k_rho_finish(const double* __restrict__ part, int ng, double* __restrict__ rho, int n1, int n2, int n3,
                             int a1, int b1, int a2, int b2, int a3, int b3) {
  const long N = (long)n1 * n2 * n3;
  const long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int pz = (int)(i % n3), py = (int)((i / n3) % n2), px = (int)(i / ((long)n3 * n2));
  const int x = perm_index(px, a1, b1), y = perm_index(py, a2, b2), z = perm_index(pz, a3, b3);
  double s = 0.0;
  for (int g = 0; g < ng; ++g) s += part[(size_t)g * N + i];
  rho[((long)x * n2 + y) * n3 + z] = s;
}

// ------------------------------------------------------------------------------------------------
// host: configuration and launch
// ------------------------------------------------------------------------------------------------
static const size_t KS_SMEM_MAX = 227 * 1024;
static const size_t KS_SMEM_MAX_K = 226 * 1024;   // the k-batched kernels keep their descriptor in static shared memory

static size_t yz_smem(const HpsiPlan& P, int zc) {
  const size_t SZ = (size_t)((P.n3 / P.zs_yz) | 1);
  return sizeof(cplx) * ((size_t)P.n2 + (P.n2 == P.n3 ? 0 : P.n3) + (size_t)P.smax * SZ + (size_t)P.n2 * zc);
}

// Tensor map of the live-plane workspace seen as a 2-D array of doubles [batch_cap * L1 * n2 rows][2 * n3], box = one y tile
// ([n2 rows][2 * zc doubles], dense in shared memory: no swizzle, no interleave).  cuTensorMapEncodeTiled is a driver entry
// point: looked up through the runtime so that libkspw.so does not link libcuda.
typedef CUresult (*ks_encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                       const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                       CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
int ks_hpsi_make_tmap(HpsiPlan& P, std::string& err) {
  P.tmap_ok = false;
  bool want = false;
#define C_(A_, B_) if (P.n2 == A_ && P.n3 == B_) want = yzcfg<A_, B_>::TMA;
  KS_YZ_PAIRS(C_)
#undef C_
  if (!want || !P.d_planes) return KS_OK;
  static ks_encode_tiled_fn enc = nullptr;
  if (!enc) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess || !fn) return KS_OK;   // no TMA path
    enc = (ks_encode_tiled_fn)fn;
  }
  const cuuint64_t dims[2] = {(cuuint64_t)2 * P.n3, (cuuint64_t)P.batch_cap * P.L1 * P.n2};
  const cuuint64_t strides[1] = {(cuuint64_t)2 * P.n3 * sizeof(double)};
  const cuuint32_t box[2] = {(cuuint32_t)(2 * P.zc_yz), (cuuint32_t)P.n2};
  const cuuint32_t estr[2] = {1, 1};
  static_assert(sizeof(CUtensorMap) == sizeof(P.tmap_planes), "tensor map storage");
  const CUresult r = enc((CUtensorMap*)P.tmap_planes, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, P.d_planes, dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { err = "cuTensorMapEncodeTiled failed for the live-plane workspace"; return KS_ECUDA; }
  P.tmap_ok = true;
  return KS_OK;
}
template <int NX> static constexpr size_t x_smem(int L1) {      // L1 = NX: the most any context of this size can need
  return sizeof(cplx) * ((size_t)NX + (size_t)NX * xcfg<NX>::ZC + (xcfg<NX>::STAGE ? (size_t)L1 * xcfg<NX>::ZC : 0)) +
         sizeof(unsigned) * (fac<NX>::R2 + 1) * ((fac<NX>::R1 + 3) & ~3);
}

// the forward yz kernel runs as clusters of ZS CTAs along x when the plane's z' positions are split (yzcfg)
template <int NY, int NZ>
static cudaError_t launch_fwd_yz(dim3 grid, size_t smem, cudaStream_t st, const YzArgs& a) {
  if (yzcfg<NY, NZ>::ZS == 1) {
    k_fwd_yz<NY, NZ><<<grid, yzcfg<NY, NZ>::NT, smem, st>>>(a);
    return cudaSuccess;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = dim3(yzcfg<NY, NZ>::NT); cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = yzcfg<NY, NZ>::ZS; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, k_fwd_yz<NY, NZ>, a);
}

template <typename K>
static cudaError_t opt_in(K kern, size_t bytes) {
  return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

int ks_hpsi_configure(HpsiPlan& P, std::string& err) {
  if (!ks_fft_size_supported(P.n1) || !ks_fft_yz_supported(P.n2, P.n3)) {
    char b[200];
    snprintf(b, sizeof b, "FFT grid %dx%dx%d is not in the supported set (see ks_supported_sizes; n2,n3 must be a supported pair)",
             P.n1, P.n2, P.n3);
    err = b;
    return KS_EGRID;
  }
  cudaError_t e = cudaSuccess;
  P.zc_yz = 0;
#define C_(A_, B_)                                                              \
  if (P.n2 == A_ && P.n3 == B_) {                                               \
    P.zc_yz = yzcfg<A_, B_>::ZC;                                                \
    P.zs_yz = yzcfg<A_, B_>::ZS;                                                \
    P.smem_yz = yz_smem(P, P.zc_yz * yzcfg<A_, B_>::NG);                        \
    if (P.smem_yz > KS_SMEM_MAX) { err = "yz kernels: stick tile does not fit in 227 KB of shared memory"; return KS_ENOMEM; } \
    /* the attribute belongs to the kernel, not to the context: opt in to the hardware maximum once, so contexts  \
       with different spheres (stick tiles) on the same plane size never lower each other's limit */               \
    e = opt_in(k_inv_yz<A_, B_>, KS_SMEM_MAX);                                  \
    if (e == cudaSuccess) e = opt_in(k_inv_yz_tma<A_, B_>, KS_SMEM_MAX);        \
    if (e == cudaSuccess) e = opt_in(k_fwd_yz<A_, B_>, KS_SMEM_MAX);            \
    if (e == cudaSuccess) e = opt_in(k_inv_yz_k<A_, B_>, KS_SMEM_MAX_K);        \
    if (e == cudaSuccess) e = opt_in(k_fwd_yz_k<A_, B_>, KS_SMEM_MAX_K);        \
  }
  KS_YZ_PAIRS(C_)
#undef C_
  KS_CUDA_CHECK(e, err);
  // (opt-in to the size's maximum, L1 = n1, for the same reason as above)
#define C_(N_) if (P.n1 == N_) { P.zc_x = xcfg<N_>::ZC; P.smem_x = x_smem<N_>(P.L1); e = opt_in(k_x<N_>, x_smem<N_>(N_)); if (e == cudaSuccess) e = opt_in(k_x_k<N_>, x_smem<N_>(N_)); }
  KS_X_SIZES(C_)
#undef C_
  KS_CUDA_CHECK(e, err);
  return KS_OK;
}

// bands per k_x CTA: long enough to amortise the prologue and hide the loads, short enough that the grid
// still has several CTAs per resident slot (148 SMs x 4 CTAs)
static int ks_x_band_group(int nchunk, int nb) {
  static const int env = getenv("KSPW_X_BG") ? atoi(getenv("KSPW_X_BG")) : 0;
  if (env > 0) return std::min(env, nb);
  int bg = 8;
  while (bg > 1 && (long)nchunk * ceil_div(nb, bg) < 4L * 148 * 4) bg /= 2;
  return std::min(bg, nb);
}

// L2 prefetch distance of k_inv_yz: the number of CTAs in flight (one wave), KSPW_PF_DIST=<n> overrides (0 = off)
static int ks_pf_dist(const HpsiPlan& P) {
  static int nsm = 0;
  if (!nsm) { int dev = 0; cudaGetDevice(&dev); if (cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || nsm <= 0) nsm = 148; }
  static const int env_pf = getenv("KSPW_PF_DIST") ? atoi(getenv("KSPW_PF_DIST")) : -1;
  // CTAs per SM: one where the stick tile fills the SM, two otherwise (launch bounds of the yz kernels)
  const int per_sm = P.smem_yz > KS_SMEM_MAX / 2 ? 1 : 2;
  return env_pf >= 0 ? env_pf : nsm * per_sm;
}

int ks_hpsi_local_launch(const HpsiPlan& P, const cplx* psi, cplx* hpsi, int nb, cudaStream_t st,
                         std::string& err, int stage) {
  if (nb <= 0) return KS_OK;
  if (nb > P.batch_cap) { err = "internal: FFT batch larger than workspace"; return KS_EINVAL; }
  YzArgs a;
  a.psi = psi; a.hpsi = hpsi; a.planes = P.d_planes;
  a.plane_s0 = P.d_plane_s0; a.plane_y0 = P.d_plane_y0; a.plane_pw0 = P.d_plane_pw0; a.stick = P.d_stick;
  a.g2 = P.d_g2; a.tw_y = P.d_tw[1]; a.tw_z = P.d_tw[2];
  a.npw = P.npw; a.L1 = P.L1; a.smax = P.smax; a.nb = nb; a.invN = 1.0 / (double)P.N;
  a.pf_dist = ks_pf_dist(P);
  XArgs x;
  x.planes = P.d_planes; x.vperm = P.d_vperm; x.tw_x = P.d_tw[0];
  x.L1 = P.L1; x.x0 = P.x0; x.ncol = (long)P.n2 * P.n3;
  x.nb = nb; x.bg = ks_x_band_group(ceil_div(x.ncol, P.zc_x), nb);
  const dim3 gyz(P.L1 * P.zs_yz, nb), gx(ceil_div(x.ncol, P.zc_x), ceil_div(nb, x.bg));
  if (stage < 0 || stage == 0) {
#define C_(A_, B_)                                                                                          \
    if (P.n2 == A_ && P.n3 == B_) {                                                                         \
      if (yzcfg<A_, B_>::TMA && P.tmap_ok)                                                                  \
        k_inv_yz_tma<A_, B_><<<gyz, yzcfg<A_, B_>::NT, P.smem_yz, st>>>(a, *(const CUtensorMap*)P.tmap_planes); \
      else k_inv_yz<A_, B_><<<gyz, yzcfg<A_, B_>::NT, P.smem_yz, st>>>(a);                                 \
    }
    KS_YZ_PAIRS(C_)
#undef C_
  }
  if (stage < 0 || stage == 1) {
#define C_(N_) if (P.n1 == N_) k_x<N_><<<gx, xcfg<N_>::NT, P.smem_x, st>>>(x);
    KS_X_SIZES(C_)
#undef C_
  }
  if (stage < 0 || stage == 2) {
    cudaError_t le = cudaSuccess;
#define C_(A_, B_) if (P.n2 == A_ && P.n3 == B_) le = launch_fwd_yz<A_, B_>(gyz, P.smem_yz, st, a);
    KS_YZ_PAIRS(C_)
#undef C_
    KS_CUDA_CHECK(le, err);
  }
  KS_CUDA_CHECK(cudaGetLastError(), err);
  return KS_OK;
}

// ---- k-batched launch (ks_hpsi_batch): one grid over (plane | column chunk, band, k-point) per kernel ----
// Descriptor block of a group of nk k-points, built on the host and copied to the device by the caller:
// [YzArgs x nk][XArgs x nk].  All k-points of a group share the grid size (same kernel instantiation).
size_t ks_kdesc_bytes(int nk) { return (sizeof(YzArgs) + sizeof(XArgs)) * (size_t)nk; }

void ks_kdesc_fill(void* host_desc, const KItem* items, int nk) {
  YzArgs* ya = (YzArgs*)host_desc;
  XArgs* xa = (XArgs*)(ya + nk);
  int nbmax = 0;
  for (int i = 0; i < nk; ++i) nbmax = std::max(nbmax, items[i].nb);
  const HpsiPlan& P0 = *items[0].P;
  const long ncol = (long)P0.n2 * P0.n3;
  const int bg = ks_x_band_group(ceil_div(ncol, P0.zc_x) * nk, nbmax);
  for (int i = 0; i < nk; ++i) {
    const HpsiPlan& P = *items[i].P;
    YzArgs& a = ya[i];
    a.psi = items[i].psi; a.hpsi = items[i].hpsi; a.planes = P.d_planes;
    a.plane_s0 = P.d_plane_s0; a.plane_y0 = P.d_plane_y0; a.plane_pw0 = P.d_plane_pw0; a.stick = P.d_stick;
    a.g2 = P.d_g2; a.tw_y = P.d_tw[1]; a.tw_z = P.d_tw[2];
    a.npw = P.npw; a.L1 = P.L1; a.smax = P.smax; a.nb = items[i].nb; a.invN = 1.0 / (double)P.N;
    a.pf_dist = 0;      // k-batched grids: the launch order runs over k-points with different spheres: no prefetch
    XArgs& x = xa[i];
    x.planes = P.d_planes; x.vperm = P.d_vperm; x.tw_x = P.d_tw[0];
    x.L1 = P.L1; x.x0 = P.x0; x.ncol = ncol; x.nb = items[i].nb; x.bg = std::min(bg, std::max(1, items[i].nb));
  }
}

int ks_hpsi_local_launch_k(const KItem* items, int nk, const void* dev_desc, cudaStream_t st, std::string& err, int stage) {
  if (nk <= 0) return KS_OK;
  const HpsiPlan& P0 = *items[0].P;
  int nbmax = 0, l1max = 0;
  size_t smem_yz = 0, smem_x = 0;
  for (int i = 0; i < nk; ++i) {
    const HpsiPlan& P = *items[i].P;
    smem_x = std::max(smem_x, P.smem_x);
    if (P.n1 != P0.n1 || P.n2 != P0.n2 || P.n3 != P0.n3) { err = "ks_hpsi_batch: the k-points of a batch must share the FFT grid"; return KS_EINVAL; }
    if (items[i].nb > P.batch_cap) { err = "internal: FFT batch larger than workspace"; return KS_EINVAL; }
    nbmax = std::max(nbmax, items[i].nb); l1max = std::max(l1max, P.L1);
    smem_yz = std::max(smem_yz, P.smem_yz);
  }
  if (nbmax == 0) return KS_OK;
  if (smem_yz > KS_SMEM_MAX_K) { err = "ks_hpsi_batch: stick tile does not fit next to the descriptor in shared memory"; return KS_ENOMEM; }
  const YzArgs* ya = (const YzArgs*)dev_desc;
  const XArgs* xa = (const XArgs*)(ya + nk);
  const long ncol = (long)P0.n2 * P0.n3;
  const int bg = ks_x_band_group(ceil_div(ncol, P0.zc_x) * nk, nbmax);
  const dim3 gyz(l1max * P0.zs_yz, nbmax, nk), gx(ceil_div(ncol, P0.zc_x), ceil_div(nbmax, bg), nk);
  if (stage < 0 || stage == 0) {
#define C_(A_, B_) if (P0.n2 == A_ && P0.n3 == B_) k_inv_yz_k<A_, B_><<<gyz, yzcfg<A_, B_>::NT, smem_yz, st>>>(ya);
    KS_YZ_PAIRS(C_)
#undef C_
  }
  if (stage < 0 || stage == 1) {
#define C_(N_) if (P0.n1 == N_) k_x_k<N_><<<gx, xcfg<N_>::NT, smem_x, st>>>(xa);
    KS_X_SIZES(C_)
#undef C_
  }
  if (stage < 0 || stage == 2) {
    cudaError_t le = cudaSuccess;
#define C_(A_, B_)                                                                                      \
    if (P0.n2 == A_ && P0.n3 == B_) {                                                                   \
      if (yzcfg<A_, B_>::ZS == 1) k_fwd_yz_k<A_, B_><<<gyz, yzcfg<A_, B_>::NT, smem_yz, st>>>(ya);      \
      else {                                                                                            \
        cudaLaunchConfig_t cfg = {};                                                                    \
        cfg.gridDim = gyz; cfg.blockDim = dim3(yzcfg<A_, B_>::NT); cfg.dynamicSmemBytes = smem_yz; cfg.stream = st; \
        cudaLaunchAttribute at[1];                                                                      \
        at[0].id = cudaLaunchAttributeClusterDimension;                                                 \
        at[0].val.clusterDim.x = yzcfg<A_, B_>::ZS; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1; \
        cfg.attrs = at; cfg.numAttrs = 1;                                                               \
        le = cudaLaunchKernelEx(&cfg, k_fwd_yz_k<A_, B_>, ya);                                          \
      }                                                                                                 \
    }
    KS_YZ_PAIRS(C_)
#undef C_
    KS_CUDA_CHECK(le, err);
  }
  KS_CUDA_CHECK(cudaGetLastError(), err);
  return KS_OK;
}

// ---- density build: launchers ----
template <int NX> static size_t rho_smem(int L1) {
  return sizeof(cplx) * ((size_t)NX + (size_t)NX * rcfg<NX>::ZC + (size_t)L1 * rcfg<NX>::ZC) +
         sizeof(int) * (fac<NX>::R2 + 1) * ((fac<NX>::R1 + 3) & ~3);
}

int ks_density_batch(HpsiPlan& P, const cplx* psi, const double* occ, int nb, int first, cudaStream_t st, std::string& err) {
  if (nb <= 0) return KS_OK;
  if (nb > P.batch_cap) { err = "internal: FFT batch larger than workspace"; return KS_EINVAL; }
  const long ncol = (long)P.n2 * P.n3;
  int zc_r = 0, nt_r = 0;
#define C_(N_) if (P.n1 == N_) { zc_r = rcfg<N_>::ZC; nt_r = rcfg<N_>::NT; }
  KS_X_SIZES(C_)
#undef C_
  const int nchunk = ceil_div(ncol, zc_r);
  if (!P.d_rho_part) {
    // band groups: enough CTAs for ~3 per resident slot, at most 8 partial copies of the grid
    P.rho_ng = std::max(1, std::min(8, ceil_div(3L * 148 * 3, nchunk)));
    KS_CUDA_CHECK(cudaMalloc(&P.d_rho_part, sizeof(double) * (size_t)P.rho_ng * P.N), err);
  }
  YzArgs a;
  a.psi = psi; a.hpsi = nullptr; a.planes = P.d_planes;
  a.plane_s0 = P.d_plane_s0; a.plane_y0 = P.d_plane_y0; a.plane_pw0 = P.d_plane_pw0; a.stick = P.d_stick;
  a.g2 = P.d_g2; a.tw_y = P.d_tw[1]; a.tw_z = P.d_tw[2];
  a.npw = P.npw; a.L1 = P.L1; a.smax = P.smax; a.nb = nb; a.invN = 1.0 / (double)P.N;
  a.pf_dist = ks_pf_dist(P);
  const dim3 gyz(P.L1 * P.zs_yz, nb);
#define C_(A_, B_) if (P.n2 == A_ && P.n3 == B_) k_inv_yz<A_, B_><<<gyz, yzcfg<A_, B_>::NT, P.smem_yz, st>>>(a);
  KS_YZ_PAIRS(C_)
#undef C_
  RhoArgs r;
  r.planes = P.d_planes; r.occ = occ; r.part = P.d_rho_part; r.tw_x = P.d_tw[0];
  r.L1 = P.L1; r.x0 = P.x0; r.nb = nb; r.ng = P.rho_ng; r.accumulate = first ? 0 : 1; r.ncol = ncol;
  const dim3 gr(nchunk, P.rho_ng);
  cudaError_t e = cudaSuccess;
#define C_(N_)                                                                                         \
  if (P.n1 == N_) {                                                                                     \
    const size_t smem = rho_smem<N_>(P.L1);                                                             \
    if (smem > KS_SMEM_MAX) { err = "density kernel: tile + staging do not fit in shared memory"; return KS_ENOMEM; } \
    e = opt_in(k_rho<N_>, smem);                                                                        \
    if (e == cudaSuccess) k_rho<N_><<<gr, nt_r, smem, st>>>(r);                                 \
  }
  KS_X_SIZES(C_)
#undef C_
  KS_CUDA_CHECK(e, err);
  KS_CUDA_CHECK(cudaGetLastError(), err);
  return KS_OK;
}

int ks_density_finish(const HpsiPlan& P, double* rho, cudaStream_t st, std::string& err) {
  int f[6];
  const int nn[3] = {P.n1, P.n2, P.n3};
  for (int ax = 0; ax < 3; ++ax) ks_fft_factors(nn[ax], &f[2 * ax], &f[2 * ax + 1], ax);
  k_rho_finish<<<ceil_div(P.N, 256), 256, 0, st>>>(P.d_rho_part, P.rho_ng, rho, P.n1, P.n2, P.n3, f[0], f[1], f[2], f[3], f[4], f[5]);
  KS_CUDA_CHECK(cudaGetLastError(), err);
  return KS_OK;
}
