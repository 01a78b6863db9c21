// plan.h -- internal (host) description of one k-point's H*psi plan and the launchers the
// translation units of libkspw.so share.  Not part of the C ABI (include/kspw.h).
#pragma once
#include "common.cuh"
#include <vector>

struct HpsiPlan {
  int n1 = 0, n2 = 0, n3 = 0, npw = 0;
  long N = 0;
  int L1 = 0;          // number of live x-planes (distinct m1 of the sphere)
  int x0 = 0;          // natural x index (m1min mod n1) of live plane 0; plane lx is x = (x0+lx) mod n1
  int nsticks = 0;     // z-sticks (distinct (m1,m2)) of the sphere
  int smax = 0;        // max sticks in one plane
  int zc_yz = 0, zc_x = 0;        // z-chunk sizes of the yz kernels and of the x kernel
  int zs_yz = 1;                  // CTAs that share one (band, plane) of the yz kernels, each owning n3/zs_yz z' positions
  size_t smem_yz = 0, smem_x = 0;
  // device arrays
  int* d_plane_s0 = nullptr;   // [L1+1] first stick of each plane
  int* d_plane_y0 = nullptr;   // [L1]   natural y index (m2min mod n2) of the plane's first stick
  int* d_plane_pw0 = nullptr;  // [L1+1] first plane wave of each plane (the plane's coefficients are one contiguous run of psi)
  int4* d_stick = nullptr;     // [nsticks] {first PW, natural z index (m3min mod n3) of it, number of PWs, 0}:
                               //           a stick's coefficients are a contiguous run of psi, ascending in m3
  double* d_g2 = nullptr;      // [npw]  |k+G|^2
  double* d_vperm = nullptr;   // [n1][n2][n3] V(r) in position (type-A output) order on all three axes
  cplx* d_tw[3] = {nullptr, nullptr, nullptr};  // e^{+2 pi i t/n_i}
  cplx* d_planes = nullptr;    // workspace [batch][L1][n2][n3]
  int batch_cap = 0;           // bands the workspace holds
  alignas(64) unsigned char tmap_planes[128] = {};   // CUtensorMap of d_planes (box = one y tile); rebuilt when d_planes moves
  bool tmap_ok = false;
  double* d_rho_part = nullptr;  // density build: [rho_ng][n1][n2][n3] partial sums in position order (lazy)
  int rho_ng = 0;
};

bool ks_fft_size_supported(int n);
bool ks_fft_yz_supported(int n2, int n3);
int ks_fft_sizes(int* out, int cap);
void ks_fft_factors(int n, int* R1, int* R2, int axis = 0);   // axis 2 (z sticks) may use its own split
cudaError_t ks_fft_init_constants();

// V(r) = Re sum_m vhat[m] e^{+2 pi i m.j/n} on the device by a plain O(N n) DFT per axis (create time
// only), checked real, stored permuted.  vhat_host: [n1][n2][n3].  Returns KS_* and fills err.
int ks_build_vperm(HpsiPlan& P, const cplx* vhat_host, cudaStream_t st, std::string& err);

// (re)build the tensor map of the live-plane workspace for the kernels that store planes by TMA (after d_planes changed)
int ks_hpsi_make_tmap(HpsiPlan& P, std::string& err);

// fill zc_*/smem_* for the plan and opt the kernels into large dynamic shared memory
int ks_hpsi_configure(HpsiPlan& P, std::string& err);

// local + kinetic part: hpsi[b][j] = g2[j] psi[b][j] + (1/N) FFT^-[ V(r) FFT^+[psi_b] ](G_j) for nb bands
// (nb <= batch_cap), three launches on `st`.
// stage: 0 = k_inv_yz, 1 = k_x, 2 = k_fwd_yz, -1 = all three in order.
int ks_hpsi_local_launch(const HpsiPlan& P, const cplx* psi, cplx* hpsi, int nb, cudaStream_t st,
                         std::string& err, int stage = -1);

// k-batched form of the same three launches (ks_hpsi_batch): the k-points of one group share the FFT grid; every kernel is
// ONE launch over (plane | column chunk, band, k-point).  The caller owns the descriptor block: ks_kdesc_fill writes
// ks_kdesc_bytes(nk) bytes on the host, the caller copies them to the device (dev_desc) before the launch.
struct KItem { const HpsiPlan* P; const cplx* psi; cplx* hpsi; int nb; };
size_t ks_kdesc_bytes(int nk);
void ks_kdesc_fill(void* host_desc, const KItem* items, int nk);
int ks_hpsi_local_launch_k(const KItem* items, int nk, const void* dev_desc, cudaStream_t st, std::string& err, int stage = -1);

// density build: rho(r) += occ_b |psi_b(r)|^2 for one batch of bands (k_inv_yz + k_rho; first != 0 starts a new sum),
// then ks_density_finish adds the band groups in order and writes rho[n1][n2][n3] in natural order.
int ks_density_batch(HpsiPlan& P, const cplx* psi, const double* occ, int nb, int first, cudaStream_t st, std::string& err);
int ks_density_finish(const HpsiPlan& P, double* rho, cudaStream_t st, std::string& err);

// ---- dense kernels (gemm.cu, eigh.cu) ----
struct GemmWs {          // split-K partial sums
  cplx* part = nullptr;
  size_t bytes = 0;
};
// herm_r0 >= 0: rows herm_r0 .. herm_r0 + N - 1 of C form a Hermitian N x N block (A's columns herm_r0.. and B's columns
// span it: a Gram matrix T^H T with herm_r0 = 0, the corner V_new^H (H V_new) of the subspace matrix); only the tiles
// that reach its upper triangle (row - herm_r0 <= column) are computed, the elements strictly below the diagonal are
// NOT written (the caller mirrors or ignores them).
int ks_gemm_hn(cudaStream_t st, int M, int N, int K, const cplx* A, long lda, const cplx* B, long ldb,
               cplx* C, long ldc, GemmWs* ws, std::string& err, int herm_r0 = -1);
// btri_c0 >= 0: B is upper triangular in the sense B[k][n] = 0 for k > btri_c0 + n (an inverse Cholesky factor, btri_c0 = 0):
// every N-tile stops its K loop at its last non-zero row.
int ks_gemm_nn(cudaStream_t st, int M, int N, int K, const cplx* A, long lda, const cplx* B, long ldb,
               cplx* C, long ldc, int accumulate, std::string& err, int btri_c0 = -1);

// grouped launches (ks_hpsi_batch): ng independent problems of similar size in one launch; dev_probs is a DEVICE array
struct GemmProb {
  const cplx* A; const cplx* B;     // hn: A is K x M, B is K x N ; nn: A is M x K, B is K x N (column-major)
  cplx* C;                          // hn: partial sums [nsplit][N][M] ; nn: M x N with ldc
  int M, N, K;
  long lda, ldb, ldc;
};
int ks_gemm_hn_group_nsplit(int ng, int M, int N, int K);
int ks_gemm_hn_group(cudaStream_t st, const GemmProb* dev_probs, int ng, int M, int N, int nsplit, std::string& err);
int ks_gemm_nn_group(cudaStream_t st, const GemmProb* dev_probs, int ng, int M, int N, int accumulate, std::string& err);

int ks_dmma_latency_run(double* clk_per_dmma, double sm_ghz, std::string& err);
int ks_fp64_mix_run(double* tflops4, std::string& err);
int ks_peak_run(double* dmma_tf, double* dfma_tf, std::string& err);

struct EighWs {
  cplx* U = nullptr;       // per-pair rotation blocks [nblk/2][64*64]
  cplx* Ap = nullptr;      // padded working copy of A   [np*np]
  cplx* Vp = nullptr;      // padded eigenvector accumulator [np*np]
  double* diag = nullptr;  // [np]
  double* red = nullptr;   // [2] off^2, tot^2
  double* red_sweeps = nullptr;   // cooperative solve: [2 x 40] off^2, tot^2 per sweep, then the sweep count (int)
  int* order = nullptr;    // [np]
  int2* pairs = nullptr;   // [(nblk-1)][nblk/2] block pairs of every round
  int2* where = nullptr;   // [(nblk-1)][nblk] block -> (index of its pair in the round, 0/1 = first/second of the pair)
  cplx* Ap2 = nullptr;     // second copy of A: the one-launch-per-round path reads one and writes the other
  int cap = 0;             // padded n the buffers hold
  int np = 0;              // padded n of the current run
  int pairs_nblk = 0;      // nblk the pair table was built for
};
int ks_eigh_run(cudaStream_t st, int n, cplx* A, long lda, double* theta, cplx* C, long ldc, EighWs* ws,
                int* sweeps_out, std::string& err);
void ks_eigh_free(EighWs* ws);
