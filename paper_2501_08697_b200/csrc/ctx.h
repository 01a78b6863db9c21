// ctx.h -- the opaque ks_ctx behind include/kspw.h (internal).
#pragma once
#include "plan.h"

struct DavidsonWs {
  int nb_cap = 0;
  cplx *V = nullptr, *W = nullptr;       // [2 nb][npw]
  cplx *X = nullptr, *HX = nullptr;      // [nb][npw]
  cplx *T = nullptr;                     // [nb][npw]
  cplx *SV = nullptr, *SX = nullptr, *ST = nullptr;   // generalised problem only: S V [2nb], S X [nb], S T scratch [nb]
  int s_cap = 0;
  cplx *Hc = nullptr, *Cm = nullptr;     // [2nb x 2nb] subspace matrix / eigenvectors (column-major)
  cplx *Hwork = nullptr;                 // [2nb x 2nb] copy destroyed by the eigensolver
  cplx *Cp = nullptr, *Cq = nullptr;     // [2nb x 2nb] eigenvectors of the previous iteration / of the rotated matrix
  double *thp = nullptr;                 // [2nb] Ritz values of the previous iteration
  double *thf = nullptr;                 // [2nb] eigenvalues of the deflated (unlocked) subspace problem
  int *lst = nullptr;                    // [3 x 2nb] locked rows L, free rows F, row -> position in F (or -1)
  int2 *src = nullptr;                   // [2nb] merged order: (is_locked, index into L or F)
  cplx *S = nullptr, *Us = nullptr;      // [2nb x nb] projections / [nb x nb] Gram matrices
  double *theta = nullptr;               // [2nb]
  double *rho = nullptr, *ekin = nullptr, *lam = nullptr;   // [nb]
  double *lam0 = nullptr, *thr = nullptr;                   // [nb] squared column norms before the projection; drop thresholds
  int *idx = nullptr;                    // [nb] unconverged band list / kept column list
  int *act = nullptr;                    // [nb] bands whose Ritz vectors are rotated this iteration
};

struct KBatchWs {     // ks_hpsi_batch / ks_davidson_batch state kept in the FIRST context of the batch
  char* h = nullptr;                 // pinned host descriptor block
  char* d = nullptr;                 // its device copy
  size_t bytes = 0;
  cudaEvent_t ev = nullptr;          // recorded after the descriptor copy of the last call
  bool ev_pending = false;
  std::vector<cudaStream_t> pool;    // ks_davidson_batch: one stream per worker thread
  std::vector<cudaEvent_t> pool_ev;
};

struct ks_ctx {
  HpsiPlan P;
  int nproj = 0, natom = 0;
  cplx* d_beta = nullptr;        // [nproj][npw]
  double* d_D = nullptr;         // concatenated blocks
  double* d_Q = nullptr;         // overlap blocks q^a (same layout); nullptr: S = I
  int* d_proj_atom = nullptr;    // [nproj]
  int* d_off = nullptr;          // [natom+1]
  long* d_doff = nullptr;        // [natom]
  cplx *d_B = nullptr, *d_DB = nullptr;   // [nproj x nb_cap] column-major
  int nl_cap = 0;
  cplx *d_hin = nullptr, *d_hout = nullptr;   // staging for the *_host entry points
  cplx *d_cheb[3] = {nullptr, nullptr, nullptr};   // ks_chebyshev: T_{n-1}, T_n, H T_n  [nb_cap][npw] each
  size_t cheb_bytes = 0;
  size_t host_stage_bytes = 0;
  GemmWs gws;
  EighWs ews;
  DavidsonWs dws;
  KBatchWs kb;
  cudaStream_t stream = 0;
  // ks_hpsi_host pipeline: copy-in / copy-out streams and per-chunk events (created at first use)
  cudaStream_t s_in = nullptr, s_out = nullptr;
  cudaEvent_t ev_in[8] = {}, ev_done[8] = {}, ev_start = nullptr;
  int fft_batch = 0;             // bands per FFT batch
  double prof_ms[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  // per-kernel CUDA-event timing of ks_hpsi (ks_profile_begin / ks_profile_end); no host syncs while on
  bool kprof_on = false;
  struct KRec { int phase; cudaEvent_t a, b; };
  std::vector<KRec> krecs;
  std::vector<cudaEvent_t> kpool;
  long long klaunch[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  std::string err;
};

enum { KP_INV_YZ = 0, KP_X = 1, KP_FWD_YZ = 2, KP_GEMM_HN = 3, KP_APPLY_D = 4, KP_GEMM_NN = 5, KP_RHO = 6 };
void ks_kprof_begin(ks_ctx* c, int phase, int launches);
void ks_kprof_end(ks_ctx* c);

int ks_hpsi_impl(ks_ctx* c, const cplx* psi, cplx* hpsi, int nb);
int ks_ensure_planes(ks_ctx* c, int nb, cudaStream_t sync_stream);   // live-plane workspace for min(fft_batch, nb) bands
int ks_ensure_nl(ks_ctx* c, int nb, int nsplit);                     // d_DB [nproj x nb] and split-K partials [nsplit][nb][nproj]
void ks_kbatch_free(KBatchWs* w);
int ks_spsi_impl(ks_ctx* c, const cplx* psi, cplx* spsi, int nb);   // S psi = psi + beta q (beta^H psi); a copy when S = I
int ks_davidson_impl(ks_ctx* c, cplx* psi, double* eig, int nb, double tol, int max_iter, double* resid,
                     int* iters_out, long long* nhpsi_out);
void ks_davidson_free(DavidsonWs* w);
int ks_cg_impl(ks_ctx* c, cplx* psi, double* eig, int nb, double tol, int kmaxiter, double* resid, int* steps_out,
               long long* nhpsi_out);
