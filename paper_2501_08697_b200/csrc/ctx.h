// ctx.h -- the opaque ks_ctx behind include/kspw.h (internal).
#pragma once
#include "plan.h"

struct DavidsonWs {
  int nb_cap = 0;
  cplx *V = nullptr, *W = nullptr;       // [2 nb][npw]
  cplx *X = nullptr, *HX = nullptr;      // [nb][npw]
  cplx *T = nullptr;                     // [nb][npw]
  cplx *Hc = nullptr, *Cm = nullptr;     // [2nb x 2nb] subspace matrix / eigenvectors (column-major)
  cplx *Hwork = nullptr;                 // [2nb x 2nb] copy destroyed by the eigensolver
  cplx *S = nullptr, *Us = nullptr;      // [2nb x nb] projections / [nb x nb] Gram matrices
  double *theta = nullptr;               // [2nb]
  double *rho = nullptr, *ekin = nullptr, *lam = nullptr;   // [nb]
  int *idx = nullptr;                    // [nb] unconverged band list / kept column list
};

struct ks_ctx {
  HpsiPlan P;
  int nproj = 0, natom = 0;
  cplx* d_beta = nullptr;        // [nproj][npw]
  double* d_D = nullptr;         // concatenated blocks
  int* d_proj_atom = nullptr;    // [nproj]
  int* d_off = nullptr;          // [natom+1]
  long* d_doff = nullptr;        // [natom]
  cplx *d_B = nullptr, *d_DB = nullptr;   // [nproj x nb_cap] column-major
  int nl_cap = 0;
  cplx *d_hin = nullptr, *d_hout = nullptr;   // staging for the *_host entry points
  size_t host_stage_bytes = 0;
  GemmWs gws;
  EighWs ews;
  DavidsonWs dws;
  cudaStream_t stream = 0;
  int fft_batch = 0;             // bands per FFT batch
  double prof_ms[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  std::string err;
};

int ks_hpsi_impl(ks_ctx* c, const cplx* psi, cplx* hpsi, int nb);
int ks_davidson_impl(ks_ctx* c, cplx* psi, double* eig, int nb, double tol, int max_iter, double* resid,
                     int* iters_out, long long* nhpsi_out);
void ks_davidson_free(DavidsonWs* w);
