/* kspw.h -- C ABI of libkspw.so: plane-wave Kohn-Sham H*psi and block-Davidson on one B200 (sm_100a).
 *
 * What the calls compute is fixed by arxiv 2501.08697 (ABACUS review; /root/reference/PAPER.md):
 *   - plane-wave expansion psi_nk(r) = sum_G c_nk(G) e^{i(k+G).r}                  Eq. 31
 *   - KS equation in the PW basis: kinetic (k+G)^2 delta_GG' + V(G-G')            Eq. 32
 *     (Rydberg atomic units here: |k+G|^2, no 1/2 -- DESIGN.md reading C1)
 *   - norm-conserving nonlocal part V_KB = sum D_ll' |beta_lm><beta_l'm'|          Eq. 3-4
 *   - H*psi = FFTs + BLAS, the expensive step of iterative diagonalization         L572-574
 *   - Davidson iterative diagonalization (named only; listing = DESIGN.md §3)     L326, L547, L578
 *   - r->G transform sign and 1/N normalisation                                   Eq. 36
 *
 * Conventions:
 *   ks_c128      interleaved complex128 (re, im).
 *   PW order     m1 slowest, m3 fastest, each ascending over the sphere |k+G|^2 <= ecutwfc (C2, C3);
 *                ks_pw_list returns exactly this order; psi / hpsi / beta use it.
 *   Block layout psi[nbands][npw], band-major (a band is a contiguous vector).
 *   Grid layout  [n1][n2][n3], n3 fastest, FFT index order (m mod n) -- only vloc_g uses it (C5).
 *   HOST / DEVICE is stated per pointer.  Every call returns int: 0 ok, >0 soft status, <0 error.
 *   Nothing here throws or aborts; ks_last_error() gives the text of the last failure.
 *   All device work is enqueued on the context's stream (default: the legacy default stream).
 *   There is no CPU fallback: without a CUDA device ks_create returns KS_ECUDA.
 */
#ifndef KSPW_H
#define KSPW_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ks_ctx ks_ctx;              /* opaque, owned by the library */
typedef struct { double re, im; } ks_c128;

#define KS_OK        0
#define KS_NOTCONV   1   /* ks_davidson: max_iter reached; best X, eps, residuals still written */
#define KS_EINVAL   -1   /* bad argument */
#define KS_EGRID    -2   /* grid violates n_i > 2 m_psi,i + m_V,i, n_i > 2 m_V,i, or size unsupported */
#define KS_ENOMEM   -3   /* device or host allocation failed / shared memory budget exceeded */
#define KS_ECUDA    -4   /* CUDA runtime error (no device, launch failure, ...) */
#define KS_EVLOC    -5   /* V(r) not real within 1e-12 max|V| */

/* ---- pure host helpers (no GPU needed): the G sphere of Eq. 31 ------------------------------- */
/* cell: HOST [9], rows a1 a2 a3 (bohr).  k_frac: HOST [3], k in units of b1 b2 b3.  ecutwfc in Ry. */
int ks_pw_count(const double cell[9], const double k_frac[3], double ecutwfc, int* npw /*HOST out*/);
/* miller: HOST out [npw][3];  g2: HOST out [npw] = |k+G|^2 (Ry), may be NULL. */
int ks_pw_list(const double cell[9], const double k_frac[3], double ecutwfc, int* miller, double* g2);

/* ---- context: one k-point -------------------------------------------------------------------- */
/* All inputs are HOST arrays and are copied; the caller may free them on return.
 *   grid        n1 n2 n3; each must be one of ks_supported_sizes() and satisfy the alias rule.
 *   vloc_g      [n1][n2][n3] Fourier-series coefficients of V_loc (Eq. 32's V(G-G')), FFT index order.
 *   beta        [nproj][npw], ks_pw_list order (Eq. 4's |beta_lm>, as beta(k+G)).  nproj may be 0.
 *   proj_offset [natom+1], projector rows of atom a are proj_offset[a] .. proj_offset[a+1]-1.
 *   D           concatenated per-atom real symmetric blocks, atom a's block is np_a x np_a row-major. */
int ks_create(ks_ctx** out, const double cell[9], const double k_frac[3], double ecutwfc,
              const int grid[3], const ks_c128* vloc_g, int nproj, const ks_c128* beta, int natom,
              const int* proj_offset, const double* D);
void ks_destroy(ks_ctx* ctx);
int ks_npw(const ks_ctx* ctx);
int ks_set_stream(ks_ctx* ctx, void* cuda_stream /* cudaStream_t; NULL = default stream */);
/* bands per launch of the three FFT kernels (0 = automatic: as many as 9 GB of live-plane workspace hold, at most 1024;
 * the planes stream through HBM -- a batch small enough to stay in L2 measured slower) */
int ks_set_fft_batch(ks_ctx* ctx, int nbatch);
const char* ks_last_error(const ks_ctx* ctx);   /* ctx may be NULL: last ks_create failure */
/* writes up to cap supported FFT lengths to sizes (HOST), returns how many exist */
int ks_supported_sizes(int* sizes, int cap);

/* ---- the hot path ---------------------------------------------------------------------------- */
/* hpsi = H psi for a block of bands (steps H1-H8 of DESIGN.md §1).
 * psi, hpsi: DEVICE [nbands][npw], caller-owned, must not alias.  Asynchronous on the stream. */
int ks_hpsi(ks_ctx* ctx, const ks_c128* psi, ks_c128* hpsi, int nbands);
/* same through HOST buffers (copies H2D / D2H inside, synchronises before returning).  The block is processed in chunks of
 * bands so that the copies overlap the kernels (the first chunk half as long as the others); the projector sums of a chunk are
 * split over K differently from those of the whole block, so the result equals ks_hpsi's to rounding, not bit for bit. */
int ks_hpsi_host(ks_ctx* ctx, const ks_c128* psi_host, ks_c128* hpsi_host, int nbands);

/* ---- many k-points at once (the batched multi-k entry point) ------------------------------
 * The KS equation is solved independently for every k-point of the Monkhorst-Pack mesh (ref 128; Eq. 32
 * L507 holds per k; "independently for each k point" L900).  One context = one k-point; these calls take the contexts of
 * nk k-points that share the FFT grid (the same cell and grid, different k: different spheres, beta, |k+G|^2).
 *
 * ks_hpsi_batch: hpsi[i] = H(k_i) psi[i] for every i, the same arithmetic as nk ks_hpsi calls (bit for bit in the local
 * and kinetic part; the projector sums are split differently over K, so equal to rounding).  Every kernel of the path is
 * ONE launch over (plane | column chunk | tile, band, k-point) per group of k-points (default: one group).
 *   ctxs    HOST [nk]  contexts, all distinct, same grid; work is enqueued on the stream of ctxs[0]
 *   psi     HOST [nk]  of DEVICE pointers, psi[i] is [nbands[i]][npw_i]
 *   hpsi    HOST [nk]  of DEVICE pointers, same shapes, must not alias psi[i]
 *   nbands  HOST [nk]  (entries may be 0; then psi[i] / hpsi[i] may be NULL)
 * Asynchronous on the stream.  Errors: KS_EINVAL (NULL, aliasing, mixed grids, a context twice), KS_ENOMEM, KS_ECUDA;
 * the text is ks_last_error(ctxs[0]). */
int ks_hpsi_batch(ks_ctx* const* ctxs, int nk, const ks_c128* const* psi, ks_c128* const* hpsi, const int* nbands);
/* ks_davidson_batch: ks_davidson on every k-point (arguments per k as in ks_davidson; resid, iters_out,
 * band_applications_out, status_out may be NULL).  The solves are independent host-driven iterations: they run on
 * internal worker threads, one CUDA stream each, after the work already enqueued on ctxs[0]'s stream, and the call
 * returns when all have finished.  status_out[i] = that solve's return value; the call returns the first error (< 0)
 * if any, else KS_NOTCONV if some solve hit max_iter, else KS_OK. */
int ks_davidson_batch(ks_ctx* const* ctxs, int nk, ks_c128* const* psi, double* const* eig, const int* nbands, double tol,
                      int max_iter, double* const* resid, int* iters_out, long long* band_applications_out, int* status_out);

/* Density build (the step after diagonalisation in the SCF loop, Fig. 3):
 *   rho(r) = sum_b occ[b] |psi_b(r)|^2,  psi_b(r) = sum_G psi_b(G) e^{+i G.r}  (Eq. 31, unnormalised; the caller
 *   owns 1/Omega and k weights).  Reuses the scatter + inverse-FFT half of ks_hpsi.
 *   psi  DEVICE [nbands][npw];  occ  DEVICE [nbands];  rho  DEVICE out [n1][n2][n3], n3 fastest, natural grid order.
 * The sum over bands has a fixed order (no atomics): the result is reproducible bit for bit.  nbands = 0 gives zeros.
 * Asynchronous on the stream.  Errors: KS_EINVAL (NULL pointer, nbands < 0), KS_ENOMEM, KS_ECUDA. */
int ks_density(ks_ctx* ctx, const ks_c128* psi, const double* occ, int nbands, double* rho);
/* same through HOST buffers (copies inside, synchronises before returning) */
int ks_density_host(ks_ctx* ctx, const ks_c128* psi_host, const double* occ_host, int nbands, double* rho_host);

/* Generalised problem H psi = eps S psi (ultrasoft pseudopotentials):
 *   S = 1 + sum_a sum_{p,p' in a} |beta_p> q^a_pp' <beta_p'|,   q^a real symmetric per atom.
 * ks_set_overlap copies Q (HOST, concatenated per-atom blocks, the layout of D in ks_create); NULL restores S = I.
 * With an overlap set, ks_davidson solves the generalised problem: the returned vectors satisfy X^H S X = I and the
 * residuals are ||H x - eps S x||_2.  ks_hpsi, ks_density, ks_chebyshev and ks_cg are unaffected (they do not use S).
 * ks_spsi: spsi = S psi for a block (DEVICE [nbands][npw], must not alias); a copy when S = I. */
int ks_set_overlap(ks_ctx* ctx, const double* Q);
int ks_spsi(ks_ctx* ctx, const ks_c128* psi, ks_c128* spsi, int nbands);

/* Lowest nbands eigenpairs by the band-by-band preconditioned conjugate gradient of PAPER.md Fig. 10 (L549-570), the
 * eigensolver the paper prints; what the listing omits follows reading C19 of DESIGN.md
 * (K = Teter-Payne-Allan, gamma = Polak-Ribiere, theta = minimiser of the Rayleigh quotient, stop at ||r|| <= tol/2,
 * one closing Rayleigh-Ritz step).  Same arguments and results as ks_davidson; kmaxiter = CG steps allowed per band;
 * steps_out = CG steps taken in total (HOST), band_applications_out = H applications (steps + nbands).
 * Returns KS_OK, KS_NOTCONV (some band used all kmaxiter steps; best pairs still written) or < 0. */
int ks_cg(ks_ctx* ctx, ks_c128* psi, double* eig, int nbands, double tol, int kmaxiter, double* resid,
          int* steps_out, long long* band_applications_out);

/* Chebyshev expansion of an operator function on a block (the inner loop of sDFT: PAPER.md L588,
 * stochastic orbitals Eq. 52, gamma = f_H^{1/2} chi Eq. 54, orders 25..1200 L714):
 *   out = sum_{n=0}^{ncoef-1} coef[n] T_n(Ht) chi,  Ht = (H - ebar)/de,  T_0 = chi, T_1 = Ht chi, T_{n+1} = 2 Ht T_n - T_{n-1}.
 * The caller supplies the coefficients and a scaling with the spectrum of Ht inside [-1, 1] (otherwise T_n grows).
 *   chi, out  DEVICE [nbands][npw], must not alias;  coef  HOST [ncoef];  ncoef - 1 ks_hpsi block applies.
 * Asynchronous on the stream.  Errors: KS_EINVAL (NULL, aliasing, de <= 0, ncoef < 0), KS_ENOMEM, KS_ECUDA. */
int ks_chebyshev(ks_ctx* ctx, const ks_c128* chi, ks_c128* out, int nbands, int ncoef, const double* coef,
                 double ebar, double de);

/* Lowest nbands eigenpairs by block Davidson (steps D0-D9), subspace <= 2 nbands, S = I.
 *   psi    DEVICE [nbands][npw]  in: start vectors (any full-rank block), out: orthonormal eigvecs
 *   eig    DEVICE [nbands] out, ascending (Ry)
 *   resid  DEVICE [nbands] out, ||H x_i - eps_i x_i||_2, may be NULL
 *   tol    convergence: every residual norm <= tol;  max_iter: subspace expansions allowed
 *   iters_out, band_applications_out: HOST out, may be NULL
 * Synchronises the stream once per iteration (reads nbands residual norms back). */
int ks_davidson(ks_ctx* ctx, ks_c128* psi, double* eig, int nbands, double tol, int max_iter,
                double* resid, int* iters_out, long long* band_applications_out);
int ks_davidson_host(ks_ctx* ctx, ks_c128* psi_host, double* eig_host, int nbands, double tol,
                     int max_iter, double* resid_host, int* iters_out,
                     long long* band_applications_out);
/* per-phase device time of the last ks_davidson, milliseconds, HOST out [8]:
 * hpsi, projection GEMMs, eigensolves, rotation GEMMs, residual+precondition, orthonormalise GEMMs,
 * total, reserved.  Only filled when KSPW_PROFILE=1 is set in the environment (adds syncs). */
int ks_davidson_profile(const ks_ctx* ctx, double* ms);

/* Per-kernel device time of ks_hpsi between ks_profile_begin and ks_profile_end, by CUDA events recorded
 * on the context's stream around each launch (no host synchronisation while profiling is on).
 * ms, launches: HOST out [8], indexed 0 k_inv_yz (H1+H2 z,y), 1 k_x (H2 x, H3, H4 x), 2 k_fwd_yz (H4 y,z, H5),
 * 3 beta^H psi GEMM + split-K reduce (H6), 4 D apply (H7), 5 beta (D B) GEMM (H8); 6-7 reserved.
 * launches counts the kernels launched per entry since ks_profile_begin.  ks_profile_end synchronises. */
int ks_profile_begin(ks_ctx* ctx);
int ks_profile_end(ks_ctx* ctx, double* ms, long long* launches);

/* ---- building blocks, exported for unit parity tests and the roofline microbenchmarks -------- */
/* C[M][N] (column-major, ldc) = A^H B;  A: DEVICE K x M column-major lda, B: K x N column-major ldb. */
int ks_zgemm_hn(void* stream, int M, int N, int K, const ks_c128* A, long lda, const ks_c128* B,
                long ldb, ks_c128* C, long ldc);
/* The same product for callers that cannot call cudaMalloc (CUDA graph capture, serving loops): the split-K
 * partial tiles live in a file-scope device array of 8 MiB (held by every GPU that loads the library until the
 * process exits), so the call allocates nothing -- it launches two kernels on `stream`.  Limit: M * N <= 524 288
 * complex128 elements (8 MiB / 16 B); beyond it the call returns KS_EINVAL with the limit in ks_last_error(NULL).
 * Other errors: KS_EINVAL (M, N < 1, K < 0, NULL C, NULL A or B with K > 0, lda/ldb < K, ldc < M), KS_ECUDA.  Every call shares the one array:
 * calls that overlap on the GPU (different streams) race; calls on one stream are ordered.  The array keeps the last
 * call's contents, none of which a later call reads before writing.  The first call on a device looks up the array's
 * device address and opts the kernels in to their shared memory (no allocation either); make it outside a capture.
 * Same arithmetic as ks_zgemm_hn up to the split count (summation order over K).  ("BLAS".) */
int ks_zgemm_hn_static(void* stream, int M, int N, int K, const ks_c128* A, long lda, const ks_c128* B,
                       long ldb, ks_c128* C, long ldc);
/* C[M][N] (column-major) = A B (accumulate=0) or C += A B (accumulate=1); A: M x K, B: K x N. */
int ks_zgemm_nn(void* stream, int M, int N, int K, const ks_c128* A, long lda, const ks_c128* B,
                long ldb, ks_c128* C, long ldc, int accumulate);
/* Hermitian eigenproblem A = C diag(theta) C^H by (block) Jacobi.  A: DEVICE n x n column-major (lda),
 * destroyed; theta: DEVICE [n] ascending; C: DEVICE n x n column-major (ldc), column i <-> theta[i].
 * Returns KS_NOTCONV (best pairs still written) if 40 sweeps did not reach off_F(A) <= 1e-14 ||A||_F (n > 64 only). */
int ks_eigh(void* stream, int n, ks_c128* A, long lda, double* theta, ks_c128* C, long ldc,
            int* sweeps_out /*HOST, may be NULL*/);
/* register-resident DMMA m8n8k4 microbenchmark: achieved FP64 tensor TFLOP/s (roofline denominator) */
int ks_dmma_peak(double* tflops_out /*HOST*/, double* dfma_tflops_out /*HOST, plain DFMA, may be NULL*/);
/* DMMA result latency probe: SM clocks per DMMA of ONE warp per SM sub-partition that keeps 1, 2, 3, 4, 6, 8 independent
 * accumulator tiles in flight (HOST out [6]); the first entry is the dependent-issue latency, the last the issue interval.
 * sm_ghz: the SM clock the times are converted with (bench.py passes the clock it sampled). */
int ks_dmma_latency(double* clk_per_dmma, double sm_ghz);
/* Do the FP64 tensor (DMMA) and the plain FP64 (DFMA) instructions draw on separate issue capacity?  HOST out [4], summed
 * TFLOP/s of register-resident loops: [0] every warp DMMA, [1] every warp DFMA, [2] per SM sub-partition one DMMA warp next
 * to one DFMA warp, [3] every warp interleaves both.  [2], [3] above [0] would mean the roofline denominator of the GEMMs
 * (ks_dmma_peak) is too low; DESIGN.md section 5 records what the B200 measured. */
int ks_fp64_mix_peak(double* tflops4);
#ifdef __cplusplus
}
#endif
#endif /* KSPW_H */
