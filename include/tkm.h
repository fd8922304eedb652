/* tkm.h -- C ABI of libtkm: the B200 (sm_100a) spectral solution-path + exact cross-validation
 * library for kernel machines (smoothed-hinge SVM, kernel logistic regression, kernel quantile
 * regression).  Method: "TorchKM", arxiv/paper_2606_06742; citations below are PAPER.md:<line>
 * of that paper's text, plus the readings G1..G19 of SURVEY.md section 8(c) / DESIGN.md.
 *
 * Conventions
 *   - extern "C"; every call returns a tkm_status (0 = TKM_OK).  tkm_last_error() returns a
 *     thread-local, NUL-terminated description of the last failure on the calling thread.
 *     No exception crosses the boundary.  Process-wide state: that string, the launch counter and a small pinned
 *     read-back buffer (all thread-local); per device, created on first use and kept until the process exits: one
 *     library-owned stream-ordered memory pool that serves EVERY device allocation of the library (temporaries and
 *     handle memory; up to 8 GiB of freed memory is retained; never the device's default pool), the worker threads,
 *     streams and cuSOLVER handles of tkm_spectral_setup_multi, "kernel attributes set" bits, and the 512 KB static
 *     device array of tkm_predict_noalloc.
 *   - [dev]  = pointer to DEVICE memory owned by the caller (e.g. a torch tensor's data_ptr()).
 *     [host] = pointer to HOST memory owned by the caller.  Nothing passed in is retained after
 *     the call returns except where stated (tkm_path keeps a pointer to its tkm_spectral).
 *   - Matrices are row-major with an explicit leading dimension in ELEMENTS.
 *   - Handles (tkm_spectral*, tkm_path*) are owned by the library: free with tkm_*_free.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls that
 *     write [host] outputs synchronise the stream before returning; the others are asynchronous
 *     with respect to the host.
 *   - There is no CPU fallback: without a CUDA device every compute call returns TKM_ECUDA.
 *
 * Column ordering of a path:  c = (t (V+1) + v) L + l, with t the loss variant
 * (quantile level), v the held-out fold (v = V: nothing held out, the final model) and l the
 * index into the lambda grid.  B = T L (V+1) columns.
 */
#ifndef TKM_H
#define TKM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TKM_VERSION_MAJOR 0
#define TKM_VERSION_MINOR 1

typedef enum {
  TKM_OK = 0,
  TKM_EINVAL = 1,    /* bad argument (message says which) */
  TKM_ENOMEM = 2,    /* device or host allocation failed */
  TKM_ECUDA = 3,     /* CUDA runtime error / no device */
  TKM_ESOLVER = 4,   /* cuSOLVER failure or info != 0 */
  TKM_ENOTCONV = 5,  /* warning: some column hit maxit; all outputs are still written */
  TKM_ENOTIMPL = 6
} tkm_status;

typedef enum { TKM_F32 = 0, TKM_F64 = 1 } tkm_dtype;   /* element type of an OUTPUT array (tkm_gram); all inputs and  */
                                                        /* the whole sweep are FP64                                    */

typedef enum {
  TKM_LOSS_HINGE = 0,    /* delta-smoothed hinge */
  TKM_LOSS_LOGISTIC = 1, /* log(1 + exp(-y f)); reading G9 */
  TKM_LOSS_QUANTILE = 2, /* gamma-smoothed check loss; reading G10 */
  TKM_LOSS_DWD = 3       /* distance-weighted discrimination; reading G20:   */
                         /* V(u) = 1 - u (u <= 1/2), 1/(4u) (u > 1/2); smooth, one round           */
} tkm_loss;

typedef struct tkm_spectral tkm_spectral; /* K = U Lam U^T and derived device arrays */
typedef struct tkm_path tkm_path;         /* the fitted columns (a, beta0) of one grid */

/* Options of the loss / smoothing schedule (reading G7: fixed schedule
 * smooth_k = smooth0 * eta^k, k = 0..rounds-1, each round warm-started from the previous one). */
typedef struct {
  double smooth0;     /* delta_0 (hinge) / gamma_0 (quantile); ignored for logistic          */
  double eta;         /* shrink factor, the paper's 0.125                      */
  int32_t rounds;     /* R >= 1 smoothing rounds (forced to 1 for logistic)                   */
  int32_t T;          /* number of quantile levels (0 or 1 => one variant)                    */
  const double* taus; /* [host] T quantile levels in (0,1); NULL unless loss == QUANTILE      */
  int32_t restart;    /* 1: gradient restart of the Nesterov sequence (default), 0: plain     */
  int32_t check_every;/* iterations between host convergence polls; <= 0 => library default   */
  double warm_tol;    /* tolerance of rounds 0..R-2 (warm starts only); <= 0 => same as tol   */
  int32_t profile;    /* 1: time the two contractions of the first iteration after every poll */
                      /* with CUDA events (read with tkm_path_profile); 0: no events;         */
                      /* 2: time EVERY contraction launch and count the column-iterations of  */
                      /* each kernel family on the device (a measurement mode: ~4 events and  */
                      /* two atomics per iteration; not for timed runs)                       */
  int32_t tf32_delta; /* 0: every contraction in FP64 (DMMA).  1: delta form of GEMM-B: zeta = U^T z is kept in FP64  */
                      /* and advanced by zeta += U^T (z - z_old), the increment contracted in 3xTF32 on the tcgen05  */
                      /* tensor cores (its error is relative to the increment, which vanishes at convergence).      */
                      /* 2: also GEMM-A: F+ = Fbar - U Lam da.  The recurrences restart from exact FP64 products on  */
                      /* the first iteration of a round and the last iteration of every batch (check_every, twice  */
                      /* that in wide batches), and only those exact iterations decide convergence.  Same fixed    */
                      /* point and tolerances as 0; DESIGN.md section 12.                                           */
                      /* 3: as 2 with SINGLE-TF32 increment products (operands rounded to TF32, hi parts only: half  */
                      /* the operand bytes, a third of the MMAs).  The increments then carry a relative error of     */
                      /* 2^-11 instead of 2^-21; state, exact restarts and every convergence decision stay FP64, so   */
                      /* the result meets the same tolerances (the trajectory, not the fixed point, is perturbed);    */
                      /* an option beyond the "3xTF32 split" BASELINE.json names -- not the default of bench.py.     */
  double gap_tol;     /* outer control of PAPER.md:220-222 ("shrink delta ... until the KKT conditions of  */
                      /* all SVM models are satisfied"; reading G23).  <= 0: the fixed schedule of `rounds`  */
                      /* levels for every column.  > 0: after round k < rounds-1 a column whose solution     */
                      /* certifies a duality gap of the NON-smoothed problem <= gap_tol (the certificate of   */
                      /* tkm_path_duality_gap) keeps that level's minimiser and leaves the schedule; a warm_tol */
                      /* iterate only screens: the column is first finished to `tol` at that level and tested  */
                      /* again.  `rounds` is the cap: a column that reaches it with a larger gap gets flag 2.  */
  int32_t delta_min_live; /* live columns (all groups) at or below which a delta-form sweep runs all-FP64; <= 0:   */
                      /* the library's cost model of the two contraction kernels (58 at 5 x n = 2000, 8 once U     */
                      /* streams from HBM; never engaged for tiny problems).  Tests set it to exercise the delta   */
                      /* forms on small inputs.                                                                    */
} tkm_loss_opts;

/* Nystrom inputs for tkm_spectral_setup (reading G11). */
typedef struct {
  const double* K_nm;        /* [dev] n x m cross kernel k(x_i, x_landmark_j), FP64            */
  int64_t ld_nm;             /* leading dimensions must be EVEN (16-byte aligned rows), else TKM_EINVAL */
  const double* K_mm;        /* [dev] m x m landmark kernel, FP64                              */
  int64_t ld_mm;
  int64_t m;                 /* number of landmarks                                            */
  const int64_t* landmark_idx; /* [host] m row indices into X, each in [0, n) (kept for tkm_predict) */
} tkm_nystrom;

/* ---- S1  RBF Gram matrix (PAPER.md:69 kernel="rbf"; reading G12) -----------------------------
 * K[i][j] = exp(-||X[i,:] - X2[j,:]||^2 / (2 sigma^2)), FP64 arithmetic, direct differences.
 * X  [dev] n x p FP64 (ldx >= p).  X2 [dev] n2 x p FP64 or NULL: NULL => X2 = X, n2 = n, only
 * the upper-triangular tiles are computed and mirrored, so K is bit-exactly symmetric with an
 * exact unit diagonal.  K [dev] n x n2, out_dt FP64 or FP32 (rounded once from FP64), ldk >= n2.
 * Errors: sigma <= 0, n/p/ld out of range -> TKM_EINVAL.  Asynchronous. */
int tkm_gram(const void* X, int64_t n, int64_t p, int64_t ldx,
             const void* X2, int64_t n2, int64_t ldx2,
             double sigma, tkm_dtype out_dt, void* K, int64_t ldk, void* stream);

/* The same for G <= 8 bandwidths in ONE pass: the squared distances are computed once and every bandwidth
 * costs one exp and one write per entry.  sigmas [host] G values > 0; Ks [host] G [dev] output matrices with
 * the same ldk and out_dt.  Bit-identical to G separate tkm_gram calls.  Asynchronous. */
int tkm_gram_multi(const void* X, int64_t n, int64_t p, int64_t ldx,
                   const void* X2, int64_t n2, int64_t ldx2,
                   const double* sigmas, int32_t G, tkm_dtype out_dt, void* const* Ks, int64_t ldk,
                   void* stream);

/* ---- S2  one-time spectral setup (Alg.1 l.3, 226; readings G11, G16, G19) --------
 * Full kernel (ny == NULL): K [dev] n x n FP64 symmetric (not modified); decomposes in FP64 with
 * cuSOLVER syevd, clamps Lam >= 0, forms u1 = U^T 1, and keeps U Lam (n x r) and U^T (r x n) in
 * FP64 for the two contractions of the sweep.  PRECISION, stated once: the sweep's state, stop test and results
 * are always FP64.  There is no all-FP32 sweep (FP32-accumulated contractions cannot meet the stop test on
 * ill-conditioned columns); the configurations BASELINE.json labels "fp32" run as FP64
 * state + 3xTF32 increments on the tcgen05 tensor cores (tkm_loss_opts.tf32_delta), which meets the FP64
 * parity bar.  r = n.
 * Nystrom (ny != NULL): K is ignored (may be NULL); thin U (n x r, r <= m) from K_nm, K_mm.
 * The handle is shared by every lambda, fold and quantile level.  Synchronises `stream`.
 * Errors: TKM_ESOLVER if cuSOLVER reports info != 0; TKM_ENOMEM. */
int tkm_spectral_setup(const void* K, int64_t n, int64_t ldk, const tkm_nystrom* ny,
                       tkm_spectral** out, void* stream);
/* Nystrom setup straight from the training matrix (n ~ 10^6 rows):
 * X [dev] n x p FP64 (ldx >= p), RBF bandwidth sigma, landmark_idx [host] m row indices into X.  The
 * landmark rows are gathered, K_mm is formed, and K_nm is produced by the Gram kernel and consumed
 * block_rows rows at a time (0 = 32768), so it is never resident: beyond X the peak is one r x n array
 * (Phi^T, overwritten block by block by U^T), the n x r array U Lam and three blocks.  Same handle, same
 * truncations (reading G11) as tkm_spectral_setup with a tkm_nystrom.  Synchronises `stream`. */
int tkm_spectral_setup_nystrom_x(const void* X, int64_t n, int64_t p, int64_t ldx, double sigma,
                                 const int64_t* landmark_idx, int64_t m, int64_t block_rows,
                                 tkm_spectral** out, void* stream);
/* G full-kernel setups (Ks [host]: G [dev] n x n FP64 matrices with the same n, ldk) run concurrently on
 * G internal streams ordered after `stream`; out [host] G slots.  Same results as G separate calls.
 * Returns after all G decompositions have finished. */
int tkm_spectral_setup_multi(const void* const* Ks, int32_t G, int64_t n, int64_t ldk,
                             tkm_spectral** out, void* stream);
void tkm_spectral_free(tkm_spectral* s);
/* n, r, and [host] copies of Lam (r) and u1 (r); either output pointer may be NULL. */
int tkm_spectral_info(const tkm_spectral* s, int64_t* n, int64_t* r, double* lam, double* u1);
/* Copy U (n x r, FP64, row-major, ld = r) to [dev] U_out -- test / diagnostic accessor. */
int tkm_spectral_get_u(const tkm_spectral* s, double* U_out, void* stream);

/* ---- S3-S8  the batched spectral MM sweep (Alg.1 178-224, 226-232) --
 * Fits all B = T L (V+1) columns: for column (t, l, v) the minimiser of
 *   (1/n_c) sum_{j: foldid_j != v} loss_t(y_j, K_j^T alpha + beta0) + lambda_l alpha^T K alpha
 * (eq.(1), 166) at the final smoothing level, by the Nesterov-accelerated
 * majorise-minimise iteration applied through the spectral block inverse (all columns stacked,
 * two contractions with U per iteration).  State is kept in spectral coordinates a = U^T alpha.
 *   y       [dev]  n FP64 (+-1 for HINGE / LOGISTIC / DWD, checked; real for QUANTILE)
 *   lambdas [host] L values > 0          foldid [host] n values in [0, V), every fold non-empty
 *   tol     stop when max(|1^T z|, n_c ||rho||_2 / sqrt(n)) <= tol per column (reading G6)
 *   maxit   per column per round; columns that hit it are flagged and TKM_ENOTCONV is returned (in the delta
 *           forms both decisions -- converged, or out of iterations -- are taken on the exact iterations only,
 *           so a column may run up to 2 check_every - 1 iterations past maxit before it is flagged)
 *   warm    optional path of the same shape on the same spectral handle to start from, or NULL
 * The path keeps a pointer to `s`, which must outlive it.  Synchronises `stream`. */
int tkm_fit_path(const tkm_spectral* s, const void* y, tkm_loss loss, const tkm_loss_opts* opts,
                 const double* lambdas, int32_t L, const int32_t* foldid, int32_t V,
                 double tol, int32_t maxit, const tkm_path* warm, tkm_path** out, void* stream);
/* The same sweep for G <= 8 independent problems that share y, the folds, the loss and the lambda
 * grid -- e.g. the bandwidths of a sigma grid, one spectral handle each (all with the same n, r and
 * sweep precision).  Every iteration is ONE launch per kernel over all groups' live columns, which
 * keeps the device full when each group's batch has become narrow.  Every column reaches the same
 * minimiser as in G separate tkm_fit_path calls to the stop tolerance (tile shapes, hence summation
 * orders, depend on the totals over the groups).  specs [host] G handles; warm [host] G paths or NULL; out [host] G
 * slots, out[g] belongs to specs[g].  The sampled timings of tkm_path_profile are those of the shared
 * launches and are reported on out[0] only. */
int tkm_fit_path_multi(const tkm_spectral* const* specs, int32_t G, const void* y, tkm_loss loss,
                       const tkm_loss_opts* opts, const double* lambdas, int32_t L,
                       const int32_t* foldid, int32_t V, double tol, int32_t maxit,
                       const tkm_path* const* warm, tkm_path** out, void* stream);
void tkm_path_free(tkm_path* p);
/* Shape and per-column diagnostics, all [host], any pointer may be NULL:
 * B, r; iters[B] (total over rounds), kkt[B] (last residual), flags[B] (bit 0 = hit maxit, bit 1 = reached the
 * cap of the smoothing schedule with a duality gap > gap_tol; only with gap_tol > 0),
 * beta0[B]; total_col_iters = sum of iters (the unit of the roofline). */
int tkm_path_info(const tkm_path* p, int32_t* B, int64_t* r, int32_t* iters, double* kkt,
                  int32_t* flags, double* beta0, int64_t* total_col_iters);
/* T, L, V of the grid and n of its spectral handle; any pointer may be NULL. */
int tkm_path_shape(const tkm_path* p, int32_t* T, int32_t* L, int32_t* V, int64_t* n);
/* Smoothing level every column ended on (reading G23): level[B] in [0, rounds), rounds - 1 under the fixed schedule,
 * and smooth[B] = smooth0 eta^level (0 for the smooth losses); both [host], either may be NULL. */
int tkm_path_levels(const tkm_path* p, int32_t* level, double* smooth);
/* Sampled kernel timings of the sweep (only when tkm_loss_opts.profile was 1), all [host] arrays of 4, one
 * entry per kernel family and contraction: [0] FP64 DMMA GEMM-A, [1] FP64 DMMA GEMM-B, [2] tcgen05 3xTF32
 * delta GEMM-A, [3] tcgen05 3xTF32 delta GEMM-B (the contraction launches alone, not the elementwise passes that
 * consume their products).  ms = summed CUDA-event durations of the sampled launches (the
 * first iteration after every compaction -- every slot live -- and, in the delta forms, the exact last
 * iteration of the batch), flops = summed algorithmic flops 2 n r (live columns) of those launches
 * (4 n r per column-iteration over the two contractions), launches = their number.
 * With profile == 2 the three arrays are totals over ALL launches of the sweep and flops counts, per family,
 * 2 n r for every column-iteration that was still unconverged when the launch ran (frozen slots that wait for
 * the next compaction are multiplied but not counted): flops / ms is the time-weighted useful rate. */
int tkm_path_profile(const tkm_path* p, double* ms, double* flops, int64_t* launches);
/* Spectral coordinates of all columns: [dev] a_out, B x r FP64 row-major (ld = r). */
int tkm_path_get_a(const tkm_path* p, double* a_out, void* stream);

/* ---- S9  exact cross-validation scores (readings G14, G15) -------------
 * For every (t, l, v), v < V: decision values f_j = [U (Lam * a_c)]_j + beta0_c on the rows of
 * fold v, cv_loss = mean nominal loss (hinge / deviance / check), cv_err = #{label(f_j) != y_j}
 * (classifiers; -1 for QUANTILE), cv_mean[t][l] = (1/n) sum_v |v| cv_loss[t][l][v],
 * best_l[t] = argmin_l cv_mean[t][l], ties -> the largest lambda.  No refitting.
 *   cv_loss [host] T x L x V doubles, cv_err [host] T x L x V int64 or NULL,
 *   cv_mean [host] T x L, best_l [host] T.   Synchronises `stream`. */
int tkm_exact_cv(const tkm_path* p, const void* y, const int32_t* foldid,
                 double* cv_loss, int64_t* cv_err, double* cv_mean, int32_t* best_l, void* stream);

/* tkm_path_duality_gap: diagnostic of the fixed delta-schedule ("until the KKT conditions of
 * all SVM models are satisfied"; readings G7, G22).  For every column c = (t (V+1) + v) L + l of a hinge or
 * quantile path: primal[c] = (1/n_c) sum over training rows of the NON-smoothed loss + lambda alpha^T K alpha, and
 * gap[c] = primal[c] - dual[c] >= primal[c] - optimum, with the dual point the smoothed solution supplies
 * (theta_j = -L'_delta(y_j f_j)).  One GEMM-A pass over all columns.  y [dev] n, foldid [host] n, primal and
 * gap [host] B.  TKM_EINVAL for the smooth losses (no smoothing, nothing to certify).  Synchronises `stream`. */
int tkm_path_duality_gap(const tkm_path* p, const void* y, const int32_t* foldid, double* primal,
                         double* gap, void* stream);

/* tkm_cv_select: the selection step of tkm_exact_cv on its own (lambda columns sharded
 * over GPUs, the T x L x V loss table gathered before the argmin).  cv_loss [host] T x L x V fold means,
 * fold_sizes [host] V (> 0), lambdas [host] L; writes [host] cv_mean T x L (pooled over folds, weights
 * fold_sizes / n) and best_l T (argmin, ties -> largest lambda, reading G14).  Synchronises `stream`. */
int tkm_cv_select(const double* cv_loss, const double* fold_sizes, const double* lambdas, int32_t T,
                  int32_t L, int32_t V, double* cv_mean, int32_t* best_l, void* stream);

/* Fold sizes of a fold assignment: sizes [host] V doubles (the weights tkm_cv_select expects).  Integer-only,
 * host; TKM_EINVAL if a label is outside [0, V). */
int tkm_fold_sizes(const int32_t* foldid, int64_t n, int32_t V, double* sizes);

/* ---- S10 coefficients and prediction (readings G11, G15) --------------------
 * tkm_path_coef: alpha = U a of column (t, l, v) into [dev] alpha (n FP64; Nystrom: the m landmark
 * weights gamma), and beta0 into [host] *beta0.  Synchronises `stream`. */
int tkm_path_coef(const tkm_path* p, int32_t t, int32_t l, int32_t v, double* alpha, double* beta0,
                  void* stream);
/* tkm_predict: f(x) = sum_i exp(-||x - x_i||^2 / (2 sigma^2)) alpha_i + beta0 with the v = V
 * column of (t, l); the cross-kernel is fused with the contraction and never written.
 *   X_train [dev] n x p FP64 (the training matrix; Nystrom: landmark rows are gathered from it)
 *   X_new   [dev] n_new x p FP64;  f_out [dev] n_new FP64;  label_out [dev] n_new int8 (+1 if
 *   f >= 0 else -1) or NULL.  Asynchronous after an internal coefficient computation. */
int tkm_predict(const tkm_path* p, int32_t t, int32_t l,
                const void* X_train, int64_t ldx, const void* X_new, int64_t n_new, int64_t ldxn,
                int64_t pdim, double sigma, void* f_out, int8_t* label_out, void* stream);

/* tkm_predict_noalloc: tkm_predict for callers that may not allocate (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc).  Same arguments, same two kernels, same result; it calls no
 * cudaMalloc / cudaFree / stream-ordered allocation and no allocating library routine, and it does not synchronise
 * (fully asynchronous on `stream`).  The coefficient vector between the two kernels -- tkm_predict's only device
 * temporary -- lives in a static device array of TKM_PREDICT_NOALLOC_MAX_COEF FP64 (512 KB, held by every GPU
 * that loads the library until the process exits).
 *   Limit: the number of coefficients (training rows n; Nystrom: landmarks m) must not exceed
 *   TKM_PREDICT_NOALLOC_MAX_COEF, else TKM_EINVAL with a message naming the limit (use tkm_predict).
 *   Sharing: every call on one device uses the same array, and it keeps the last call's contents (each call
 *   overwrites all entries it reads, so nothing needs clearing).  Calls that can overlap on the GPU -- different
 *   streams, or graph branches without a dependency -- RACE on it: serialise them. */
#define TKM_PREDICT_NOALLOC_MAX_COEF 65536
int tkm_predict_noalloc(const tkm_path* p, int32_t t, int32_t l,
                        const void* X_train, int64_t ldx, const void* X_new, int64_t n_new, int64_t ldxn,
                        int64_t pdim, double sigma, void* f_out, int8_t* label_out, void* stream);

/* ---- probability calibration on the exact-CV path (G21) ----
 * tkm_cv_decision_values: f_out [dev] n FP64, f_out[j] = held-out decision value of training row j at
 * (t, lambda_l), i.e. from the column that held out fold foldid[j] (no refitting).  foldid [host] n.
 * Synchronises `stream`. */
int tkm_cv_decision_values(const tkm_path* p, int32_t t, int32_t l, const int32_t* foldid, double* f_out,
                           void* stream);
/* tkm_platt_fit: Platt's sigmoid P(y = +1 | f) = 1 / (1 + exp(A f + B)) fitted to scores f [dev] n and labels
 * y [dev] n (+-1) with the targets and the Newton iteration of Lin, Lin & Weng (2007); A, B [host], iters
 * [host] or NULL.  TKM_ENOTCONV if the line search fails (A, B still written).  Synchronises `stream`. */
int tkm_platt_fit(const double* f, const double* y, int64_t n, double* A, double* B, int32_t* iters,
                  void* stream);
/* p_out[i] = 1 / (1 + exp(A f[i] + B)); f, p_out [dev] n.  Asynchronous. */
int tkm_platt_proba(const double* f, int64_t n, double A, double B, double* p_out, void* stream);

/* ---- whole pipeline from HOST buffers (the end-to-end call timed as `e2e` by bench.py) ---------
 * X [host] n x p FP64, y [host] n FP64, sigmas [host] G <= 8 bandwidths; copies X, y to the device,
 * runs S1 and S2 per bandwidth, S3-S8 for all bandwidths together (tkm_fit_path_multi), S9 per
 * bandwidth, and returns, per bandwidth g, the [host] cv tables as in tkm_exact_cv (cv_loss
 * G x T x L x V, cv_err G x T x L x V or NULL, cv_mean G x T x L, best_l G x T) plus the final-model
 * coefficients of the selected lambda of variant 0 (alpha_best G x n doubles or NULL, beta0_best G).
 * Full kernel only.  stage_ms [host] 5 floats or NULL: copy-in, gram, eig, sweep, cv + copy-out (ms). */
int tkm_train_tune_host(const double* X, int64_t n, int64_t p, const double* y, const double* sigmas,
                        int32_t G, tkm_loss loss, const tkm_loss_opts* opts, const double* lambdas,
                        int32_t L, const int32_t* foldid, int32_t V, double tol, int32_t maxit,
                        double* cv_loss, int64_t* cv_err, double* cv_mean,
                        int32_t* best_l, double* alpha_best, double* beta0_best, float* stage_ms,
                        void* stream);

/* ---- helpers ------------------------------------------------------------------------------------
 * tkm_make_folds: integer-only fold assignment (reading G13): SplitMix64(seed) -> Fisher-Yates
 * permutation pi (j = next() mod (i+1), i = n-1..1) -> foldid[pi[i]] = i mod V.  [host] output.
 * Needs 2 <= V <= n. */
int tkm_make_folds(int64_t n, int32_t V, uint64_t seed, int32_t* foldid);
/* Number of kernels launched by this library on the calling thread since the last reset
 * (bench.py's `gpu_launches`). */
int64_t tkm_launch_count(void);
void tkm_launch_count_reset(void);
/* Dense FP64 GEMM probe on the library's own TMA + DMMA kernel (tests):
 * Dt[N][M] = P[N][K] Q[M][K]^T, all [dev] FP64 row-major, 16-byte aligned, with even leading
 * dimensions ldp, ldq >= K and ldd >= M.  Nothing beyond K is read.  Asynchronous. */
int tkm_dgemm_nt(const double* P, int64_t ldp, const double* Q, int64_t ldq, double* Dt, int64_t ldd,
                 int64_t N, int64_t M, int64_t K, void* stream);
/* Roofline calibration of the same kernel: G independent products Dt_g[N][M] = P_g[N][K] Q_g[M][K]^T
 * on library-owned buffers, `iters` back-to-back launches of tile configuration `cfg` (0..7; -1 = the
 * library's own shape-based choice) timed with CUDA events on `stream`; *ms [host] = milliseconds
 * per launch.  Synchronises `stream`. */
int tkm_gemm_probe(int32_t cfg, int32_t G, int32_t N, int32_t M, int32_t K, int32_t iters, float* ms,
                   void* stream);
/* 3xTF32 contraction on the tcgen05 tensor cores (the FP32 variant of the sweep's products), test and
 * calibration entry: Dt[N][M] (FP64, [dev]) = P[N][K] Q[M][K]^T with the FP64 inputs split on the fly into
 * TF32 (hi, lo) pairs and accumulated in FP32 as lo*hi + hi*lo + hi*hi.  cfg is ignored (the CTA-pair kernel has
 * one tile shape: 256 rows x up to 512 slots, stream-K over K).  ms [host] NULL or the milliseconds per launch over
 * `iters` timed launches.
 * Synchronises `stream`. */
int tkm_tf32x3_gemm_nt(const double* P, int64_t ldp, const double* Q, int64_t ldq, double* Dt, int64_t ldd,
                       int64_t N, int64_t M, int64_t K, int32_t cfg, int32_t iters, float* ms, void* stream);
int tkm_version(void);
const char* tkm_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* TKM_H */
