// handles.cuh -- the two opaque handles of the C ABI (include/tkm.h) and internal entry points
// shared between translation units.
#pragma once

#include <vector>

#include "common.cuh"

// K = U Lam U^T and what the sweep derives from it once (data D4/D7).
struct tkm_spectral {
  int64_t n = 0, r = 0;
  int64_t ldr = 0;   // round_up(r, 16): leading dimension of every [.][r] array (zero padded)
  int64_t ldn = 0;   // round_up(n, 16): leading dimension of every [.][n] array (zero padded)
  tkm::DevBuf UL;    // [n][ldr] FP64   U * diag(Lam)   (Q operand of GEMM-A)
  tkm::DevBuf Ut;    // [r][ldn] FP64   U^T             (Q operand of GEMM-B)
  tkm::DevBuf lam;   // [ldr]    FP64   eigenvalues >= 0 (padding 0)
  tkm::DevBuf u1;    // [ldr]    FP64   U^T 1            (padding 0)
  double thin = 0.0; // n - ||u1||^2 for a thin U, exactly 0 for the full kernel (reading G1)
  std::vector<double> h_lam, h_u1;
  // Nystrom (reading G11)
  int64_t m = 0;
  int64_t ldm = 0;
  tkm::DevBuf lmap_t;             // [r][ldm]: gamma = lmap_t^T a  (landmark weights)
  tkm::DevBuf d_landmark_idx;     // [m] int64
  std::vector<int64_t> landmark_idx;
};

// The fitted columns of one grid (data D6).
struct tkm_path {
  const tkm_spectral* spec = nullptr;
  int32_t L = 0, V = 0, T = 1, B = 0;
  tkm_loss loss = TKM_LOSS_HINGE;
  double smooth_final = 0.0;
  std::vector<double> lambdas, taus;
  tkm::DevBuf a;        // [B][ldr] FP64 spectral coordinates, one column of the batch per row
  tkm::DevBuf beta0;    // [B]
  tkm::DevBuf col_lam, col_tau, col_nc;   // [B] per-column lambda, tau, n_c
  tkm::DevBuf col_v;    // [B] int32 held-out fold (V = none)
  tkm::DevBuf col_smooth;   // [B] smoothing level each column ended on (reading G23), unset for the smooth losses
  std::vector<double> h_beta0, h_kkt, h_smooth;
  std::vector<int32_t> h_iters, h_flags, h_level;
  int64_t total_col_iters = 0;
  // sampled CUDA-event timings of the two contractions (tkm_loss_opts.profile)
  // by kernel family and contraction: [0] DMMA GEMM-A, [1] DMMA GEMM-B, [2] tcgen05 A, [3] tcgen05 B
  double prof_ms[4] = {0.0, 0.0, 0.0, 0.0};       // summed CUDA-event durations of the sampled launches
  double prof_flops[4] = {0.0, 0.0, 0.0, 0.0};    // summed 2 n r (live columns) of those launches
  int64_t prof_launches[4] = {0, 0, 0, 0};
};

namespace tkm {
// cv_predict.cu: duality-gap certificate of every column (reading G22) on device arrays, asynchronous
int path_gap_device(const tkm_path* p, const double* y, const int32_t* d_fold, const double* beta0, double smooth,
                    const double* col_smooth, double* d_P, double* d_gap, cudaStream_t st);
// transpose.cu-style helpers living in spectral.cu
int transpose_scale_f64(const double* src, int64_t lds, int64_t rows, int64_t cols, const double* row_scale,
                        double* dst, int64_t ldd, cudaStream_t st);   // dst[c][r] = src[r][c] * row_scale[r]
}  // namespace tkm
