// cv_predict.cu -- S9 exact cross-validation scores and S10 coefficients / prediction.
//
// S9 (readings G14, G15): the masked full-size fit restricted to the training
// rows IS the refit without fold v, so the held-out decision values are f_j = [U (Lam a_c)]_j + b0_c,
// j in fold v -- one more GEMM-A over all columns whose epilogue scores the held-out rows.  Nothing is
// refitted and F never reaches HBM.
// S10: alpha = U a; f(x) = sum_i k(x, x_i) alpha_i + beta0 with the cross-kernel
// fused into the contraction (K_new is never written).
#include <cmath>

#include "gemm_f64.cuh"
#include "handles.cuh"
#include "losses.cuh"

namespace tkm {

struct CvEpi {
  const double* y;
  const int32_t* foldid;
  const double* beta0;     // [B]
  const double* col_tau;   // [B]
  const int32_t* col_v;    // [B]
  int V, loss;
  double* lpart;           // [m blocks][ldpart] partial loss sums over held-out rows
  double* epart;           // [m blocks][ldpart] partial misclassification counts (exact in FP64)
  int64_t ldpart;
  template <class Cfg>
  __device__ __forceinline__ void run(double (&acc)[Cfg::TN][Cfg::TM][2], int n_blk0, int m_blk0, int warp_n,
                                      int warp_m, int lane, int N, int M, int, double* scratch) const {
    constexpr int TN = Cfg::TN, TM = Cfg::TM;
    double ls[TN], es[TN];
#pragma unroll
    for (int i = 0; i < TN; ++i) {
      ls[i] = es[i] = 0.0;
      const int col = n_blk0 + (warp_n * TN + i) * 8 + (lane >> 2);
      if (col >= N) continue;
      const int v = col_v[col];
      if (v >= V) continue;   // final-model column: nothing held out
      const double b0 = beta0[col], tau = col_tau[col];
#pragma unroll
      for (int j = 0; j < TM; ++j)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int m = m_blk0 + (warp_m * TM + j) * 8 + 2 * (lane & 3) + e;
          if (m < M && foldid[m] == v) {
            const double f = acc[i][j][e] + b0, yy = y[m];
            ls[i] += nominal_loss_dev(loss, yy, f, tau);
            const double lab = (f >= 0.0) ? 1.0 : -1.0;   // label(0) = +1 (G15)
            es[i] += (lab != yy) ? 1.0 : 0.0;
          }
        }
    }
    double tot;
    if (cta_row_reduce<Cfg>(ls, warp_n, warp_m, lane, scratch, tot)) {
      const int col = n_blk0 + (int)threadIdx.x;
      if (col < N) lpart[(int64_t)gemm_m_block() * ldpart + col] = tot;
    }
    if (cta_row_reduce<Cfg>(es, warp_n, warp_m, lane, scratch, tot)) {
      const int col = n_blk0 + (int)threadIdx.x;
      if (col < N) epart[(int64_t)gemm_m_block() * ldpart + col] = tot;
    }
  }
};

// Duality-gap diagnostic (reading G22): same GEMM-A pass, but over the TRAINING rows of every
// column: partial sums of the nominal loss and of the dual variable times y, d_j = -y_j psi_delta(y_j, f_j)
// (hinge: theta_j in [0, 1]; check loss: s_j y_j with s_j in [tau - 1, tau]).
struct GapEpi {
  const double* y;
  const int32_t* foldid;
  const double* beta0;
  const double* col_tau;
  const int32_t* col_v;
  int loss;
  double smooth;             // smoothing level of every column, unless
  const double* col_smooth;  // [B] per-column levels (reading G23: columns may end on different levels), or NULL
  double* lpart;   // [m blocks][ldpart] sum of the nominal loss over training rows
  double* dpart;   // [m blocks][ldpart] sum of d_j over training rows
  int64_t ldpart;
  template <class Cfg>
  __device__ __forceinline__ void run(double (&acc)[Cfg::TN][Cfg::TM][2], int n_blk0, int m_blk0, int warp_n,
                                      int warp_m, int lane, int N, int M, int, double* scratch) const {
    constexpr int TN = Cfg::TN, TM = Cfg::TM;
    double ls[TN], ds[TN];
#pragma unroll
    for (int i = 0; i < TN; ++i) {
      ls[i] = ds[i] = 0.0;
      const int col = n_blk0 + (warp_n * TN + i) * 8 + (lane >> 2);
      if (col >= N) continue;
      const int v = col_v[col];
      const double b0 = beta0[col], tau = col_tau[col];
      const double sm = col_smooth ? col_smooth[col] : smooth;
#pragma unroll
      for (int j = 0; j < TM; ++j)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int m = m_blk0 + (warp_m * TM + j) * 8 + 2 * (lane & 3) + e;
          if (m < M && foldid[m] != v) {
            const double f = acc[i][j][e] + b0, yy = y[m];
            ls[i] += nominal_loss_dev(loss, yy, f, tau);
            ds[i] -= yy * psi_dev(loss, yy, f, sm, tau);
          }
        }
    }
    double tot;
    if (cta_row_reduce<Cfg>(ls, warp_n, warp_m, lane, scratch, tot)) {
      const int col = n_blk0 + (int)threadIdx.x;
      if (col < N) lpart[(int64_t)gemm_m_block() * ldpart + col] = tot;
    }
    if (cta_row_reduce<Cfg>(ds, warp_n, warp_m, lane, scratch, tot)) {
      const int col = n_blk0 + (int)threadIdx.x;
      if (col < N) dpart[(int64_t)gemm_m_block() * ldpart + col] = tot;
    }
  }
};

// one CTA per column: P = sum loss / n_c + lam a^T Lam a,  D = sum d / n_c - lam a^T Lam a  (fixed summation order)
__global__ void __launch_bounds__(256) gap_finalize_kernel(const double* __restrict__ lpart, const double* __restrict__ dpart,
                                                           int64_t ldpart, int nblk, const double* __restrict__ a, int64_t lda,
                                                           const double* __restrict__ lam_spec, int r,
                                                           const double* __restrict__ col_lam, const double* __restrict__ col_nc,
                                                           double* __restrict__ primal, double* __restrict__ gap) {
  __shared__ double red[8];
  const int c = blockIdx.x;
  double q = 0.0;
  for (int i = threadIdx.x; i < r; i += 256) {
    const double ai = a[(int64_t)c * lda + i];
    q += lam_spec[i] * ai * ai;
  }
  q = warp_sum(q);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = q;
  __syncthreads();
  if (threadIdx.x == 0) {
    double quad = 0.0, ls = 0.0, ds = 0.0;
    for (int w = 0; w < 8; ++w) quad += red[w];
    for (int b = 0; b < nblk; ++b) {
      ls += lpart[(int64_t)b * ldpart + c];
      ds += dpart[(int64_t)b * ldpart + c];
    }
    const double P = ls / col_nc[c] + col_lam[c] * quad, D = ds / col_nc[c] - col_lam[c] * quad;
    primal[c] = P;
    gap[c] = P - D;
  }
}

// one thread per (t, l, v): sum the per-block partials in fixed order, normalise by the fold size
__global__ void cv_finalize_kernel(const double* __restrict__ lpart, const double* __restrict__ epart,
                                   int64_t ldpart, int nblk, int T, int L, int V, const double* __restrict__ fsize,
                                   int classifier, double* __restrict__ cv_loss, long long* __restrict__ cv_err) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= T * L * V) return;
  const int v = idx % V, l = (idx / V) % L, t = idx / (V * L);
  const int col = (t * (V + 1) + v) * L + l;
  double ls = 0.0, es = 0.0;
  for (int b = 0; b < nblk; ++b) {
    ls += lpart[(int64_t)b * ldpart + col];
    es += epart[(int64_t)b * ldpart + col];
  }
  cv_loss[idx] = ls / fsize[v];
  cv_err[idx] = classifier ? (long long)(es + 0.5) : -1LL;
}

// one thread per t: pooled mean and argmin with ties -> largest lambda (G14)
__global__ void cv_select_kernel(const double* __restrict__ cv_loss, int T, int L, int V,
                                 const double* __restrict__ fsize, double n, const double* __restrict__ lambdas,
                                 double* __restrict__ cv_mean, int* __restrict__ best_l) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= T) return;
  double best = INFINITY;
  int bl = 0;
  for (int l = 0; l < L; ++l) {
    double m = 0.0;
    for (int v = 0; v < V; ++v) m += fsize[v] * cv_loss[((int64_t)t * L + l) * V + v];
    m /= n;
    cv_mean[t * L + l] = m;
    if (m < best || (m == best && lambdas[l] > lambdas[bl])) {
      best = m;
      bl = l;
    }
  }
  best_l[t] = bl;
}

// out[i] = sum_j Mt[j][i] a[j], i < cols (alpha = U a from U^T; gamma = lmap a from lmap^T).  One CTA per 32
// outputs: 8 row lanes x 32 columns walk the rows with coalesced 256-byte reads and are summed in a fixed
// order (deterministic); rows / 8 dependent loads per thread instead of rows.
__global__ void __launch_bounds__(256) tmatvec_kernel(const double* __restrict__ Mt, int64_t ld, int rows, int cols,
                                                      const double* __restrict__ a, double* __restrict__ out) {
  __shared__ double part[8][33];
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  const int i = blockIdx.x * 32 + tx;
  double s = 0.0;
  if (i < cols)
    for (int j = ty; j < rows; j += 8) s = fma(Mt[(int64_t)j * ld + i], a[j], s);
  part[ty][tx] = s;
  __syncthreads();
  if (ty == 0 && i < cols) {
    double t = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) t += part[k][tx];
    out[i] = t;
  }
}

// f(x_q) = sum_i exp(-||x_q - x_i||^2 / (2 sigma^2)) alpha_i + beta0, PQ new points per CTA
constexpr int PQ = 8;     // new points per CTA
constexpr int PCH = 64;   // feature chunk held in shared memory
__global__ void __launch_bounds__(128)
    predict_kernel(const double* __restrict__ Xtr, int64_t ldx, const int64_t* __restrict__ row_idx, int ntr,
                   const double* __restrict__ Xnew, int64_t ldxn, int n_new, int p, double neg_inv_2s2,
                   const double* __restrict__ alpha, const double* __restrict__ beta0_ptr, double* __restrict__ f_out,
                   int8_t* __restrict__ label_out) {
  __shared__ double xq[PQ][PCH];
  __shared__ double red[32];
  const int q0 = blockIdx.x * PQ;
  double facc[PQ];
#pragma unroll
  for (int q = 0; q < PQ; ++q) facc[q] = 0.0;
  for (int i0 = 0; i0 < ntr; i0 += blockDim.x) {
    const int i = i0 + threadIdx.x;
    const double* xi = nullptr;
    if (i < ntr) xi = Xtr + (row_idx ? row_idx[i] : (int64_t)i) * ldx;
    double d2[PQ];
#pragma unroll
    for (int q = 0; q < PQ; ++q) d2[q] = 0.0;
    for (int k0 = 0; k0 < p; k0 += PCH) {
      __syncthreads();
      for (int id = threadIdx.x; id < PQ * PCH; id += blockDim.x) {
        const int q = id / PCH, k = id % PCH;
        xq[q][k] = (q0 + q < n_new && k0 + k < p) ? Xnew[(int64_t)(q0 + q) * ldxn + k0 + k] : 0.0;
      }
      __syncthreads();
      if (xi) {
        const int kend = min(PCH, p - k0);
        for (int k = 0; k < kend; ++k) {
          const double x = xi[k0 + k];
#pragma unroll
          for (int q = 0; q < PQ; ++q) {
            const double d = xq[q][k] - x;
            d2[q] = fma(d, d, d2[q]);
          }
        }
      }
    }
    if (xi) {
      const double al = alpha[i];
#pragma unroll
      for (int q = 0; q < PQ; ++q) facc[q] += exp(d2[q] * neg_inv_2s2) * al;
    }
  }
  const double b0 = *beta0_ptr;
#pragma unroll
  for (int q = 0; q < PQ; ++q) {
    const double f = block_sum(facc[q], red) + b0;
    if (threadIdx.x == 0 && q0 + q < n_new) {
      f_out[q0 + q] = f;
      if (label_out) label_out[q0 + q] = (f >= 0.0) ? (int8_t)1 : (int8_t)-1;
    }
  }
}

static int coef_device(const tkm_path* p, int col, double* out, cudaStream_t st) {
  const tkm_spectral* s = p->spec;
  const double* a = p->a.as<double>() + (int64_t)col * s->ldr;
  if (s->m > 0) {
    tmatvec_kernel<<<(unsigned)ceil_div(s->m, 32), 256, 0, st>>>(s->lmap_t.as<double>(), s->ldm, (int)s->r, (int)s->m, a, out);
  } else {
    tmatvec_kernel<<<(unsigned)ceil_div(s->n, 32), 256, 0, st>>>(s->Ut.as<double>(), s->ldn, (int)s->r, (int)s->n, a, out);
  }
  TKM_LAUNCH_CHECK();
  return TKM_OK;
}

// Gap certificate of every column of `p` at the coefficients (p->a, beta0) -- beta0 [dev] B, d_fold [dev] n --
// for the level `smooth` (col_smooth == NULL) or per-column levels: primal and gap [dev] B.  Asynchronous;
// the partial-sum scratch is stream-ordered.  Used by tkm_path_duality_gap and by the sweep's outer control.
int path_gap_device(const tkm_path* p, const double* y, const int32_t* d_fold, const double* beta0, double smooth,
                    const double* col_smooth, double* d_P, double* d_gap, cudaStream_t st) {
  const tkm_spectral* s = p->spec;
  const int64_t n = s->n, r = s->r;
  const int B = p->B;
  const int nblk = (int)ceil_div(n, gemm_f64_choose(&B, 1, (int)n, (int)r).BM);
  const int64_t ldpart = round_up(B, 16);
  DevBuf lpart, dpart;
  TKM_TRY(lpart.alloc((size_t)nblk * ldpart * sizeof(double), true, st, true));
  TKM_TRY(dpart.alloc((size_t)nblk * ldpart * sizeof(double), true, st, true));
  GapEpi epi{y, d_fold, beta0, p->col_tau.as<double>(), p->col_v.as<int32_t>(), (int)p->loss, smooth, col_smooth,
             lpart.as<double>(), dpart.as<double>(), ldpart};
  TKM_TRY(gemm_f64_once(p->a.as<double>(), s->ldr, s->UL.as<double>(), s->ldr, B, (int)n, (int)r, epi, st));
  gap_finalize_kernel<<<(unsigned)B, 256, 0, st>>>(lpart.as<double>(), dpart.as<double>(), ldpart, nblk, p->a.as<double>(),
                                                   s->ldr, s->lam.as<double>(), (int)r, p->col_lam.as<double>(),
                                                   p->col_nc.as<double>(), d_P, d_gap);
  TKM_LAUNCH_CHECK();
  return TKM_OK;
}

}  // namespace tkm

using namespace tkm;

extern "C" int tkm_exact_cv(const tkm_path* p, const void* y, const int32_t* foldid, double* cv_loss,
                            int64_t* cv_err, double* cv_mean, int32_t* best_l, void* stream) {
  tkm::NvtxRange nvtx_range("tkm_exact_cv");
  if (!p || !y || !foldid || !cv_loss || !cv_mean || !best_l) return set_error(TKM_EINVAL, "tkm_exact_cv: NULL argument");
  TKM_TRY(device_check());
  cudaStream_t st = (cudaStream_t)stream;
  const tkm_spectral* s = p->spec;
  const int64_t n = s->n, r = s->r;
  const int B = p->B, T = p->T, L = p->L, V = p->V;
  std::vector<double> fsize(V, 0.0);
  for (int64_t j = 0; j < n; ++j) {
    if (foldid[j] < 0 || foldid[j] >= V) return set_error(TKM_EINVAL, "tkm_exact_cv: foldid out of range");
    fsize[foldid[j]] += 1.0;
  }
  const int nblk = (int)ceil_div(n, gemm_f64_choose(&B, 1, (int)n, (int)r).BM);
  const int64_t ldpart = round_up(B, 16);
  const int nout = T * L * V;
  DevBuf lpart, epart, d_fold, d_fsize, d_lam, d_loss, d_err, d_mean, d_best;
  TKM_TRY(lpart.alloc((size_t)nblk * ldpart * sizeof(double), true, st));
  TKM_TRY(epart.alloc((size_t)nblk * ldpart * sizeof(double), true, st));
  TKM_TRY(d_fold.alloc((size_t)n * sizeof(int32_t), false, st));
  TKM_TRY(d_fsize.alloc((size_t)V * sizeof(double), false, st));
  TKM_TRY(d_lam.alloc((size_t)L * sizeof(double), false, st));
  TKM_TRY(d_loss.alloc((size_t)nout * sizeof(double), false, st));
  TKM_TRY(d_err.alloc((size_t)nout * sizeof(long long), false, st));
  TKM_TRY(d_mean.alloc((size_t)T * L * sizeof(double), false, st));
  TKM_TRY(d_best.alloc((size_t)T * sizeof(int), false, st));
  TKM_CUDA(cudaMemcpyAsync(d_fold.p, foldid, n * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  TKM_CUDA(cudaMemcpyAsync(d_fsize.p, fsize.data(), V * sizeof(double), cudaMemcpyHostToDevice, st));
  TKM_CUDA(cudaMemcpyAsync(d_lam.p, p->lambdas.data(), L * sizeof(double), cudaMemcpyHostToDevice, st));
  CvEpi epi{(const double*)y, d_fold.as<int32_t>(), p->beta0.as<double>(), p->col_tau.as<double>(),
            p->col_v.as<int32_t>(), V, (int)p->loss, lpart.as<double>(), epart.as<double>(), ldpart};
  TKM_TRY(gemm_f64_once(p->a.as<double>(), s->ldr, s->UL.as<double>(), s->ldr, B, (int)n, (int)r, epi, st));
  cv_finalize_kernel<<<(unsigned)ceil_div(nout, 128), 128, 0, st>>>(
      lpart.as<double>(), epart.as<double>(), ldpart, nblk, T, L, V, d_fsize.as<double>(),
      p->loss != TKM_LOSS_QUANTILE ? 1 : 0, d_loss.as<double>(), d_err.as<long long>());
  TKM_LAUNCH_CHECK();
  cv_select_kernel<<<(unsigned)ceil_div(T, 32), 32, 0, st>>>(d_loss.as<double>(), T, L, V, d_fsize.as<double>(),
                                                            (double)n, d_lam.as<double>(), d_mean.as<double>(),
                                                            d_best.as<int>());
  TKM_LAUNCH_CHECK();
  TKM_CUDA(cudaMemcpyAsync(cv_loss, d_loss.p, nout * sizeof(double), cudaMemcpyDeviceToHost, st));
  if (cv_err) TKM_CUDA(cudaMemcpyAsync(cv_err, d_err.p, nout * sizeof(long long), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaMemcpyAsync(cv_mean, d_mean.p, T * L * sizeof(double), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaMemcpyAsync(best_l, d_best.p, T * sizeof(int), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaStreamSynchronize(st));
  return TKM_OK;
}

extern "C" int tkm_path_duality_gap(const tkm_path* p, const void* y, const int32_t* foldid, double* primal,
                                    double* gap, void* stream) {
  if (!p || !y || !foldid || !primal || !gap) return set_error(TKM_EINVAL, "tkm_path_duality_gap: NULL argument");
  if (p->loss != TKM_LOSS_HINGE && p->loss != TKM_LOSS_QUANTILE)
    return set_error(TKM_EINVAL, "tkm_path_duality_gap: defined for the smoothed losses (hinge, quantile) only");
  TKM_TRY(device_check());
  cudaStream_t st = (cudaStream_t)stream;
  const tkm_spectral* s = p->spec;
  const int64_t n = s->n;
  const int B = p->B;
  for (int64_t j = 0; j < n; ++j)
    if (foldid[j] < 0 || foldid[j] >= p->V) return set_error(TKM_EINVAL, "tkm_path_duality_gap: foldid out of range");
  DevBuf d_fold, d_P, d_gap;
  TKM_TRY(d_fold.alloc((size_t)n * sizeof(int32_t), false, st));
  TKM_TRY(d_P.alloc((size_t)B * sizeof(double), false, st));
  TKM_TRY(d_gap.alloc((size_t)B * sizeof(double), false, st));
  TKM_CUDA(cudaMemcpyAsync(d_fold.p, foldid, n * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  // every column at the level it ended on (all the same under the fixed schedule)
  TKM_TRY(path_gap_device(p, (const double*)y, d_fold.as<int32_t>(), p->beta0.as<double>(), p->smooth_final,
                          p->col_smooth.p ? p->col_smooth.as<double>() : nullptr, d_P.as<double>(), d_gap.as<double>(), st));
  TKM_CUDA(cudaMemcpyAsync(primal, d_P.p, (size_t)B * sizeof(double), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaMemcpyAsync(gap, d_gap.p, (size_t)B * sizeof(double), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaStreamSynchronize(st));
  return TKM_OK;
}

// Pooled mean and selected lambda from a (gathered) fold-loss table: the last step of S9 on its own, for a
// lambda grid whose columns were fitted on several GPUs.  All arguments [host].
extern "C" int tkm_cv_select(const double* cv_loss, const double* fold_sizes, const double* lambdas, int32_t T,
                             int32_t L, int32_t V, double* cv_mean, int32_t* best_l, void* stream) {
  if (!cv_loss || !fold_sizes || !lambdas || !cv_mean || !best_l || T < 1 || L < 1 || V < 1)
    return set_error(TKM_EINVAL, "tkm_cv_select: bad arguments");
  TKM_TRY(device_check());
  cudaStream_t st = (cudaStream_t)stream;
  double n = 0.0;
  for (int v = 0; v < V; ++v) {
    if (!(fold_sizes[v] > 0.0)) return set_error(TKM_EINVAL, "tkm_cv_select: empty fold");
    n += fold_sizes[v];
  }
  const size_t nout = (size_t)T * L * V;
  DevBuf d_loss, d_fsize, d_lam, d_mean, d_best;
  TKM_TRY(d_loss.alloc(nout * sizeof(double), false, st));
  TKM_TRY(d_fsize.alloc((size_t)V * sizeof(double), false, st));
  TKM_TRY(d_lam.alloc((size_t)L * sizeof(double), false, st));
  TKM_TRY(d_mean.alloc((size_t)T * L * sizeof(double), false, st));
  TKM_TRY(d_best.alloc((size_t)T * sizeof(int), false, st));
  TKM_CUDA(cudaMemcpyAsync(d_loss.p, cv_loss, nout * sizeof(double), cudaMemcpyHostToDevice, st));
  TKM_CUDA(cudaMemcpyAsync(d_fsize.p, fold_sizes, V * sizeof(double), cudaMemcpyHostToDevice, st));
  TKM_CUDA(cudaMemcpyAsync(d_lam.p, lambdas, L * sizeof(double), cudaMemcpyHostToDevice, st));
  cv_select_kernel<<<(unsigned)ceil_div(T, 32), 32, 0, st>>>(d_loss.as<double>(), T, L, V, d_fsize.as<double>(), n,
                                                            d_lam.as<double>(), d_mean.as<double>(), d_best.as<int>());
  TKM_LAUNCH_CHECK();
  TKM_CUDA(cudaMemcpyAsync(cv_mean, d_mean.p, (size_t)T * L * sizeof(double), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaMemcpyAsync(best_l, d_best.p, (size_t)T * sizeof(int), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaStreamSynchronize(st));
  return TKM_OK;
}

extern "C" int tkm_path_coef(const tkm_path* p, int32_t t, int32_t l, int32_t v, double* alpha, double* beta0,
                             void* stream) {
  if (!p || !alpha) return set_error(TKM_EINVAL, "tkm_path_coef: NULL argument");
  if (t < 0 || t >= p->T || l < 0 || l >= p->L || v < 0 || v > p->V)
    return set_error(TKM_EINVAL, "tkm_path_coef: (t, l, v) out of range");
  TKM_TRY(device_check());
  const int col = (t * (p->V + 1) + v) * p->L + l;
  TKM_TRY(coef_device(p, col, alpha, (cudaStream_t)stream));
  if (beta0) *beta0 = p->h_beta0[col];
  TKM_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
  return TKM_OK;
}

extern "C" int tkm_predict(const tkm_path* p, int32_t t, int32_t l, const void* X_train, int64_t ldx,
                           const void* X_new, int64_t n_new, int64_t ldxn, int64_t pdim, double sigma,
                           void* f_out, int8_t* label_out, void* stream) {
  tkm::NvtxRange nvtx_range("tkm_predict");
  if (!p || !X_train || !X_new || !f_out) return set_error(TKM_EINVAL, "tkm_predict: NULL argument");
  if (t < 0 || t >= p->T || l < 0 || l >= p->L) return set_error(TKM_EINVAL, "tkm_predict: (t, l) out of range");
  if (n_new <= 0 || pdim <= 0 || ldx < pdim || ldxn < pdim || !(sigma > 0.0))
    return set_error(TKM_EINVAL, "tkm_predict: bad shape or sigma");
  TKM_TRY(device_check());
  cudaStream_t st = (cudaStream_t)stream;
  const tkm_spectral* s = p->spec;
  const int col = (t * (p->V + 1) + p->V) * p->L + l;
  const int64_t ncoef = s->m > 0 ? s->m : s->n;
  DevBuf coef;
  TKM_TRY(coef.alloc((size_t)ncoef * sizeof(double), false, st));
  TKM_TRY(coef_device(p, col, coef.as<double>(), st));
  predict_kernel<<<(unsigned)ceil_div(n_new, PQ), 128, 0, st>>>(
      (const double*)X_train, ldx, s->m > 0 ? s->d_landmark_idx.as<int64_t>() : nullptr, (int)ncoef,
      (const double*)X_new, ldxn, (int)n_new, (int)pdim, -1.0 / (2.0 * sigma * sigma), coef.as<double>(),
      p->beta0.as<double>() + col, (double*)f_out, label_out);
  TKM_LAUNCH_CHECK();
  TKM_CUDA(cudaStreamSynchronize(st));   // `coef` is freed on return
  return TKM_OK;
}

// ---- tkm_predict_noalloc: the serving call for callers that may not allocate -------------------------------
// Same two kernels as tkm_predict (tmatvec_kernel: alpha = U a of the selected column; predict_kernel: the fused
// cross-kernel contraction); the coefficient vector `alpha` between them -- tkm_predict's only device temporary --
// lives in a file-scope device array instead of a cudaMalloc'ed buffer.  Every device that loads the library
// holds these 512 KB until the process exits.
namespace tkm {
static __device__ __align__(256) double g_predict_coef[TKM_PREDICT_NOALLOC_MAX_COEF];

// In host code `g_predict_coef` is the host-side shadow of the symbol, not a device address: the kernels get the
// address cudaGetSymbolAddress returns for the CURRENT device, looked up once per device (no allocation: the array
// is part of the loaded module) and cached.
static int predict_coef_scratch(double** out) {
  static double* addr[64] = {};
  static std::atomic<unsigned long long> have{0};
  int dev = -1;
  TKM_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return set_error(TKM_EINVAL, "tkm_predict_noalloc: device ordinal %d outside 0..63", dev);
  const unsigned long long bit = 1ull << dev;
  if (!(have.load(std::memory_order_acquire) & bit)) {
    double* ptr = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g_predict_coef);
    if (e != cudaSuccess || !ptr)
      return set_error(TKM_ECUDA, "tkm_predict_noalloc: cudaGetSymbolAddress failed on device %d: %s", dev,
                       cudaGetErrorString(e));
    addr[dev] = ptr;   // racing first calls on one device store the same address
    have.fetch_or(bit, std::memory_order_release);
  }
  *out = addr[dev];
  return TKM_OK;
}
}  // namespace tkm

extern "C" int tkm_predict_noalloc(const tkm_path* p, int32_t t, int32_t l, const void* X_train, int64_t ldx,
                                   const void* X_new, int64_t n_new, int64_t ldxn, int64_t pdim, double sigma,
                                   void* f_out, int8_t* label_out, void* stream) {
  if (!p || !X_train || !X_new || !f_out) return set_error(TKM_EINVAL, "tkm_predict_noalloc: NULL argument");
  if (t < 0 || t >= p->T || l < 0 || l >= p->L) return set_error(TKM_EINVAL, "tkm_predict_noalloc: (t, l) out of range");
  if (n_new <= 0 || pdim <= 0 || ldx < pdim || ldxn < pdim || !(sigma > 0.0))
    return set_error(TKM_EINVAL, "tkm_predict_noalloc: bad shape or sigma");
  const tkm_spectral* s = p->spec;
  const int64_t ncoef = s->m > 0 ? s->m : s->n;
  if (ncoef > TKM_PREDICT_NOALLOC_MAX_COEF)
    return set_error(TKM_EINVAL,
                     "tkm_predict_noalloc: %lld coefficients (training rows, or Nystrom landmarks) exceed the static "
                     "scratch of TKM_PREDICT_NOALLOC_MAX_COEF = %d; use tkm_predict",
                     (long long)ncoef, (int)TKM_PREDICT_NOALLOC_MAX_COEF);
  if (n_new > (int64_t)PQ * 2147483647LL) return set_error(TKM_EINVAL, "tkm_predict_noalloc: n_new too large");
  TKM_TRY(device_check());
  cudaStream_t st = (cudaStream_t)stream;
  double* coef = nullptr;
  TKM_TRY(predict_coef_scratch(&coef));
  const int col = (t * (p->V + 1) + p->V) * p->L + l;
  // tmatvec_kernel writes all `ncoef` entries predict_kernel reads: nothing of the previous call's contents is used
  TKM_TRY(coef_device(p, col, coef, st));
  predict_kernel<<<(unsigned)ceil_div(n_new, PQ), 128, 0, st>>>(
      (const double*)X_train, ldx, s->m > 0 ? s->d_landmark_idx.as<int64_t>() : nullptr, (int)ncoef,
      (const double*)X_new, ldxn, (int)n_new, (int)pdim, -1.0 / (2.0 * sigma * sigma), coef,
      p->beta0.as<double>() + col, (double*)f_out, label_out);
  TKM_LAUNCH_CHECK();
  return TKM_OK;   // asynchronous: nothing to free, so no synchronisation
}
