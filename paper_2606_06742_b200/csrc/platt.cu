// platt.cu -- probability calibration on top of the exact-CV path (PAPER.md:49, 73-74, 79,
// 250-256; reading G21).
//
//   tkm_cv_decision_values : held-out decision value of every training row at one (t, lambda): row j is scored
//                            by the column that held out fold foldid[j] -- one GEMM-A over
//                            the V columns of (t, l) whose epilogue keeps only the held-out rows.
//   tkm_platt_fit          : Platt's sigmoid p = 1/(1 + exp(A f + B)) by the Newton iteration with backtracking
//                            of Lin, Lin & Weng (2007), whole fit in ONE single-CTA kernel (every sum in a fixed
//                            order => deterministic); the only host work is reading A and B back.
//   tkm_platt_proba        : p_i for new decision values.
#include <cmath>

#include "gemm_f64.cuh"
#include "handles.cuh"

namespace tkm {

// GEMM-A epilogue: f_out[m] = acc + beta0 for the rows m of the fold this column held out.
struct HeldOutEpi {
  const int32_t* foldid;   // [n]
  const double* beta0;     // [B] by column
  int col0, col_stride;    // column of slot v = col0 + v * col_stride
  double* f_out;           // [n]
  template <class Cfg>
  __device__ __forceinline__ void run(double (&acc)[Cfg::TN][Cfg::TM][2], int n_blk0, int m_blk0, int warp_n,
                                      int warp_m, int lane, int N, int M, int, double*) const {
#pragma unroll
    for (int i = 0; i < Cfg::TN; ++i) {
      const int v = n_blk0 + (warp_n * Cfg::TN + i) * 8 + (lane >> 2);
      if (v >= N) continue;
      const double b0 = beta0[col0 + v * col_stride];
#pragma unroll
      for (int j = 0; j < Cfg::TM; ++j)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int m = m_blk0 + (warp_m * Cfg::TM + j) * 8 + 2 * (lane & 3) + e;
          if (m < M && foldid[m] == v) f_out[m] = acc[i][j][e] + b0;
        }
    }
  }
};

// ---- block-wide sums of K values (1024 threads), fixed order ------------------------------------------
template <int K>
__device__ __forceinline__ void block_sum_k(double (&v)[K], double (*red)[32]) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < K; ++k) v[k] = warp_sum(v[k]);
  __syncthreads();
  if (lane == 0)
#pragma unroll
    for (int k = 0; k < K; ++k) red[k][w] = v[k];
  __syncthreads();
#pragma unroll
  for (int k = 0; k < K; ++k) {
    double t = red[k][lane];   // 32 warps
    v[k] = warp_sum(t);
  }
}

__device__ __forceinline__ double platt_term(double t, double s) {   // t s + log(1 + e^-s) or (t-1) s + log(1 + e^s)
  return (s >= 0.0 ? t * s : (t - 1.0) * s) + log1p(exp(-fabs(s)));
}

// out[0] = A, out[1] = B, out[2] = Newton iterations used, out[3] = 1 if the line search failed
__global__ void __launch_bounds__(1024) platt_fit_kernel(const double* __restrict__ f, const double* __restrict__ y,
                                                         int n, int maxit, double* __restrict__ out) {
  __shared__ double red[5][32];
  const int tid = threadIdx.x;
  double c[1] = {0.0};
  for (int i = tid; i < n; i += 1024) c[0] += (y[i] > 0.0) ? 1.0 : 0.0;
  block_sum_k<1>(c, red);
  const double n_pos = c[0], n_neg = (double)n - c[0];
  const double t_pos = (n_pos + 1.0) / (n_pos + 2.0), t_neg = 1.0 / (n_neg + 2.0);
  double A = 0.0, B = log((n_neg + 1.0) / (n_pos + 1.0));
  double o0[1] = {0.0};
  for (int i = tid; i < n; i += 1024) o0[0] += platt_term(y[i] > 0.0 ? t_pos : t_neg, A * f[i] + B);
  block_sum_k<1>(o0, red);
  double fval = o0[0];
  int it = 0, failed = 0;
  for (; it < maxit; ++it) {
    double s5[5] = {0.0, 0.0, 0.0, 0.0, 0.0};   // h11, h22, h21, g1, g2
    for (int i = tid; i < n; i += 1024) {
      const double fi = f[i], s = A * fi + B, e = exp(-fabs(s));
      const double p = (s >= 0.0) ? e / (1.0 + e) : 1.0 / (1.0 + e);
      const double d2 = p * (1.0 - p), d1 = (y[i] > 0.0 ? t_pos : t_neg) - p;
      s5[0] += fi * fi * d2;
      s5[1] += d2;
      s5[2] += fi * d2;
      s5[3] += fi * d1;
      s5[4] += d1;
    }
    block_sum_k<5>(s5, red);
    const double h11 = 1e-12 + s5[0], h22 = 1e-12 + s5[1], h21 = s5[2], g1 = s5[3], g2 = s5[4];
    if (fabs(g1) < 1e-5 && fabs(g2) < 1e-5) break;
    const double det = h11 * h22 - h21 * h21;
    const double dA = -(h22 * g1 - h21 * g2) / det, dB = -(-h21 * g1 + h11 * g2) / det;
    const double gd = g1 * dA + g2 * dB;
    double step = 1.0;
    bool ok = false;
    while (step >= 1e-10) {
      const double nA = A + step * dA, nB = B + step * dB;
      double o1[1] = {0.0};
      for (int i = tid; i < n; i += 1024) o1[0] += platt_term(y[i] > 0.0 ? t_pos : t_neg, nA * f[i] + nB);
      block_sum_k<1>(o1, red);
      if (o1[0] < fval + 1e-4 * step * gd) {
        A = nA;
        B = nB;
        fval = o1[0];
        ok = true;
        break;
      }
      step *= 0.5;
    }
    if (!ok) {
      failed = 1;
      break;
    }
  }
  if (tid == 0) {
    out[0] = A;
    out[1] = B;
    out[2] = (double)it;
    out[3] = (double)failed;
  }
}

__global__ void platt_proba_kernel(const double* __restrict__ f, int64_t n, double A, double B, double* __restrict__ p) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double s = A * f[i] + B, e = exp(-fabs(s));
  p[i] = (s >= 0.0) ? e / (1.0 + e) : 1.0 / (1.0 + e);
}

}  // namespace tkm

using namespace tkm;

extern "C" int tkm_cv_decision_values(const tkm_path* p, int32_t t, int32_t l, const int32_t* foldid, double* f_out,
                                      void* stream) {
  if (!p || !foldid || !f_out) return set_error(TKM_EINVAL, "tkm_cv_decision_values: NULL argument");
  if (t < 0 || t >= p->T || l < 0 || l >= p->L) return set_error(TKM_EINVAL, "tkm_cv_decision_values: (t, l) out of range");
  TKM_TRY(device_check());
  cudaStream_t st = (cudaStream_t)stream;
  const tkm_spectral* s = p->spec;
  const int64_t n = s->n;
  for (int64_t j = 0; j < n; ++j)
    if (foldid[j] < 0 || foldid[j] >= p->V) return set_error(TKM_EINVAL, "tkm_cv_decision_values: foldid out of range");
  DevBuf d_fold;
  TKM_TRY(d_fold.alloc((size_t)n * sizeof(int32_t), false, st));
  TKM_CUDA(cudaMemcpyAsync(d_fold.p, foldid, n * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  const int col0 = (t * (p->V + 1)) * p->L + l;
  HeldOutEpi epi{d_fold.as<int32_t>(), p->beta0.as<double>(), col0, p->L, f_out};
  // the V columns (t, l, v = 0..V-1) are rows col0 + v L of `a`: a strided view with leading dimension L ldr
  TKM_TRY(gemm_f64_once(p->a.as<double>() + (int64_t)col0 * s->ldr, (int64_t)p->L * s->ldr, s->UL.as<double>(), s->ldr,
                        p->V, (int)n, (int)s->r, epi, st));
  TKM_CUDA(cudaStreamSynchronize(st));   // d_fold is freed on return
  return TKM_OK;
}

extern "C" int tkm_platt_fit(const double* f, const double* y, int64_t n, double* A, double* B, int32_t* iters,
                             void* stream) {
  if (!f || !y || !A || !B || n < 2 || n > (1 << 30)) return set_error(TKM_EINVAL, "tkm_platt_fit: bad arguments");
  TKM_TRY(device_check());
  cudaStream_t st = (cudaStream_t)stream;
  DevBuf out;
  TKM_TRY(out.alloc(4 * sizeof(double), true, st));
  platt_fit_kernel<<<1, 1024, 0, st>>>(f, y, (int)n, 100, out.as<double>());
  TKM_LAUNCH_CHECK();
  double h[4];
  TKM_CUDA(cudaMemcpyAsync(h, out.p, sizeof(h), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaStreamSynchronize(st));
  *A = h[0];
  *B = h[1];
  if (iters) *iters = (int32_t)h[2];
  if (h[3] != 0.0) return set_error(TKM_ENOTCONV, "tkm_platt_fit: line search failed (degenerate scores?)");
  return TKM_OK;
}

extern "C" int tkm_platt_proba(const double* f, int64_t n, double A, double B, double* p_out, void* stream) {
  if (!f || !p_out || n < 1) return set_error(TKM_EINVAL, "tkm_platt_proba: bad arguments");
  TKM_TRY(device_check());
  platt_proba_kernel<<<(unsigned)ceil_div(n, 256), 256, 0, (cudaStream_t)stream>>>(f, n, A, B, p_out);
  TKM_LAUNCH_CHECK();
  return TKM_OK;
}
