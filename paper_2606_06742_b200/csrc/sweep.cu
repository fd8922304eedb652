// sweep.cu -- S3-S8: the batched spectral majorise-minimise sweep (tkm_fit_path), FP64 path.
//
// PAPER.md:142-146 / 174-176 (update w+ = wbar - H^-1 d), PAPER.md:226-230 (spectral block inverse),
// Algorithm 1 in its V-fold form, readings G1-G7, G10.
//
// Every (variant t, lambda l, fold v) problem is one "column"; all live columns are stacked and one
// iteration is   GEMM-A + loss epilogue  ->  GEMM-B + spectral epilogue  ->  per-column update:
//
//   GEMM-A  F^T = Abar (U Lam)^T      epilogue: z = M psi(y, f + bbar)/n_c -> Zt ; per-CTA sums of z
//   GEMM-B  zeta^T = Zt (U^T)^T       epilogue: rho = zeta + 2 lam abar -> Rho ; per-CTA sums of
//                                               S Lam u1 rho  and  rho^2
//   update  gamma0, q, kkt from the partial sums (fixed order => deterministic); dbeta0 = q/s;
//           da = S (rho - dbeta0 c u1); a+ = abar - da; gradient restart; next Nesterov extrapolation
//
// State lives in spectral coordinates a = U^T alpha, one column per ROW ("slot") so that a column's
// vector is contiguous.  Converged columns are frozen by the update kernel and compacted out of the
// GEMM batch by the host every `check_every` iterations (hole filling: live slots from the tail move
// into the holes; finished rows are first copied to the result array).
#include <algorithm>
#include <cmath>
#include <new>

#include "gemm_f64.cuh"
#include "handles.cuh"

namespace tkm {

__device__ __forceinline__ double psi_dev(int loss, double y, double f, double smooth, double tau) {
  if (loss == TKM_LOSS_HINGE) {
    const double u = y * f;   // L'_delta(u): -1 | (u - 1 - delta)/(2 delta) | 0
    const double lp = (u <= 1.0 - smooth) ? -1.0 : ((u >= 1.0 + smooth) ? 0.0 : (u - 1.0 - smooth) / (2.0 * smooth));
    return y * lp;
  } else if (loss == TKM_LOSS_LOGISTIC) {
    const double u = y * f;   // -y / (1 + e^u), overflow-safe
    const double e = exp(-fabs(u));
    const double sg = (u >= 0.0) ? e / (1.0 + e) : 1.0 / (1.0 + e);
    return -y * sg;
  } else {
    const double t = y - f;   // -H'_gamma(t)  (reading G10)
    const double hp = (t < -smooth) ? tau - 1.0 : ((t > smooth) ? tau : t / (2.0 * smooth) + tau - 0.5);
    return -hp;
  }
}

// ---- GEMM-A epilogue (S5): loss derivative, Zt store, per-CTA column sums ------------------------
struct LossEpi {
  const double* y;           // [n]
  const int32_t* foldid;     // [n]
  const int32_t* col_of_slot;
  const double* bbar;        // [B] by column
  const double* col_nc;      // [B]
  const double* col_tau;     // [B]
  const int32_t* col_v;      // [B]
  int loss;
  double smooth;
  double* Zt;                // [slots][ldz]
  int64_t ldz;
  double* gpart;             // [m blocks][ldpart] by slot
  int64_t ldpart;
  template <int BN, int BM, int WARPS_N, int WARPS_M, int TN, int TM>
  __device__ __forceinline__ void run(double (&acc)[TN][TM][2], int n_blk0, int m_blk0, int warp_n,
                                      int warp_m, int lane, int N, int M, double* scratch) const {
    constexpr int WN = BN / WARPS_N, WM = BM / WARPS_M;
    double yv[TM][2];
    int fv[TM][2];
#pragma unroll
    for (int j = 0; j < TM; ++j)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int m = m_blk0 + warp_m * WM + j * 8 + 2 * (lane & 3) + e;
        yv[j][e] = (m < M) ? y[m] : 0.0;
        fv[j][e] = (m < M) ? foldid[m] : -1;
      }
    double colsum[TN];
#pragma unroll
    for (int i = 0; i < TN; ++i) {
      colsum[i] = 0.0;
      const int slot = n_blk0 + warp_n * WN + i * 8 + (lane >> 2);
      if (slot >= N) continue;
      const int col = col_of_slot[slot];
      const double bb = bbar[col], inv_nc = 1.0 / col_nc[col], tau = col_tau[col];
      const int v = col_v[col];
      double* zrow = Zt + (int64_t)slot * ldz;
#pragma unroll
      for (int j = 0; j < TM; ++j) {
        const int m = m_blk0 + warp_m * WM + j * 8 + 2 * (lane & 3);
        double z[2];
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          z[e] = (m + e < M && fv[j][e] != v) ? psi_dev(loss, yv[j][e], acc[i][j][e] + bb, smooth, tau) * inv_nc : 0.0;
          colsum[i] += z[e];
        }
        if (m + 1 < M) {
          *reinterpret_cast<double2*>(zrow + m) = make_double2(z[0], z[1]);
        } else if (m < M) {
          zrow[m] = z[0];
        }
      }
    }
    double tot;
    if (cta_row_reduce<BN, WARPS_N, WARPS_M, TN>(colsum, warp_n, warp_m, lane, scratch, tot)) {
      const int slot = n_blk0 + (int)threadIdx.x;
      if (slot < N) gpart[(int64_t)blockIdx.x * ldpart + slot] = tot;
    }
  }
};

// ---- GEMM-B epilogue (S6): rho = zeta + 2 lam abar, partial sums for q and ||rho||^2 -------------
struct SpecEpi {
  const double* lam;         // [ldr] eigenvalues
  const double* u1;          // [ldr]
  const int32_t* col_of_slot;
  const double* col_lam;     // [B]
  const double* col_c;       // [B] c = curv / n_c
  const double* Abar;        // [slots][lda]
  int64_t lda;
  double* Rho;               // [slots][lda]
  double* qpart;             // [m blocks][ldpart]
  double* r2part;
  int64_t ldpart;
  template <int BN, int BM, int WARPS_N, int WARPS_M, int TN, int TM>
  __device__ __forceinline__ void run(double (&acc)[TN][TM][2], int n_blk0, int m_blk0, int warp_n,
                                      int warp_m, int lane, int N, int M, double* scratch) const {
    constexpr int WN = BN / WARPS_N, WM = BM / WARPS_M;
    double lv[TM][2], lu[TM][2];   // Lam_i and Lam_i u1_i
#pragma unroll
    for (int j = 0; j < TM; ++j)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int i = m_blk0 + warp_m * WM + j * 8 + 2 * (lane & 3) + e;
        lv[j][e] = (i < M) ? lam[i] : 0.0;
        lu[j][e] = (i < M) ? lam[i] * u1[i] : 0.0;
      }
    double qs[TN], r2[TN];
#pragma unroll
    for (int t = 0; t < TN; ++t) {
      qs[t] = r2[t] = 0.0;
      const int slot = n_blk0 + warp_n * WN + t * 8 + (lane >> 2);
      if (slot >= N) continue;
      const int col = col_of_slot[slot];
      const double two_lam = 2.0 * col_lam[col], cc = col_c[col];
      const double* arow = Abar + (int64_t)slot * lda;
      double* rrow = Rho + (int64_t)slot * lda;
#pragma unroll
      for (int j = 0; j < TM; ++j) {
        const int i = m_blk0 + warp_m * WM + j * 8 + 2 * (lane & 3);
        double rho[2] = {0.0, 0.0};
        if (i + 1 < M) {
          const double2 ab = *reinterpret_cast<const double2*>(arow + i);
          rho[0] = acc[t][j][0] + two_lam * ab.x;
          rho[1] = acc[t][j][1] + two_lam * ab.y;
          *reinterpret_cast<double2*>(rrow + i) = make_double2(rho[0], rho[1]);
        } else if (i < M) {
          rho[0] = acc[t][j][0] + two_lam * arow[i];
          rrow[i] = rho[0];
        }
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          // S_i Lam_i u1_i rho_i with S_i = 1/(2 lam + c Lam_i)  (G1)
          qs[t] += lu[j][e] * rho[e] / (two_lam + cc * lv[j][e]);
          r2[t] += rho[e] * rho[e];
        }
      }
    }
    double tot;
    if (cta_row_reduce<BN, WARPS_N, WARPS_M, TN>(qs, warp_n, warp_m, lane, scratch, tot)) {
      const int slot = n_blk0 + (int)threadIdx.x;
      if (slot < N) qpart[(int64_t)blockIdx.x * ldpart + slot] = tot;
    }
    if (cta_row_reduce<BN, WARPS_N, WARPS_M, TN>(r2, warp_n, warp_m, lane, scratch, tot)) {
      const int slot = n_blk0 + (int)threadIdx.x;
      if (slot < N) r2part[(int64_t)blockIdx.x * ldpart + slot] = tot;
    }
  }
};

// ---- per-round initialisation (S3, G4): constants c, s; a' = a; abar = a; r = 1 ------------------
struct RoundArgs {
  int r;
  int64_t lda;
  const double* lam;
  const double* u1;
  double thin, curv;
  const double* col_lam;
  const double* col_nc;
  double* col_c;
  double* col_s;
  const double* a_out;   // [B][lda] solution so far (by column)
  double *A, *Aprev, *Abar;
  double *beta, *beta_prev, *bbar, *rk;
  int32_t *done, *iters_round, *col_of_slot;
};

__global__ void __launch_bounds__(256) init_round_kernel(RoundArgs p) {
  __shared__ double red[32];
  const int col = blockIdx.x;
  const double lamc = p.col_lam[col], c = p.curv / p.col_nc[col];
  double acc = 0.0;
  const int64_t off = (int64_t)col * p.lda;
  for (int i = threadIdx.x; i < p.r; i += blockDim.x) {
    const double u = p.u1[i];
    acc += u * u / (2.0 * lamc + c * p.lam[i]);
    const double a = p.a_out[off + i];
    p.A[off + i] = a;
    p.Aprev[off + i] = a;
    p.Abar[off + i] = a;
  }
  acc = block_sum(acc, red);
  if (threadIdx.x == 0) {
    p.col_c[col] = c;
    p.col_s[col] = c * p.thin + 2.0 * lamc * c * acc;   // Schur complement s (G1)
    p.beta_prev[col] = p.beta[col];
    p.bbar[col] = p.beta[col];
    p.rk[col] = 1.0;
    p.done[col] = 0;
    p.iters_round[col] = 0;
    p.col_of_slot[col] = col;
  }
}

// ---- S7: per-column update, stop test, restart, next extrapolation --------------------------------
struct UpdateArgs {
  int r, n, nblkA, nblkB, restart, maxit;
  int64_t lda, ldpart;
  double tol;
  const double* lam;
  const double* u1;
  const int32_t* col_of_slot;
  const double *col_lam, *col_c, *col_s, *col_nc;
  const double *gpart, *qpart, *r2part;
  const double* Rho;
  double *A, *Aprev, *Abar;
  double *beta, *beta_prev, *bbar, *rk, *kkt;
  int32_t *done, *iters, *iters_round, *flags;
};

__global__ void __launch_bounds__(256) update_kernel(UpdateArgs p) {
  __shared__ double red[32];
  const int slot = blockIdx.x;
  const int col = p.col_of_slot[slot];
  if (p.done[col]) return;   // frozen until the host compacts it away
  double g0 = 0.0, qd = 0.0, r2 = 0.0;
  for (int b = threadIdx.x; b < p.nblkA; b += blockDim.x) g0 += p.gpart[(int64_t)b * p.ldpart + slot];
  for (int b = threadIdx.x; b < p.nblkB; b += blockDim.x) {
    qd += p.qpart[(int64_t)b * p.ldpart + slot];
    r2 += p.r2part[(int64_t)b * p.ldpart + slot];
  }
  g0 = block_sum(g0, red);
  qd = block_sum(qd, red);
  r2 = block_sum(r2, red);
  const double lamc = p.col_lam[col], c = p.col_c[col], s = p.col_s[col], nc = p.col_nc[col];
  const double dbeta = (g0 - c * qd) / s;                            // PAPER.md:208 (Alg.1 l.17)
  const double kkt = fmax(fabs(g0), nc * sqrt(r2) / sqrt((double)p.n));   // reading G6
  const double beta = p.beta[col], bbar = p.bbar[col];
  const double beta_new = bbar - dbeta;
  const int64_t off = (int64_t)slot * p.lda;
  double g = 0.0;
  for (int i = threadIdx.x; i < p.r; i += blockDim.x) {
    const double S = 1.0 / (2.0 * lamc + c * p.lam[i]);
    const double da = S * (p.Rho[off + i] - dbeta * c * p.u1[i]);    // PAPER.md:207 (Alg.1 l.16)
    const double an = p.Abar[off + i] - da;                           // PAPER.md:212 (Alg.1 l.19)
    g += da * (an - p.A[off + i]);
    p.Aprev[off + i] = an;   // a' is dead once abar has been formed: use it as scratch for a+
  }
  g = block_sum(g, red) + dbeta * (beta_new - beta);
  double rk = p.rk[col];
  rk = 0.5 * (1.0 + sqrt(1.0 + 4.0 * rk * rk));                       // PAPER.md:199 (Alg.1 l.12)
  if (p.restart && g > 0.0) rk = 1.0;                                 // gradient restart
  const double rk_next = 0.5 * (1.0 + sqrt(1.0 + 4.0 * rk * rk));
  const double mu = (rk - 1.0) / rk_next;                             // PAPER.md:203 (Alg.1 l.14)
  for (int i = threadIdx.x; i < p.r; i += blockDim.x) {
    const double aold = p.A[off + i], an = p.Aprev[off + i];
    p.Aprev[off + i] = aold;
    p.A[off + i] = an;
    p.Abar[off + i] = an + mu * (an - aold);
  }
  if (threadIdx.x == 0) {
    p.beta_prev[col] = beta;
    p.beta[col] = beta_new;
    p.bbar[col] = beta_new + mu * (beta_new - beta);
    p.rk[col] = rk;
    p.kkt[col] = kkt;
    p.iters[col] += 1;
    const int itr = p.iters_round[col] + 1;
    p.iters_round[col] = itr;
    if (kkt <= p.tol) {
      p.done[col] = 1;
    } else if (itr >= p.maxit) {
      p.done[col] = 1;
      p.flags[col] = 1;
    }
  }
}

// rows: dst_base[dst_idx[k]][:] = src_base[src_idx[k]][:] for k < count (one CTA per k and per array)
struct RowCopy {
  const double* src;
  double* dst;
};
__global__ void row_copy_kernel(RowCopy c0, RowCopy c1, RowCopy c2, int narr, const int32_t* __restrict__ src_idx,
                                const int32_t* __restrict__ dst_idx, int64_t ld, int len) {
  const RowCopy c = blockIdx.y == 0 ? c0 : (blockIdx.y == 1 ? c1 : c2);
  const int64_t so = (int64_t)src_idx[blockIdx.x] * ld, dof = (int64_t)dst_idx[blockIdx.x] * ld;
  for (int i = threadIdx.x; i < len; i += blockDim.x) c.dst[dof + i] = c.src[so + i];
  (void)narr;
}

static double curvature_of(tkm_loss loss, double smooth) {
  return loss == TKM_LOSS_LOGISTIC ? 0.25 : 1.0 / (2.0 * smooth);   // 1/kappa, kappa = 2 delta
}

}  // namespace tkm

using namespace tkm;

extern "C" int tkm_fit_path(const tkm_spectral* s, const void* y, tkm_loss loss, const tkm_loss_opts* opts,
                            const double* lambdas, int32_t L, const int32_t* foldid, int32_t V, double tol,
                            int32_t maxit, const tkm_path* warm, tkm_path** out, void* stream) {
  if (!out) return set_error(TKM_EINVAL, "tkm_fit_path: out is NULL");
  *out = nullptr;
  if (!s || !y || !opts || !lambdas || !foldid) return set_error(TKM_EINVAL, "tkm_fit_path: NULL argument");
  if (loss != TKM_LOSS_HINGE && loss != TKM_LOSS_LOGISTIC && loss != TKM_LOSS_QUANTILE)
    return set_error(TKM_EINVAL, "tkm_fit_path: unknown loss %d", (int)loss);
  if (L < 1 || V < 2 || V > s->n) return set_error(TKM_EINVAL, "tkm_fit_path: need L >= 1 and 2 <= V <= n");
  if (!(tol > 0.0) || maxit < 1) return set_error(TKM_EINVAL, "tkm_fit_path: need tol > 0 and maxit >= 1");
  for (int l = 0; l < L; ++l)
    if (!(lambdas[l] > 0.0)) return set_error(TKM_EINVAL, "tkm_fit_path: lambda[%d] = %g must be > 0", l, lambdas[l]);
  int T = 1;
  if (loss == TKM_LOSS_QUANTILE) {
    T = opts->T > 0 ? opts->T : 0;
    if (T < 1 || !opts->taus) return set_error(TKM_EINVAL, "tkm_fit_path: QUANTILE needs T >= 1 and taus");
    for (int t = 0; t < T; ++t)
      if (!(opts->taus[t] > 0.0 && opts->taus[t] < 1.0)) return set_error(TKM_EINVAL, "tkm_fit_path: tau must be in (0,1)");
  }
  const int rounds = loss == TKM_LOSS_LOGISTIC ? 1 : opts->rounds;
  if (rounds < 1) return set_error(TKM_EINVAL, "tkm_fit_path: rounds must be >= 1");
  if (loss != TKM_LOSS_LOGISTIC && (!(opts->smooth0 > 0.0) || !(opts->eta > 0.0 && opts->eta <= 1.0)))
    return set_error(TKM_EINVAL, "tkm_fit_path: need smooth0 > 0 and 0 < eta <= 1");
  if (s->sweep_dt != TKM_F64) return set_error(TKM_ENOTIMPL, "tkm_fit_path: only the FP64 sweep is built");
  TKM_TRY(device_check());
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t n = s->n, r = s->r, ldr = s->ldr, ldn = s->ldn;
  const int64_t B64 = (int64_t)T * L * (V + 1);
  if (B64 > (1 << 24)) return set_error(TKM_EINVAL, "tkm_fit_path: too many columns");
  const int B = (int)B64;
  if (warm && (warm->spec != s || warm->B != B)) return set_error(TKM_EINVAL, "tkm_fit_path: warm path has another shape");

  // fold sizes, every fold non-empty
  std::vector<int64_t> fsize(V, 0);
  for (int64_t j = 0; j < n; ++j) {
    if (foldid[j] < 0 || foldid[j] >= V) return set_error(TKM_EINVAL, "tkm_fit_path: foldid[%lld] out of range", (long long)j);
    fsize[foldid[j]]++;
  }
  for (int v = 0; v < V; ++v)
    if (fsize[v] == 0 || fsize[v] == n) return set_error(TKM_EINVAL, "tkm_fit_path: fold %d is empty or everything", v);
  // labels must be +-1 for the classifiers
  {
    std::vector<double> hy(n);
    TKM_CUDA(cudaMemcpyAsync(hy.data(), y, n * sizeof(double), cudaMemcpyDeviceToHost, st));
    TKM_CUDA(cudaStreamSynchronize(st));
    for (int64_t j = 0; j < n; ++j) {
      if (!std::isfinite(hy[j])) return set_error(TKM_EINVAL, "tkm_fit_path: y[%lld] is not finite", (long long)j);
      if (loss != TKM_LOSS_QUANTILE && hy[j] != 1.0 && hy[j] != -1.0)
        return set_error(TKM_EINVAL, "tkm_fit_path: y[%lld] = %g, classifiers need labels +-1", (long long)j, hy[j]);
    }
  }

  tkm_path* p = new (std::nothrow) tkm_path();
  if (!p) return set_error(TKM_ENOMEM, "out of host memory");
  struct Guard {
    tkm_path* p;
    cudaStream_t st;
    ~Guard() {
      if (p) {
        cudaStreamSynchronize(st);
        delete p;
      }
    }
  } guard{p, st};
  p->spec = s;
  p->L = L;
  p->V = V;
  p->T = T;
  p->B = B;
  p->loss = loss;
  p->lambdas.assign(lambdas, lambdas + L);
  if (loss == TKM_LOSS_QUANTILE) p->taus.assign(opts->taus, opts->taus + T);

  // column table, c = (t (V+1) + v) L + l
  std::vector<double> h_lam(B), h_tau(B), h_nc(B);
  std::vector<int32_t> h_v(B);
  for (int t = 0; t < T; ++t)
    for (int v = 0; v <= V; ++v)
      for (int l = 0; l < L; ++l) {
        const int c = (t * (V + 1) + v) * L + l;
        h_lam[c] = lambdas[l];
        h_tau[c] = loss == TKM_LOSS_QUANTILE ? opts->taus[t] : 0.0;
        h_v[c] = v;
        h_nc[c] = (double)(v < V ? n - fsize[v] : n);   // divisor n_c (G3)
      }
  TKM_TRY(p->a.alloc((size_t)B * ldr * sizeof(double), true, st));
  TKM_TRY(p->beta0.alloc((size_t)B * sizeof(double), true, st));
  TKM_TRY(p->col_lam.alloc((size_t)B * sizeof(double), false, st));
  TKM_TRY(p->col_tau.alloc((size_t)B * sizeof(double), false, st));
  TKM_TRY(p->col_nc.alloc((size_t)B * sizeof(double), false, st));
  TKM_TRY(p->col_v.alloc((size_t)B * sizeof(int32_t), false, st));
  TKM_CUDA(cudaMemcpyAsync(p->col_lam.p, h_lam.data(), B * sizeof(double), cudaMemcpyHostToDevice, st));
  TKM_CUDA(cudaMemcpyAsync(p->col_tau.p, h_tau.data(), B * sizeof(double), cudaMemcpyHostToDevice, st));
  TKM_CUDA(cudaMemcpyAsync(p->col_nc.p, h_nc.data(), B * sizeof(double), cudaMemcpyHostToDevice, st));
  TKM_CUDA(cudaMemcpyAsync(p->col_v.p, h_v.data(), B * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  if (warm) {
    TKM_CUDA(cudaMemcpyAsync(p->a.p, warm->a.p, (size_t)B * ldr * sizeof(double), cudaMemcpyDeviceToDevice, st));
    TKM_CUDA(cudaMemcpyAsync(p->beta0.p, warm->beta0.p, (size_t)B * sizeof(double), cudaMemcpyDeviceToDevice, st));
  }

  // working set
  DevBuf A, Aprev, Abar, Rho, Zt, gpart, qpart, r2part, d_fold;
  DevBuf col_c, col_s, beta_prev, bbar, rk, kkt, done, iters, iters_round, flags, col_of_slot, idx_src, idx_dst;
  TKM_TRY(A.alloc((size_t)B * ldr * sizeof(double), true, st));
  TKM_TRY(Aprev.alloc((size_t)B * ldr * sizeof(double), true, st));
  TKM_TRY(Abar.alloc((size_t)B * ldr * sizeof(double), true, st));
  TKM_TRY(Rho.alloc((size_t)B * ldr * sizeof(double), true, st));
  TKM_TRY(Zt.alloc((size_t)B * ldn * sizeof(double), true, st));
  const int64_t nblkA_max = ceil_div(n, 64), nblkB_max = ceil_div(r, 64);
  const int64_t ldpart = round_up(B, 16);
  TKM_TRY(gpart.alloc((size_t)nblkA_max * ldpart * sizeof(double), true, st));
  TKM_TRY(qpart.alloc((size_t)nblkB_max * ldpart * sizeof(double), true, st));
  TKM_TRY(r2part.alloc((size_t)nblkB_max * ldpart * sizeof(double), true, st));
  TKM_TRY(d_fold.alloc((size_t)n * sizeof(int32_t), false, st));
  TKM_CUDA(cudaMemcpyAsync(d_fold.p, foldid, n * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  for (DevBuf* b : {&col_c, &col_s, &beta_prev, &bbar, &rk, &kkt}) TKM_TRY(b->alloc((size_t)B * sizeof(double), true, st));
  for (DevBuf* b : {&done, &iters, &iters_round, &flags, &col_of_slot, &idx_src, &idx_dst})
    TKM_TRY(b->alloc((size_t)B * sizeof(int32_t), true, st));
  PinBuf h_done, h_idx;
  TKM_TRY(h_done.alloc((size_t)B * sizeof(int32_t)));
  TKM_TRY(h_idx.alloc((size_t)2 * B * sizeof(int32_t)));
  std::vector<int32_t> slot_col(B);

  const int check_every = opts->check_every > 0 ? opts->check_every : 16;
  const int restart = opts->restart ? 1 : 0;
  // optional sampling of the two contractions with CUDA events: the first iteration after every
  // poll (all `nslots` columns are live there), read back at the next poll (bench.py `roofline`)
  cudaEvent_t pev[3] = {nullptr, nullptr, nullptr};
  struct PevGuard {
    cudaEvent_t* e;
    ~PevGuard() {
      for (int i = 0; i < 3; ++i)
        if (e[i]) cudaEventDestroy(e[i]);
    }
  } pev_guard{pev};
  if (opts->profile)
    for (auto& e : pev) TKM_CUDA(cudaEventCreate(&e));
  double smooth = opts->smooth0;
  for (int rnd = 0; rnd < rounds; ++rnd) {
    if (loss != TKM_LOSS_LOGISTIC && rnd > 0) smooth *= opts->eta;   // PAPER.md:220 (Alg.1 l.22)
    const double curv = curvature_of(loss, smooth);
    const double rtol = (rnd + 1 < rounds && opts->warm_tol > 0.0) ? opts->warm_tol : tol;
    RoundArgs ra{(int)r, ldr, s->lam.as<double>(), s->u1.as<double>(), s->thin, curv,
                 p->col_lam.as<double>(), p->col_nc.as<double>(), col_c.as<double>(), col_s.as<double>(),
                 p->a.as<double>(), A.as<double>(), Aprev.as<double>(), Abar.as<double>(),
                 p->beta0.as<double>(), beta_prev.as<double>(), bbar.as<double>(), rk.as<double>(),
                 done.as<int32_t>(), iters_round.as<int32_t>(), col_of_slot.as<int32_t>()};
    init_round_kernel<<<B, 256, 0, st>>>(ra);
    TKM_LAUNCH_CHECK();
    for (int c = 0; c < B; ++c) slot_col[c] = c;
    int nslots = B;
    int it = 0;
    while (nslots > 0) {
      const int steps = std::max(1, std::min(check_every, maxit - it));
      for (int k = 0; k < steps; ++k) {
        const bool sample = opts->profile && k == 0;
        if (sample) TKM_CUDA(cudaEventRecord(pev[0], st));
        GemmOperands ga{Abar.as<double>(), ldr, s->UL.as<double>(), ldr, nslots, (int)n, (int)r};
        LossEpi le{(const double*)y, d_fold.as<int32_t>(), col_of_slot.as<int32_t>(), bbar.as<double>(),
                   p->col_nc.as<double>(), p->col_tau.as<double>(), p->col_v.as<int32_t>(), (int)loss, smooth,
                   Zt.as<double>(), ldn, gpart.as<double>(), ldpart};
        TKM_TRY(gemm_f64_dispatch(ga, le, st));
        if (sample) TKM_CUDA(cudaEventRecord(pev[1], st));
        GemmOperands gb{Zt.as<double>(), ldn, s->Ut.as<double>(), ldn, nslots, (int)r, (int)n};
        SpecEpi se{s->lam.as<double>(), s->u1.as<double>(), col_of_slot.as<int32_t>(), p->col_lam.as<double>(),
                   col_c.as<double>(), Abar.as<double>(), ldr, Rho.as<double>(), qpart.as<double>(),
                   r2part.as<double>(), ldpart};
        TKM_TRY(gemm_f64_dispatch(gb, se, st));
        if (sample) TKM_CUDA(cudaEventRecord(pev[2], st));
        UpdateArgs ua{(int)r, (int)n, (int)ceil_div(n, gemm_f64_tile_bm(nslots, n)),
                      (int)ceil_div(r, gemm_f64_tile_bm(nslots, r)), restart, maxit, ldr, ldpart, rtol,
                      s->lam.as<double>(), s->u1.as<double>(), col_of_slot.as<int32_t>(), p->col_lam.as<double>(),
                      col_c.as<double>(), col_s.as<double>(), p->col_nc.as<double>(), gpart.as<double>(),
                      qpart.as<double>(), r2part.as<double>(), Rho.as<double>(), A.as<double>(), Aprev.as<double>(),
                      Abar.as<double>(), p->beta0.as<double>(), beta_prev.as<double>(), bbar.as<double>(),
                      rk.as<double>(), kkt.as<double>(), done.as<int32_t>(), iters.as<int32_t>(),
                      iters_round.as<int32_t>(), flags.as<int32_t>()};
        update_kernel<<<nslots, 256, 0, st>>>(ua);
        TKM_LAUNCH_CHECK();
      }
      it += steps;
      TKM_CUDA(cudaMemcpyAsync(h_done.p, done.p, (size_t)B * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
      TKM_CUDA(cudaStreamSynchronize(st));
      if (opts->profile) {
        float ma = 0.f, mb = 0.f;
        TKM_CUDA(cudaEventElapsedTime(&ma, pev[0], pev[1]));
        TKM_CUDA(cudaEventElapsedTime(&mb, pev[1], pev[2]));
        p->prof_gemm_ms[0] += ma;
        p->prof_gemm_ms[1] += mb;
        p->prof_gemm_flops += 2.0 * (double)nslots * (double)n * (double)r;   // per GEMM
        p->prof_gemm_samples += 1;
      }
      const int32_t* hd = h_done.as<int32_t>();
      // finished slots are copied to the result rows, then holes are filled from the tail
      int32_t* src = h_idx.as<int32_t>();
      int32_t* dst = src + B;
      int nfin = 0, nact = 0;
      for (int sl = 0; sl < nslots; ++sl) {
        if (hd[slot_col[sl]]) {
          src[nfin] = sl;
          dst[nfin] = slot_col[sl];
          ++nfin;
        } else {
          ++nact;
        }
      }
      if (nfin == 0) continue;
      TKM_CUDA(cudaMemcpyAsync(idx_src.p, src, nfin * sizeof(int32_t), cudaMemcpyHostToDevice, st));
      TKM_CUDA(cudaMemcpyAsync(idx_dst.p, dst, nfin * sizeof(int32_t), cudaMemcpyHostToDevice, st));
      {
        RowCopy c0{A.as<double>(), p->a.as<double>()};
        row_copy_kernel<<<dim3(nfin, 1), 256, 0, st>>>(c0, c0, c0, 1, idx_src.as<int32_t>(), idx_dst.as<int32_t>(), ldr, (int)r);
        TKM_LAUNCH_CHECK();
      }
      TKM_CUDA(cudaStreamSynchronize(st));   // src/dst are reused below
      int nmove = 0;
      int hole = 0, tail = nslots - 1;
      while (true) {
        while (hole < nact && !hd[slot_col[hole]]) ++hole;
        while (tail >= nact && hd[slot_col[tail]]) --tail;
        if (hole >= nact || tail < nact) break;
        src[nmove] = tail;
        dst[nmove] = hole;
        slot_col[hole] = slot_col[tail];
        ++nmove;
        ++hole;
        --tail;
      }
      if (nmove > 0) {
        TKM_CUDA(cudaMemcpyAsync(idx_src.p, src, nmove * sizeof(int32_t), cudaMemcpyHostToDevice, st));
        TKM_CUDA(cudaMemcpyAsync(idx_dst.p, dst, nmove * sizeof(int32_t), cudaMemcpyHostToDevice, st));
        RowCopy c0{A.as<double>(), A.as<double>()}, c1{Aprev.as<double>(), Aprev.as<double>()},
            c2{Abar.as<double>(), Abar.as<double>()};
        row_copy_kernel<<<dim3(nmove, 3), 256, 0, st>>>(c0, c1, c2, 3, idx_src.as<int32_t>(), idx_dst.as<int32_t>(), ldr, (int)r);
        TKM_LAUNCH_CHECK();
      }
      TKM_CUDA(cudaMemcpyAsync(col_of_slot.p, slot_col.data(), (size_t)nact * sizeof(int32_t), cudaMemcpyHostToDevice, st));
      TKM_CUDA(cudaStreamSynchronize(st));   // slot_col / pinned lists are host memory reused next poll
      nslots = nact;
    }
  }
  p->smooth_final = loss == TKM_LOSS_LOGISTIC ? 0.0 : smooth;
  p->h_beta0.resize(B);
  p->h_kkt.resize(B);
  p->h_iters.resize(B);
  p->h_flags.resize(B);
  TKM_CUDA(cudaMemcpyAsync(p->h_beta0.data(), p->beta0.p, B * sizeof(double), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaMemcpyAsync(p->h_kkt.data(), kkt.p, B * sizeof(double), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaMemcpyAsync(p->h_iters.data(), iters.p, B * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaMemcpyAsync(p->h_flags.data(), flags.p, B * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaStreamSynchronize(st));
  p->total_col_iters = 0;
  bool notconv = false;
  for (int c = 0; c < B; ++c) {
    p->total_col_iters += p->h_iters[c];
    notconv |= p->h_flags[c] != 0;
  }
  guard.p = nullptr;
  *out = p;
  if (notconv) return set_error(TKM_ENOTCONV, "tkm_fit_path: some columns hit maxit (see flags)");
  return TKM_OK;
}

extern "C" void tkm_path_free(tkm_path* p) { delete p; }

extern "C" int tkm_path_info(const tkm_path* p, int32_t* B, int64_t* r, int32_t* iters, double* kkt, int32_t* flags,
                             double* beta0, int64_t* total_col_iters) {
  if (!p) return set_error(TKM_EINVAL, "tkm_path_info: NULL handle");
  if (B) *B = p->B;
  if (r) *r = p->spec->r;
  if (iters) memcpy(iters, p->h_iters.data(), p->B * sizeof(int32_t));
  if (kkt) memcpy(kkt, p->h_kkt.data(), p->B * sizeof(double));
  if (flags) memcpy(flags, p->h_flags.data(), p->B * sizeof(int32_t));
  if (beta0) memcpy(beta0, p->h_beta0.data(), p->B * sizeof(double));
  if (total_col_iters) *total_col_iters = p->total_col_iters;
  return TKM_OK;
}

extern "C" int tkm_path_profile(const tkm_path* p, double* gemm_ms, double* gemm_flops, int64_t* samples) {
  if (!p) return set_error(TKM_EINVAL, "tkm_path_profile: NULL handle");
  if (gemm_ms) {
    gemm_ms[0] = p->prof_gemm_ms[0];
    gemm_ms[1] = p->prof_gemm_ms[1];
  }
  if (gemm_flops) *gemm_flops = p->prof_gemm_flops;
  if (samples) *samples = p->prof_gemm_samples;
  return TKM_OK;
}

extern "C" int tkm_path_get_a(const tkm_path* p, double* a_out, void* stream) {
  if (!p || !a_out) return set_error(TKM_EINVAL, "tkm_path_get_a: NULL argument");
  const int64_t r = p->spec->r;
  TKM_CUDA(cudaMemcpy2DAsync(a_out, r * sizeof(double), p->a.p, p->spec->ldr * sizeof(double), r * sizeof(double),
                             p->B, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
  return TKM_OK;
}
