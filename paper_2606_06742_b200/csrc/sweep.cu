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
// vector is contiguous.  Several independent problems that share y, the folds and the lambda grid
// (the bandwidths of a sigma grid: one spectral handle each) are swept together as GROUPS of one
// launch (tkm_fit_path_multi), which keeps the SMs full when each group's live batch is narrow.
//
// Converged columns are frozen by the update kernel and compacted out of the GEMM batch ON THE DEVICE
// every `check_every` iterations (hole filling: live slots from the tail move into the holes; finished
// rows are first copied to the result array).  All kernels read the live-slot counts from device
// memory, so the host never waits for the GPU inside a round: it enqueues the next batch of
// iterations first and only then reads the previous batch's counts (an upper bound for the grids).
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <new>

#include "gemm_f64.cuh"
#include "gemm_tf32.cuh"
#include "handles.cuh"
#include "losses.cuh"

namespace tkm {

// Element (slot row gs, sample m) of the dz operand: row-major [G*B][lddz], or K-blocked [n/32][blk_rows][32]
// (blk_rows = G*B) when the tcgen05 GEMM-B reads it that way (thin U, large n).
__device__ __forceinline__ int64_t dz_index(int64_t gs, int m, int64_t lddz, int blk_rows) {
  return blk_rows ? ((int64_t)(m >> 5) * blk_rows + gs) * 32 + (m & 31) : gs * lddz + m;
}

// Same function with the divisions hoisted: inv_2s = 1 / (2 smooth) (unused by the smooth losses).
__device__ __forceinline__ double psi_fast(int loss, double y, double f, double smooth, double inv_2s, double tau) {
  if (loss == TKM_LOSS_HINGE) {
    const double u = y * f;
    const double lp = (u <= 1.0 - smooth) ? -1.0 : ((u >= 1.0 + smooth) ? 0.0 : (u - 1.0 - smooth) * inv_2s);
    return y * lp;
  } else if (loss == TKM_LOSS_QUANTILE) {
    const double t = y - f;
    return -((t < -smooth) ? tau - 1.0 : ((t > smooth) ? tau : t * inv_2s + tau - 0.5));
  }
  return psi_dev(loss, y, f, smooth, tau);
}

// Per-group device pointers (one group = one spectral handle, e.g. one bandwidth of a sigma grid).
struct GroupPtrs {
  const double* lam[GEMM_MAX_GROUPS];   // [ldr] eigenvalues
  const double* u1[GEMM_MAX_GROUPS];    // [ldr] U^T 1
  double* a_out[GEMM_MAX_GROUPS];       // [B][ldr] result rows of the group's path
  double thin[GEMM_MAX_GROUPS];         // n - ||u1||^2 (0 for a full orthogonal U)
};

// Index conventions: B columns per group; "gc" = g*B + column, "gs" = g*B + slot.

// ---- GEMM-A epilogue (S5): loss derivative, Zt store, per-CTA column sums ------------------------
struct LossEpi {
  const double* y;           // [n]
  const int32_t* foldid;     // [n]
  const int32_t* col_of_slot;   // [G*B] by gs -> column
  const double* bbar;        // [G*B] by gc
  const double* col_nc;      // [B]
  const double* col_tau;     // [B]
  const int32_t* col_v;      // [B]
  int B, loss;
  double smooth;
  double* Zt;                // [G*B][ldz] by gs
  int64_t ldz;
  double* gpart;             // [m blocks][ldpart] by gs
  int64_t ldpart;
  float* dz_hi;              // [G*B][lddz] by gs or NULL: TF32 (hi, lo) split of z - z_old, the operand of the
  float* dz_lo;              //   delta-form GEMM-B (zeta += U^T dz on the tcgen05 tensor cores)
  int64_t lddz;
  double* Fb;                // [G*B][ldz] by gs or NULL: keeps Fbar = U Lam abar for the delta-form GEMM-A
  int dz_blk_rows;           // 0: dz row-major; G*B: dz K-blocked (dz_index)

  template <class Cfg>
  __device__ __forceinline__ void run(double (&acc)[Cfg::TN][Cfg::TM][2], int n_blk0, int m_blk0, int warp_n,
                                      int warp_m, int lane, int N, int M, int grp, double* scratch) const {
    constexpr int TN = Cfg::TN, TM = Cfg::TM;
    double yv[TM][2];
    int fv[TM][2];
#pragma unroll
    for (int j = 0; j < TM; ++j)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int m = m_blk0 + (warp_m * TM + j) * 8 + 2 * (lane & 3) + e;
        yv[j][e] = (m < M) ? y[m] : 0.0;
        fv[j][e] = (m < M) ? foldid[m] : -1;
      }
    const int g0 = grp * B;
    double colsum[TN];
#pragma unroll
    for (int i = 0; i < TN; ++i) {
      colsum[i] = 0.0;
      const int slot = n_blk0 + (warp_n * TN + i) * 8 + (lane >> 2);
      if (slot >= N) continue;
      const int col = col_of_slot[g0 + slot];
      const double bb = bbar[g0 + col], inv_nc = 1.0 / col_nc[col], tau = col_tau[col];
      const int v = col_v[col];
      double* zrow = Zt + (int64_t)(g0 + slot) * ldz;
#pragma unroll
      for (int j = 0; j < TM; ++j) {
        const int m = m_blk0 + (warp_m * TM + j) * 8 + 2 * (lane & 3);
        double z[2];
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          z[e] = (m + e < M && fv[j][e] != v) ? psi_dev(loss, yv[j][e], acc[i][j][e] + bb, smooth, tau) * inv_nc : 0.0;
          colsum[i] += z[e];
        }
        if (dz_hi && m < M) {   // m is even and lddz a multiple of 32: the pair is in bounds (padding is never read)
          const double2 zo = *reinterpret_cast<const double2*>(zrow + m);
          const double d0 = z[0] - zo.x, d1 = (m + 1 < M) ? z[1] - zo.y : 0.0;
          const float h0 = to_tf32((float)d0), h1 = to_tf32((float)d1);
          const int64_t o = dz_index(g0 + slot, m, lddz, dz_blk_rows);
          *reinterpret_cast<float2*>(dz_hi + o) = make_float2(h0, h1);
          *reinterpret_cast<float2*>(dz_lo + o) = make_float2(to_tf32((float)(d0 - (double)h0)), to_tf32((float)(d1 - (double)h1)));
        }
        if (m + 1 < M) {
          *reinterpret_cast<double2*>(zrow + m) = make_double2(z[0], z[1]);
          if (Fb) *reinterpret_cast<double2*>(Fb + (int64_t)(g0 + slot) * ldz + m) = make_double2(acc[i][j][0], acc[i][j][1]);
        } else if (m < M) {
          zrow[m] = z[0];
          if (Fb) Fb[(int64_t)(g0 + slot) * ldz + m] = acc[i][j][0];
        }
      }
    }
    double tot;
    if (cta_row_reduce<Cfg>(colsum, warp_n, warp_m, lane, scratch, tot)) {
      const int slot = n_blk0 + (int)threadIdx.x;
      if (slot < N) gpart[(int64_t)gemm_m_block() * ldpart + g0 + slot] = tot;
    }
  }
};

// ---- GEMM-B epilogue (S6): rho = zeta + 2 lam abar (the column sums of rho are taken by update_kernel) ----
struct SpecEpi {
  const int32_t* col_of_slot;   // [G*B]
  const double* col_lam;     // [B]
  int B;
  const double* Abar;        // [G*B][lda] by gs
  int64_t lda;
  double* Rho;               // [G*B][lda] by gs
  double* Zeta;              // [G*B][lda] by gs or NULL: keeps zeta = U^T z for the delta-form iterations
  template <class Cfg>
  __device__ __forceinline__ void run(double (&acc)[Cfg::TN][Cfg::TM][2], int n_blk0, int m_blk0, int warp_n,
                                      int warp_m, int lane, int N, int M, int grp, double*) const {
    constexpr int TN = Cfg::TN, TM = Cfg::TM;
    const int g0 = grp * B;
#pragma unroll
    for (int t = 0; t < TN; ++t) {
      const int slot = n_blk0 + (warp_n * TN + t) * 8 + (lane >> 2);
      if (slot >= N) continue;
      const double two_lam = 2.0 * col_lam[col_of_slot[g0 + slot]];
      const int64_t row = (int64_t)(g0 + slot) * lda;
#pragma unroll
      for (int j = 0; j < TM; ++j) {
        const int i = m_blk0 + (warp_m * TM + j) * 8 + 2 * (lane & 3);
        if (i + 1 < M) {
          const double2 ab = *reinterpret_cast<const double2*>(Abar + row + i);
          *reinterpret_cast<double2*>(Rho + row + i) =
              make_double2(acc[t][j][0] + two_lam * ab.x, acc[t][j][1] + two_lam * ab.y);
          if (Zeta) *reinterpret_cast<double2*>(Zeta + row + i) = make_double2(acc[t][j][0], acc[t][j][1]);
        } else if (i < M) {
          Rho[row + i] = acc[t][j][0] + two_lam * Abar[row + i];
          if (Zeta) Zeta[row + i] = acc[t][j][0];
        }
      }
    }
  }
};

// ---- epilogue of the tcgen05 delta-form contractions: the raw FP32 product, one slot per row ----------------------
// Thread = one output index m (a TMEM lane), 16 consecutive slots per call; for a fixed slot the 32 lanes of a
// warp store 128 contiguous bytes.  The FP64 state updates that consume the product (F+ = Fbar - U Lam da with the
// loss derivative; zeta += U^T dz) are NOT fused here: a tensor-memory epilogue has 8 warps per SM to hide the
// latency of ~8 FP64 loads and stores per element and ran at < 1 TB/s (ncu, profiles/r02_pair_kernel.md: 354 us
// per launch at full width, tensor pipe 17 %), while the same arithmetic as a plain elementwise kernel over all
// (slot, m) streams at HBM speed and the product costs 4 bytes per element to pass through L2.
struct ProdEpi {
  static constexpr bool kReduce = false;
  float* out;        // [G*B][ldo] by gs
  int64_t ldo;
  int B;
  __device__ __forceinline__ void chunk(const float (&v)[16], int m, int n0, int N, int M, int grp, double*, int) const {
    if (m >= M) return;
    float* base = out + (int64_t)(grp * B + n0) * ldo + m;
    const int cnt = min(16, N - n0);
#pragma unroll
    for (int k = 0; k < 16; ++k)
      if (k < cnt) base[(int64_t)k * ldo] = v[k];
  }
};

// ---- K-split GEMM-B (thin U: r x B outputs, n ~ 10^5..10^6 deep) ------------------------------------------------
// With few output tiles and a very long contraction the launch cannot fill the SMs, so K is cut into S ranges
// (GemmArgs::ksplit): every CTA stores its partial U^T z into part[split], and spec_finalize_kernel sums the S
// partials in a fixed order and applies the SpecEpi arithmetic.  (The tcgen05 kernel needs none of this: its
// stream-K partition cuts along K by itself.)
struct PartEpi {   // FP64 DMMA kernel
  int B, ksplit;
  int64_t lda, split_stride;
  double* part;   // [S][G*B][lda]
  template <class Cfg>
  __device__ __forceinline__ void run(double (&acc)[Cfg::TN][Cfg::TM][2], int n_blk0, int m_blk0, int warp_n,
                                      int warp_m, int lane, int N, int M, int grp, double*) const {
    constexpr int TN = Cfg::TN, TM = Cfg::TM;
    double* base = part + (int64_t)gemm_split_index(ksplit) * split_stride;
#pragma unroll
    for (int t = 0; t < TN; ++t) {
      const int slot = n_blk0 + (warp_n * TN + t) * 8 + (lane >> 2);
      if (slot >= N) continue;
      const int64_t row = (int64_t)(grp * B + slot) * lda;
#pragma unroll
      for (int j = 0; j < TM; ++j) {
        const int i = m_blk0 + (warp_m * TM + j) * 8 + 2 * (lane & 3);
        if (i + 1 < M)
          *reinterpret_cast<double2*>(base + row + i) = make_double2(acc[t][j][0], acc[t][j][1]);
        else if (i < M)
          base[row + i] = acc[t][j][0];
      }
    }
  }
};

// zeta = (accumulate ? Zeta : 0) + sum_s part[s];  Zeta <- zeta (if kept);  rho = zeta + 2 lam abar
__global__ void __launch_bounds__(256) spec_finalize_kernel(const double* __restrict__ part, int S, int64_t split_stride,
                                                            const int32_t* __restrict__ nslots,
                                                            const int32_t* __restrict__ col_of_slot,
                                                            const double* __restrict__ col_lam, int B, int r, int64_t lda,
                                                            const double* __restrict__ Abar, double* __restrict__ Zeta,
                                                            int accumulate, double* __restrict__ Rho) {
  const int grp = blockIdx.z, slot = blockIdx.y;
  if (slot >= nslots[grp]) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= r) return;
  const int64_t o = (int64_t)(grp * B + slot) * lda + i;
  double z = accumulate ? Zeta[o] : 0.0;
  double acc = 0.0;
  for (int s = 0; s < S; ++s) acc += part[(int64_t)s * split_stride + o];
  z += acc;
  if (Zeta) Zeta[o] = z;
  Rho[o] = z + 2.0 * col_lam[col_of_slot[grp * B + slot]] * Abar[o];
}

// ---- delta form of S5 (after the tcgen05 GEMM-A): F+ = Fbar - U Lam da, next extrapolation, loss derivative ------
// One thread per (slot, sample m).  State per slot: Fb = Fbar_k (what the loss saw), Fp = F_k.  With G = U Lam da_k
// from the tcgen05 product:  F_{k+1} = Fbar_k - G,  Fbar_{k+1} = F_{k+1} + mu_{k+1} (F_{k+1} - F_k), then z, dz and
// the per-block column sums of z exactly as in LossEpi (summed in a fixed order by update_kernel).
struct FLossArgs {
  const double* y;
  const int32_t* foldid;
  const int32_t* nslots;        // [G]
  const int32_t* col_of_slot;   // [G*B]
  const double* bbar;           // [G*B] by gc
  const double* mu;             // [G*B] by gc: momentum that formed the current abar
  const double* col_nc;
  const double* col_tau;
  const int32_t* col_v;
  int B, loss, n;
  double smooth, inv_2s;
  const float* prod;            // [G*B][ldprod] by gs: U Lam da
  int64_t ldprod;
  double* Fb;                   // [G*B][ldz]
  double* Fp;                   // [G*B][ldz]
  double* Zt;                   // [G*B][ldz]
  int64_t ldz;
  float* dz_hi;
  float* dz_lo;
  int64_t lddz;
  double* gpart;                // [blocks along m][ldpart] by gs
  int64_t ldpart;
  int dz_blk_rows;
};
constexpr int FLOSS_THREADS = 256, FLOSS_EPT = 4;   // samples per block: 1024
__global__ void __launch_bounds__(FLOSS_THREADS) floss_kernel(FLossArgs p) {
  __shared__ double red[32];
  const int slot = blockIdx.x, grp = blockIdx.z, mblk = blockIdx.y;   // slots on x: the leave-one-out form has > 65535
  if (slot >= p.nslots[grp]) return;
  const int gs = grp * p.B + slot, col = p.col_of_slot[gs], gc = grp * p.B + col;
  const double mu = p.mu[gc], bb = p.bbar[gc], inv_nc = 1.0 / p.col_nc[col], tau = p.col_tau[col];
  const int hv = p.col_v[col];
  const int64_t row = (int64_t)gs * p.ldz;
  const double* __restrict__ y = p.y;
  const int32_t* __restrict__ fold = p.foldid;
  const float* __restrict__ prod = p.prod + (int64_t)gs * p.ldprod;
  double* __restrict__ Fb = p.Fb + row;
  double* __restrict__ Fp = p.Fp + row;
  double* __restrict__ Zt = p.Zt + row;
  // all loads of the thread's samples first (independent round trips in flight), then the arithmetic and the stores
  double fbv[FLOSS_EPT], fpv[FLOSS_EPT], zov[FLOSS_EPT], yv[FLOSS_EPT];
  float pv[FLOSS_EPT];
  int fv[FLOSS_EPT];
#pragma unroll
  for (int e = 0; e < FLOSS_EPT; ++e) {
    const int m = (mblk * FLOSS_EPT + e) * FLOSS_THREADS + threadIdx.x;
    if (m < p.n) {
      fbv[e] = Fb[m];
      fpv[e] = Fp[m];
      zov[e] = Zt[m];
      pv[e] = prod[m];
      yv[e] = y[m];
      fv[e] = fold[m];
    }
  }
  double zsum = 0.0;
#pragma unroll
  for (int e = 0; e < FLOSS_EPT; ++e) {
    const int m = (mblk * FLOSS_EPT + e) * FLOSS_THREADS + threadIdx.x;
    if (m < p.n) {
      const double fn = fbv[e] - (double)pv[e];
      const double fb = fn + mu * (fn - fpv[e]);
      Fp[m] = fn;
      Fb[m] = fb;
      double z = 0.0;
      if (fv[e] != hv) z = psi_fast(p.loss, yv[e], fb + bb, p.smooth, p.inv_2s, tau) * inv_nc;
      const double d = z - zov[e];
      Zt[m] = z;
      const float h = to_tf32((float)d);
      const int64_t od = dz_index(gs, m, p.lddz, p.dz_blk_rows);
      p.dz_hi[od] = h;
      p.dz_lo[od] = to_tf32((float)(d - (double)h));
      zsum += z;
    }
  }
  zsum = block_sum(zsum, red);   // fixed order: deterministic
  if (threadIdx.x == 0) p.gpart[(int64_t)mblk * p.ldpart + gs] = zsum;
}

// ---- per-round initialisation (S3, G4): constants c, s; a' = a; abar = a; r = 1 ------------------
struct RoundArgs {
  int r, B;
  int64_t lda;
  GroupPtrs gp;
  double curv;
  const double* col_lam;   // [B]
  const double* col_nc;    // [B]
  double* col_c;           // [B]
  double* col_s;           // [G*B]
  double *A, *Aprev, *Abar;   // [G*B][lda]
  double *beta, *beta_prev, *bbar, *rk;   // [G*B]
  int32_t *done, *iters_round, *col_of_slot;   // [G*B]
  int32_t* nslots;         // [G]
  const int32_t* active;   // [G*B] by gc or NULL: columns that take part in this round (reading G23); the others
                           //   start as finished and leave the batch in the compaction that follows
};

__global__ void __launch_bounds__(256) init_round_kernel(RoundArgs p) {
  __shared__ double red[32];
  const int col = blockIdx.x, grp = blockIdx.y;
  const int gc = grp * p.B + col;
  const double* lam = p.gp.lam[grp];
  const double* u1 = p.gp.u1[grp];
  const double lamc = p.col_lam[col], c = p.curv / p.col_nc[col];
  double acc = 0.0;
  const double* src = p.gp.a_out[grp] + (int64_t)col * p.lda;
  const int64_t off = (int64_t)gc * p.lda;
  for (int i = threadIdx.x; i < p.r; i += blockDim.x) {
    const double u = u1[i];
    acc += u * u / (2.0 * lamc + c * lam[i]);
    const double a = src[i];
    p.A[off + i] = a;
    p.Aprev[off + i] = a;
    p.Abar[off + i] = a;
  }
  acc = block_sum(acc, red);
  if (threadIdx.x == 0) {
    if (grp == 0) p.col_c[col] = c;
    p.col_s[gc] = c * p.gp.thin[grp] + 2.0 * lamc * c * acc;   // Schur complement s (G1)
    p.beta_prev[gc] = p.beta[gc];
    p.bbar[gc] = p.beta[gc];
    p.rk[gc] = 1.0;
    p.done[gc] = (p.active && !p.active[gc]) ? 1 : 0;
    p.iters_round[gc] = 0;
    p.col_of_slot[gc] = col;
    if (col == 0) p.nslots[grp] = p.B;
  }
}

// ---- S7: per-column update, stop test, restart, next extrapolation --------------------------------
struct UpdateArgs {
  int r, n, B, nblkA, restart, maxit;
  int exact;   // 0: rho came from the delta-form recurrence -- a column may not be declared converged on it
  int64_t lda, ldpart;
  double tol;
  GroupPtrs gp;
  const int32_t* nslots;       // [G]
  const int32_t* col_of_slot;  // [G*B]
  const double *col_lam, *col_c, *col_nc;   // [B]
  const double* col_s;         // [G*B]
  const double* gpart;
  const double* Rho;
  double *A, *Aprev, *Abar;
  double *beta, *beta_prev, *bbar, *rk, *kkt;   // [G*B]
  int32_t *done, *iters, *iters_round, *flags;  // [G*B]
  float* da_hi;    // [G*B][ldda] by gs or NULL: TF32 (hi, lo) split of the step da, operand of the delta-form GEMM-A
  float* da_lo;
  int64_t ldda;
  double* mu;      // [G*B] by gc or NULL: momentum used for the new abar
  const float* zinc;   // [G*B][ldzinc] by gs or NULL: the tcgen05 product U^T dz of a delta-form iteration; then
  int64_t ldzinc;      //   zeta <- zeta + zinc (FP64 state `Zeta`), rho = zeta + 2 lam abar is formed here
  double* Zeta;        // [G*B][lda] by gs (with zinc)
  double* RhoW;        // [G*B][lda]: rho is kept for the second pass when the vector does not fit one chunk
  unsigned long long* fam_cnt;   // [4] or NULL (profile == 2): column-iterations by kernel family of this iteration's
  int famA, famB;                //   two contractions (0 DMMA A, 1 DMMA B, 2 tcgen05 A, 3 tcgen05 B)
};

// One CTA per live slot.  The vectors are walked in chunks of 256 x UPD_EPT pairs with all loads of a chunk
// issued before its arithmetic (the dependent chain is then two block reductions plus two memory round
// trips, not one round trip per element); when the whole vector fits one chunk (r <= 2048) the second
// pass works from registers.  Padded entries (i >= r) hold zeros in every array and stay zero.
constexpr int UPD_EPT = 4;   // double2 elements per thread and chunk
__global__ void __launch_bounds__(256, 2) update_kernel(UpdateArgs p) {
  __shared__ double red[3][32];
  const int slot = blockIdx.x, grp = blockIdx.y;
  if (slot >= p.nslots[grp]) return;
  const int gs = grp * p.B + slot;
  const int col = p.col_of_slot[gs];
  const int gc = grp * p.B + col;
  if (p.done[gc]) return;   // frozen until the next compaction removes it
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const double2* __restrict__ lam2 = reinterpret_cast<const double2*>(p.gp.lam[grp]);
  const double2* __restrict__ u12 = reinterpret_cast<const double2*>(p.gp.u1[grp]);
  const double lamc = p.col_lam[col], c = p.col_c[col], s = p.col_s[gc], nc = p.col_nc[col];
  const double two_lam = 2.0 * lamc;
  const int64_t off2 = ((int64_t)gs * p.lda) >> 1;   // lda is a multiple of 16
  const double2* Rho2 = reinterpret_cast<const double2*>(p.Rho) + off2;   // (may alias RhoW in the delta form)
  double2* __restrict__ A2 = reinterpret_cast<double2*>(p.A) + off2;
  double2* __restrict__ Ap2 = reinterpret_cast<double2*>(p.Aprev) + off2;
  double2* __restrict__ Ab2 = reinterpret_cast<double2*>(p.Abar) + off2;
  const int npair = (int)(p.lda >> 1);
  const bool single = npair <= 256 * UPD_EPT;
  // Column sums (fixed order => deterministic): gamma0 = 1^T z from the per-tile partials of GEMM-A's epilogue;
  // sum_i S_i Lam_i u1_i rho_i (G1) and ||rho||^2 from rho itself.  When the whole vector fits
  // one chunk the operands loaded here stay in registers for the update below.
  double2 rho[UPD_EPT], ab[UPD_EPT], lm[UPD_EPT], uu[UPD_EPT], a_old[UPD_EPT], a_new[UPD_EPT];
  double g0 = 0.0, qd = 0.0, r2 = 0.0;
  for (int b = tid; b < p.nblkA; b += 256) g0 += p.gpart[(int64_t)b * p.ldpart + gs];
  double2* __restrict__ Zeta2 = p.zinc ? reinterpret_cast<double2*>(p.Zeta) + off2 : nullptr;
  double2* RhoW2 = p.zinc ? reinterpret_cast<double2*>(p.RhoW) + off2 : nullptr;
  const float2* __restrict__ zinc2 = p.zinc ? reinterpret_cast<const float2*>(p.zinc + (int64_t)gs * p.ldzinc) : nullptr;
  for (int base = 0; base < npair; base += 256 * UPD_EPT) {
#pragma unroll
    for (int e = 0; e < UPD_EPT; ++e) {
      const int i = base + e * 256 + tid;
      if (i < npair) {
        lm[e] = lam2[i];
        uu[e] = u12[i];
        if (single || zinc2) ab[e] = Ab2[i];
        if (single) a_old[e] = A2[i];
        if (zinc2) {
          // delta form of S6: zeta += U^T dz (the tcgen05 product), rho = zeta + 2 lam abar
          const double2 ze = Zeta2[i];
          const float2 zi = zinc2[i];   // columns beyond r are never written and stay zero
          const double2 zn = make_double2(ze.x + (double)zi.x, ze.y + (double)zi.y);
          Zeta2[i] = zn;
          rho[e] = make_double2(zn.x + two_lam * ab[e].x, zn.y + two_lam * ab[e].y);
          if (!single) RhoW2[i] = rho[e];
        } else {
          rho[e] = Rho2[i];
        }
      }
    }
#pragma unroll
    for (int e = 0; e < UPD_EPT; ++e) {
      const int i = base + e * 256 + tid;
      if (i < npair) {
        qd += lm[e].x * uu[e].x * rho[e].x / (two_lam + c * lm[e].x) + lm[e].y * uu[e].y * rho[e].y / (two_lam + c * lm[e].y);
        r2 += rho[e].x * rho[e].x + rho[e].y * rho[e].y;
      }
    }
  }
  g0 = warp_sum(g0);
  qd = warp_sum(qd);
  r2 = warp_sum(r2);
  if (lane == 0) {
    red[0][w] = g0;
    red[1][w] = qd;
    red[2][w] = r2;
  }
  __syncthreads();
  g0 = qd = r2 = 0.0;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    g0 += red[0][k];
    qd += red[1][k];
    r2 += red[2][k];
  }
  const double dbeta = (g0 - c * qd) / s;                            // PAPER.md:208 (Alg.1 l.17)
  const double kkt = fmax(fabs(g0), nc * sqrt(r2) / sqrt((double)p.n));   // reading G6
  const double beta = p.beta[gc], bbar = p.bbar[gc];
  const double beta_new = bbar - dbeta;
  const double dbc = dbeta * c;
  double g = 0.0;
  for (int base = 0; base < npair; base += 256 * UPD_EPT) {
    if (!single) {
#pragma unroll
      for (int e = 0; e < UPD_EPT; ++e) {
        const int i = base + e * 256 + tid;
        if (i < npair) {
          rho[e] = zinc2 ? RhoW2[i] : Rho2[i];
          ab[e] = Ab2[i];
          a_old[e] = A2[i];
          lm[e] = lam2[i];
          uu[e] = u12[i];
        }
      }
    }
#pragma unroll
    for (int e = 0; e < UPD_EPT; ++e) {
      const int i = base + e * 256 + tid;
      if (i < npair) {
        // S_i = 1/(2 lam + c Lam_i); da = S (rho - dbeta c u1)  PAPER.md:207 (Alg.1 l.16); a+ = abar - da (l.19)
        const double dax = (rho[e].x - dbc * uu[e].x) / (two_lam + c * lm[e].x);
        const double day = (rho[e].y - dbc * uu[e].y) / (two_lam + c * lm[e].y);
        a_new[e] = make_double2(ab[e].x - dax, ab[e].y - day);
        g += dax * (a_new[e].x - a_old[e].x) + day * (a_new[e].y - a_old[e].y);
        if (!single) Ap2[i] = a_new[e];   // a' is dead once abar has been formed: scratch for a+
        if (p.da_hi) {
          const float hx = to_tf32((float)dax), hy = to_tf32((float)day);
          const int64_t o = (int64_t)gs * p.ldda + 2 * i;
          *reinterpret_cast<float2*>(p.da_hi + o) = make_float2(hx, hy);
          *reinterpret_cast<float2*>(p.da_lo + o) =
              make_float2(to_tf32((float)(dax - (double)hx)), to_tf32((float)(day - (double)hy)));
        }
      }
    }
  }
  g = warp_sum(g);
  __syncthreads();   // red[] of the first reduction has been consumed
  if (lane == 0) red[0][w] = g;
  __syncthreads();
  g = 0.0;
#pragma unroll
  for (int k = 0; k < 8; ++k) g += red[0][k];
  g += dbeta * (beta_new - beta);
  double rk = p.rk[gc];
  rk = 0.5 * (1.0 + sqrt(1.0 + 4.0 * rk * rk));                       // PAPER.md:199 (Alg.1 l.12)
  if (p.restart && g > 0.0) rk = 1.0;                                 // gradient restart
  const double rk_next = 0.5 * (1.0 + sqrt(1.0 + 4.0 * rk * rk));
  const double mu = (rk - 1.0) / rk_next;                             // PAPER.md:203 (Alg.1 l.14)
  if (single) {
#pragma unroll
    for (int e = 0; e < UPD_EPT; ++e) {
      const int i = e * 256 + tid;
      if (i < npair) {
        Ap2[i] = a_old[e];
        A2[i] = a_new[e];
        Ab2[i] = make_double2(a_new[e].x + mu * (a_new[e].x - a_old[e].x), a_new[e].y + mu * (a_new[e].y - a_old[e].y));
      }
    }
  } else {
    for (int base = 0; base < npair; base += 256 * UPD_EPT) {
#pragma unroll
      for (int e = 0; e < UPD_EPT; ++e) {
        const int i = base + e * 256 + tid;
        if (i < npair) {
          a_old[e] = A2[i];
          a_new[e] = Ap2[i];
        }
      }
#pragma unroll
      for (int e = 0; e < UPD_EPT; ++e) {
        const int i = base + e * 256 + tid;
        if (i < npair) {
          Ap2[i] = a_old[e];
          A2[i] = a_new[e];
          Ab2[i] =
              make_double2(a_new[e].x + mu * (a_new[e].x - a_old[e].x), a_new[e].y + mu * (a_new[e].y - a_old[e].y));
        }
      }
    }
  }
  if (tid == 0) {
    p.beta_prev[gc] = beta;
    p.beta[gc] = beta_new;
    p.bbar[gc] = beta_new + mu * (beta_new - beta);
    p.rk[gc] = rk;
    if (p.mu) p.mu[gc] = mu;
    p.kkt[gc] = kkt;
    p.iters[gc] += 1;
    if (p.fam_cnt) {
      atomicAdd(p.fam_cnt + p.famA, 1ull);
      atomicAdd(p.fam_cnt + p.famB, 1ull);
    }
    const int itr = p.iters_round[gc] + 1;
    p.iters_round[gc] = itr;
    // a column leaves the batch only on an exact iteration (in the delta forms rho carries the drift of the
    // recurrence): converged if its residual meets tol, else flagged once it has used up maxit
    if (p.exact) {
      if (kkt <= p.tol) {
        p.done[gc] = 1;
      } else if (itr >= p.maxit) {
        p.done[gc] = 1;
        p.flags[gc] |= 1;
      }
    }
  }
}

// ---- device-side compaction of converged columns --------------------------------------------------
// plan (one CTA per group): finished slots in slot order -> fin_list; live slots at or beyond the new
// count `nact` in slot order -> tail_list.  The first nholes entries of fin_list are exactly the
// finished slots below nact (the holes), and there are as many tail entries as holes.
struct CompactArgs {
  int B, r;
  int64_t lda;
  GroupPtrs gp;
  int32_t* nslots;          // [G]   in: live slots before, out: after
  int32_t* col_of_slot;     // [G*B]
  const int32_t* done;      // [G*B] by gc
  int32_t* fin_list;        // [G*B]
  int32_t* tail_list;       // [G*B]
  int32_t* counts;          // [G][4]: nfin, nholes, nact, previous nslots
  double *A, *Aprev, *Abar;
  double* Zeta;             // [G*B][lda] or NULL (delta form): moves with its slot
  double* Zt;               // [G*B][ldz] or NULL (delta form)
  int64_t ldz;
  int n;
  double *Fb, *Fp;          // [G*B][ldz] or NULL (delta form of GEMM-A)
  float *da_hi, *da_lo;     // [G*B][ldda] or NULL
  int64_t ldda;
};

__global__ void __launch_bounds__(1024) compact_plan_kernel(CompactArgs p) {
  __shared__ int wsum[2][32];
  __shared__ int run[2];
  __shared__ int s_nact;
  const int grp = blockIdx.x, g0 = grp * p.B;
  const int ns = p.nslots[grp];
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  // pass 1: number of live slots
  int live = 0;
  for (int sl = tid; sl < ns; sl += blockDim.x) live += p.done[g0 + p.col_of_slot[g0 + sl]] ? 0 : 1;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) live += __shfl_xor_sync(0xffffffffu, live, o);
  if (lane == 0) wsum[0][w] = live;
  if (tid == 0) run[0] = run[1] = 0;
  __syncthreads();
  if (tid == 0) {
    int t = 0;
    for (int i = 0; i < (int)(blockDim.x >> 5); ++i) t += wsum[0][i];
    s_nact = t;
  }
  __syncthreads();
  const int nact = s_nact;
  // pass 2: ordered lists by chunked ballot scans
  for (int base = 0; base < ns; base += blockDim.x) {
    const int sl = base + tid;
    int fin = 0, tail = 0;
    if (sl < ns) {
      fin = p.done[g0 + p.col_of_slot[g0 + sl]] ? 1 : 0;
      tail = (!fin && sl >= nact) ? 1 : 0;
    }
    const unsigned bf = __ballot_sync(0xffffffffu, fin), bt = __ballot_sync(0xffffffffu, tail);
    const unsigned below = (1u << lane) - 1u;
    const int pf = __popc(bf & below), pt = __popc(bt & below);
    __syncthreads();   // wsum / run of the previous chunk have been consumed
    if (lane == 0) {
      wsum[0][w] = __popc(bf);
      wsum[1][w] = __popc(bt);
    }
    __syncthreads();
    int of = run[0], ot = run[1];
    for (int i = 0; i < w; ++i) {
      of += wsum[0][i];
      ot += wsum[1][i];
    }
    if (fin) p.fin_list[g0 + of + pf] = sl;
    if (tail) p.tail_list[g0 + ot + pt] = sl;
    __syncthreads();
    if (tid == 0) {
      int tf = 0, tt = 0;
      for (int i = 0; i < (int)(blockDim.x >> 5); ++i) {
        tf += wsum[0][i];
        tt += wsum[1][i];
      }
      run[0] += tf;
      run[1] += tt;
    }
  }
  __syncthreads();
  if (tid == 0) {
    p.counts[grp * 4 + 0] = run[0];   // nfin
    p.counts[grp * 4 + 1] = run[1];   // nholes (= live slots beyond nact)
    p.counts[grp * 4 + 2] = nact;
    p.counts[grp * 4 + 3] = ns;
    p.nslots[grp] = nact;
  }
}

// apply (grid: finished-slot rank x group): save the finished row to the group's result array, then, if
// the slot is a hole below nact, pull the matching live tail row (a, a', abar and its column id) in.
__global__ void __launch_bounds__(256) compact_apply_kernel(CompactArgs p) {
  const int k = blockIdx.x, grp = blockIdx.y, g0 = grp * p.B;
  const int nfin = p.counts[grp * 4 + 0], nholes = p.counts[grp * 4 + 1];
  if (k >= nfin) return;
  const int sl = p.fin_list[g0 + k];
  const int col = p.col_of_slot[g0 + sl];
  const int64_t so = (int64_t)(g0 + sl) * p.lda;
  double* dst = p.gp.a_out[grp] + (int64_t)col * p.lda;
  for (int i = threadIdx.x; i < p.r; i += blockDim.x) dst[i] = p.A[so + i];
  if (k >= nholes) return;
  const int src = p.tail_list[g0 + k];
  const int64_t to = (int64_t)(g0 + src) * p.lda;
  __syncthreads();   // the finished row has been read by every thread before it is overwritten
  for (int i = threadIdx.x; i < p.r; i += blockDim.x) {
    p.A[so + i] = p.A[to + i];
    p.Aprev[so + i] = p.Aprev[to + i];
    p.Abar[so + i] = p.Abar[to + i];
    if (p.Zeta) p.Zeta[so + i] = p.Zeta[to + i];
  }
  if (p.Zt) {
    const int64_t zs = (int64_t)(g0 + sl) * p.ldz, zt = (int64_t)(g0 + src) * p.ldz;
    for (int i = threadIdx.x; i < p.n; i += blockDim.x) p.Zt[zs + i] = p.Zt[zt + i];
    if (p.Fb) {
      for (int i = threadIdx.x; i < p.n; i += blockDim.x) {
        p.Fb[zs + i] = p.Fb[zt + i];
        p.Fp[zs + i] = p.Fp[zt + i];
      }
      const int64_t ds = (int64_t)(g0 + sl) * p.ldda, dt = (int64_t)(g0 + src) * p.ldda;
      for (int i = threadIdx.x; i < p.r; i += blockDim.x) {
        p.da_hi[ds + i] = p.da_hi[dt + i];
        p.da_lo[ds + i] = p.da_lo[dt + i];
      }
    }
  }
  if (threadIdx.x == 0) p.col_of_slot[g0 + sl] = p.col_of_slot[g0 + src];
}

// ---- outer control of the smoothing schedule (reading G23) -------------------------------------
// mode 0 (screen):  pass[gc] = onsched[gc] && gap[gc] <= gap_tol
// mode 1 (certify): columns with pass[gc] && gap[gc] <= gap_tol leave the schedule: onsched = 0, level = rnd
// mode 2 (cap):     columns still on the schedule after the last round whose gap exceeds gap_tol get flag bit 2
__global__ void outer_control_kernel(int mode, int GB, double gap_tol, int rnd, const double* __restrict__ gap,
                                     int32_t* __restrict__ onsched, int32_t* __restrict__ pass, int32_t* __restrict__ level,
                                     int32_t* __restrict__ flags) {
  const int gc = blockIdx.x * blockDim.x + threadIdx.x;
  if (gc >= GB) return;
  const bool ok = gap[gc] <= gap_tol;
  if (mode == 0) {
    pass[gc] = (onsched[gc] && ok) ? 1 : 0;
  } else if (mode == 1) {
    if (pass[gc] && ok) {
      onsched[gc] = 0;
      level[gc] = rnd;
    }
  } else if (onsched[gc] && !ok) {
    flags[gc] |= 2;
  }
}

static double curvature_of(tkm_loss loss, double smooth) {
  if (loss == TKM_LOSS_LOGISTIC) return 0.25;
  if (loss == TKM_LOSS_DWD) return 4.0;   // sup V'' = V''(1/2+)
  return 1.0 / (2.0 * smooth);   // 1/kappa, kappa = 2 delta
}

constexpr int KSPLIT_MIN_K = 16384;   // contraction depth from which GEMM-B may be K-split (thin U, large n)
constexpr int KSPLIT_MAX = 16;
constexpr int KBLOCK_F64_MIN_K = 16384;   // thin U: from this n on, the FP64 GEMM-B reads a K-blocked copy of U^T
constexpr int KBLOCK_MIN_K = 8192;   // contraction depth from which the tcgen05 GEMM-B operands are kept K-blocked (no effect
                                    // at n = 2000, where U^T stays in L2; 2.4x at n = 581012)
constexpr int DELTA_MIN_LIVE = 24;   // live columns (all groups) below which the delta forms are switched off when U is L2-sized
constexpr int DELTA_MIN_FLOOR = 8;   // ... and when U streams from HBM
constexpr int POLL_RING = 8;   // ring of poll results: up to POLL_RING - 2 batches may be in flight

// Live columns (all groups) from which a tcgen05 delta-form launch beats the FP64 DMMA launch it replaces.  The
// pair kernel's time has a floor that does not depend on the width: its stream-K partition gives each of the 74
// pairs G ceil(M / 256) KT / 74 K-tiles, a K-tile is a chain of 12 dependent MMAs (~0.33 us at <= 128 slots,
// measured, profiles/r02_pair_kernel.md), plus ~14 us of prologue, partial exchange and epilogue.  The DMMA launch
// costs 2 n r N / (18 TFLOP/s).  5 x (n = r = 2000): 58 columns; n = r >= 10^4: the floor DELTA_MIN_LIVE.
static int delta_min_live(int64_t n, int64_t r, int G) {
  const double ktA = (double)G * (double)ceil_div(n, 256) * (double)ceil_div(r, 32) / 74.0;   // GEMM-A: M = n, K = r
  const double ktB = (double)G * (double)ceil_div(r, 256) * (double)ceil_div(n, 32) / 74.0;   // GEMM-B: M = r, K = n
  const double t_tc = 0.5 * (ktA + ktB) * 0.33e-6 + 14e-6;
  const double cols = t_tc * 18e12 / (2.0 * (double)n * (double)r);
  // Once one operand copy is far beyond L2 (n >= 10^4) even the narrowest batch is a stream of U from HBM, and the
  // pair kernel streams at 5.3-6.4 TB/s where the DMMA kernel reaches 3.0-3.7 (profiles/r02_narrow_batch.md): the
  // delta forms then stay on down to a handful of columns.  At 5 x n = 2000 (160 MB, half of it L2 hits in the
  // tail) the measured optimum is the model's 58 (1 / 16 / 32 / 58: 1265 / 736 / 710 / 680 ms sweeps).
  if ((double)G * (double)n * (double)r * 8.0 > 2.0 * 126e6) return DELTA_MIN_FLOOR;
  return std::max(DELTA_MIN_LIVE, (int)cols);
}

}  // namespace tkm

using namespace tkm;

extern "C" int tkm_fit_path_multi(const tkm_spectral* const* specs, int32_t G, const void* y, tkm_loss loss,
                                  const tkm_loss_opts* opts, const double* lambdas, int32_t L, const int32_t* foldid,
                                  int32_t V, double tol, int32_t maxit, const tkm_path* const* warm, tkm_path** out,
                                  void* stream) {
  tkm::NvtxRange nvtx_range("tkm_fit_path");
  if (!out) return set_error(TKM_EINVAL, "tkm_fit_path: out is NULL");
  if (G < 1 || G > GEMM_MAX_GROUPS) return set_error(TKM_EINVAL, "tkm_fit_path_multi: need 1 <= G <= %d", GEMM_MAX_GROUPS);
  for (int g = 0; g < G; ++g) out[g] = nullptr;
  if (!specs || !y || !opts || !lambdas || !foldid) return set_error(TKM_EINVAL, "tkm_fit_path: NULL argument");
  for (int g = 0; g < G; ++g)
    if (!specs[g]) return set_error(TKM_EINVAL, "tkm_fit_path: NULL spectral handle");
  const tkm_spectral* s0 = specs[0];
  for (int g = 1; g < G; ++g)
    if (specs[g]->n != s0->n || specs[g]->r != s0->r || specs[g]->ldr != s0->ldr || specs[g]->ldn != s0->ldn)
      return set_error(TKM_EINVAL, "tkm_fit_path_multi: all spectral handles must share n and r");
  if (loss != TKM_LOSS_HINGE && loss != TKM_LOSS_LOGISTIC && loss != TKM_LOSS_QUANTILE && loss != TKM_LOSS_DWD)
    return set_error(TKM_EINVAL, "tkm_fit_path: unknown loss %d", (int)loss);
  if (L < 1 || V < 2 || V > s0->n) return set_error(TKM_EINVAL, "tkm_fit_path: need L >= 1 and 2 <= V <= n");
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
  const bool smoothed = loss == TKM_LOSS_HINGE || loss == TKM_LOSS_QUANTILE;   // logistic and DWD are smooth
  const int rounds = smoothed ? opts->rounds : 1;
  if (rounds < 1) return set_error(TKM_EINVAL, "tkm_fit_path: rounds must be >= 1");
  if (opts->tf32_delta < 0 || opts->tf32_delta > 3) return set_error(TKM_EINVAL, "tkm_fit_path: tf32_delta must be 0..3");
  if (smoothed && (!(opts->smooth0 > 0.0) || !(opts->eta > 0.0 && opts->eta <= 1.0)))
    return set_error(TKM_EINVAL, "tkm_fit_path: need smooth0 > 0 and 0 < eta <= 1");
  TKM_TRY(device_check());
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t n = s0->n, r = s0->r, ldr = s0->ldr, ldn = s0->ldn;
  const int64_t B64 = (int64_t)T * L * (V + 1);
  if (B64 * G > (1 << 22)) return set_error(TKM_EINVAL, "tkm_fit_path: too many columns");
  const int B = (int)B64, GB = B * G;
  if (warm)
    for (int g = 0; g < G; ++g)
      if (!warm[g] || warm[g]->spec != specs[g] || warm[g]->B != B)
        return set_error(TKM_EINVAL, "tkm_fit_path: warm path has another shape");

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

  // the paths (one per group); freed by the guard unless we reach the end
  struct Guard {
    tkm_path** out;
    int G;
    cudaStream_t st;
    bool armed = true;
    ~Guard() {
      if (!armed) return;
      cudaStreamSynchronize(st);
      for (int g = 0; g < G; ++g) {
        delete out[g];
        out[g] = nullptr;
      }
    }
  } guard{out, G, st};

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
  GroupPtrs gp;
  memset(&gp, 0, sizeof(gp));
  for (int g = 0; g < G; ++g) {
    tkm_path* p = new (std::nothrow) tkm_path();
    if (!p) return set_error(TKM_ENOMEM, "out of host memory");
    out[g] = p;
    p->spec = specs[g];
    p->L = L;
    p->V = V;
    p->T = T;
    p->B = B;
    p->loss = loss;
    p->lambdas.assign(lambdas, lambdas + L);
    if (loss == TKM_LOSS_QUANTILE) p->taus.assign(opts->taus, opts->taus + T);
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
    gp.lam[g] = specs[g]->lam.as<double>();
    gp.u1[g] = specs[g]->u1.as<double>();
    gp.a_out[g] = p->a.as<double>();
    gp.thin[g] = specs[g]->thin;
  }
  const tkm_path* p0 = out[0];   // the column tables are identical in every group: use group 0's

  // working set (all groups stacked: row / entry g*B + slot or g*B + column)
  DevBuf A, Aprev, Abar, Rho, Zt, gpart, d_fold;
  DevBuf col_c, col_s, beta, beta_prev, bbar, rk, kkt, done, iters, iters_round, flags, col_of_slot;
  DevBuf nslots, fin_list, tail_list, counts;
  TKM_TRY(A.alloc((size_t)GB * ldr * sizeof(double), true, st, true));
  TKM_TRY(Aprev.alloc((size_t)GB * ldr * sizeof(double), true, st, true));
  TKM_TRY(Abar.alloc((size_t)GB * ldr * sizeof(double), true, st, true));
  TKM_TRY(Rho.alloc((size_t)GB * ldr * sizeof(double), true, st, true));
  TKM_TRY(Zt.alloc((size_t)GB * ldn * sizeof(double), true, st, true));
  const int64_t nblk_max = ceil_div(std::max(n, r), 64);   // smallest BM of any tile configuration
  const int64_t ldpart = round_up(GB, 16);
  TKM_TRY(gpart.alloc((size_t)nblk_max * ldpart * sizeof(double), true, st, true));
  TKM_TRY(d_fold.alloc((size_t)n * sizeof(int32_t), false, st, true));
  TKM_CUDA(cudaMemcpyAsync(d_fold.p, foldid, n * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  TKM_TRY(col_c.alloc((size_t)B * sizeof(double), true, st, true));
  for (DevBuf* b : {&col_s, &beta, &beta_prev, &bbar, &rk, &kkt}) TKM_TRY(b->alloc((size_t)GB * sizeof(double), true, st, true));
  for (DevBuf* b : {&done, &iters, &iters_round, &flags, &col_of_slot, &fin_list, &tail_list})
    TKM_TRY(b->alloc((size_t)GB * sizeof(int32_t), true, st, true));
  TKM_TRY(nslots.alloc((size_t)GEMM_MAX_GROUPS * sizeof(int32_t), true, st, true));
  TKM_TRY(counts.alloc((size_t)GEMM_MAX_GROUPS * 4 * sizeof(int32_t), true, st, true));
  if (warm)
    for (int g = 0; g < G; ++g) {
      TKM_CUDA(cudaMemcpyAsync(out[g]->a.p, warm[g]->a.p, (size_t)B * ldr * sizeof(double), cudaMemcpyDeviceToDevice, st));
      TKM_CUDA(cudaMemcpyAsync(beta.as<double>() + (size_t)g * B, warm[g]->beta0.p, (size_t)B * sizeof(double),
                               cudaMemcpyDeviceToDevice, st));
    }
  // delta-form GEMM-B (tkm_loss_opts.tf32_delta): zeta state, the (hi, lo) increment operand, U^T as (hi, lo)
  const bool delta = opts->tf32_delta != 0;
  const int64_t ldn32 = round_up(n, 32);
  // the operands of the tcgen05 GEMM-B (U^T and dz, both (hi, lo)) are kept K-blocked, [n/32][rows][32], so that
  // a pipeline stage is a contiguous read instead of one 128-byte piece per row (profiles/r01f: 2.4x at n = 581012)
  const bool kblk = delta && n >= KBLOCK_MIN_K;
  const int dz_blk_rows = kblk ? GB : 0;
  DevBuf Zeta, dz_hi, dz_lo, ut_hi[GEMM_MAX_GROUPS], ut_lo[GEMM_MAX_GROUPS];
  if (delta) {
    TKM_TRY(Zeta.alloc((size_t)GB * ldr * sizeof(double), true, st, true));
    TKM_TRY(dz_hi.alloc((size_t)GB * ldn32 * sizeof(float), true, st, true));
    TKM_TRY(dz_lo.alloc((size_t)GB * ldn32 * sizeof(float), true, st, true));
    for (int g = 0; g < G; ++g) {
      TKM_TRY(ut_hi[g].alloc((size_t)r * ldn32 * sizeof(float), false, st, true));   // padding beyond n is outside the
      TKM_TRY(ut_lo[g].alloc((size_t)r * ldn32 * sizeof(float), false, st, true));   // tensor maps: never read
      if (kblk)
        TKM_TRY(split_tf32_kblocked(specs[g]->Ut.as<double>(), ldn, r, n, ut_hi[g].as<float>(), ut_lo[g].as<float>(), st));
      else
        TKM_TRY(split_tf32(specs[g]->Ut.as<double>(), ldn, r, n, ut_hi[g].as<float>(), ut_lo[g].as<float>(), ldn32, st));
    }
  }
  // K-split GEMM-B (thin U with a long contraction): partial sums [KSPLIT_MAX][G*B][ldr]
  const bool ksplit_ok = n >= KSPLIT_MIN_K;
  const int64_t split_stride = (int64_t)GB * ldr;
  DevBuf zpart;
  if (ksplit_ok) TKM_TRY(zpart.alloc((size_t)KSPLIT_MAX * split_stride * sizeof(double), false, st, true));
  // F half (tf32_delta == 2): Fbar / F state, the (hi, lo) step operand, U Lam as (hi, lo), momentum per column
  const bool delta_f = opts->tf32_delta >= 2;
  const int64_t ldr32 = round_up(r, 32);
  const bool kblk_f = delta_f && n >= KBLOCK_MIN_K;   // U Lam (hi, lo) K-blocked: [r/32][n][32]
  DevBuf Fb, Fp, da_hi, da_lo, mu, ul_hi[GEMM_MAX_GROUPS], ul_lo[GEMM_MAX_GROUPS];
  if (delta_f) {
    TKM_TRY(Fb.alloc((size_t)GB * ldn * sizeof(double), true, st, true));
    TKM_TRY(Fp.alloc((size_t)GB * ldn * sizeof(double), true, st, true));
    TKM_TRY(da_hi.alloc((size_t)GB * ldr32 * sizeof(float), true, st, true));
    TKM_TRY(da_lo.alloc((size_t)GB * ldr32 * sizeof(float), true, st, true));
    TKM_TRY(mu.alloc((size_t)GB * sizeof(double), true, st, true));
    for (int g = 0; g < G; ++g) {
      TKM_TRY(ul_hi[g].alloc((size_t)n * ldr32 * sizeof(float), false, st, true));
      TKM_TRY(ul_lo[g].alloc((size_t)n * ldr32 * sizeof(float), false, st, true));
      if (kblk_f)
        TKM_TRY(split_tf32_kblocked(specs[g]->UL.as<double>(), ldr, n, r, ul_hi[g].as<float>(), ul_lo[g].as<float>(), st));
      else
        TKM_TRY(split_tf32(specs[g]->UL.as<double>(), ldr, n, r, ul_hi[g].as<float>(), ul_lo[g].as<float>(), ldr32, st));
    }
  }
  GemmProblem prA2 = {};   // F = U Lam a on the exact iterations of the F half (same tiles as GEMM-A, P = a)
  GemmArgs argsA2;
  Tf32Args targs, targsF;
  DevBuf prodA, prodB;   // FP32 products of the tcgen05 contractions: U Lam da [G*B][ldn32], U^T dz [G*B][ldr32]
  if (delta) TKM_TRY(prodB.alloc((size_t)GB * ldr32 * sizeof(float), true, st, true));
  if (delta_f) TKM_TRY(prodA.alloc((size_t)GB * ldn32 * sizeof(float), true, st, true));
  Tf32Scratch tsc;   // stream-K exchange buffers of the tcgen05 launches of this sweep
  if (opts->tf32_delta != 0) TKM_TRY(tsc.alloc(st));
  memset(&targs, 0, sizeof(targs));
  memset(&targsF, 0, sizeof(targsF));
  targs.terms = targsF.terms = opts->tf32_delta == 3 ? 1 : 3;   // mode 3: single-TF32 products (hi tiles only)
  int tcfg = -1;
  // [POLL_RING][GEMM_MAX_GROUPS] live-slot counts read back after every compaction; pinned once per host thread and
  // kept (cudaMallocHost is a kernel-mode call: none of those in a warm step, see DevBuf)
  static thread_local PinBuf h_ns;
  if (!h_ns.p) TKM_TRY(h_ns.alloc((size_t)POLL_RING * GEMM_MAX_GROUPS * sizeof(int32_t)));

  // events: one "poll landed" event per ring entry; optional GEMM sampling events per ring entry
  const int check_every = opts->check_every > 0 ? opts->check_every : 16;
  // profile == 1: two sampled iterations per batch; profile == 2: every iteration (all launches timed; the
  // useful flops come from device-side column-iteration counters) -- a measurement mode, not for timed runs
  // With the delta forms on and a wide batch the exact FP64 iteration (two DMMA contractions against 2 x (ce - 1)
  // tcgen05 ones) is the larger part of a batch: such batches run 2 x check_every iterations between exact ones.
  const char* ce_env = getenv("TKM_CE_MULT");   // tuning aid: multiplier of the batch length of wide delta-form batches
  const int ce_mult = ce_env && *ce_env ? std::max(1, std::min(8, atoi(ce_env))) : 2;
  const int ce_max = opts->tf32_delta != 0 ? ce_mult * check_every : check_every;
  const int nsamp = opts->profile == 2 ? ce_max : 2;
  const int dmin = opts->delta_min_live > 0 ? opts->delta_min_live : delta_min_live(s0->n, s0->r, G);
  struct Events {
    cudaEvent_t poll[POLL_RING] = {};
    std::vector<cudaEvent_t> pev;   // [POLL_RING][nsamp][4]: (A0, A1, B0, B1) per sampled iteration
    ~Events() {
      for (auto& e : poll)
        if (e) cudaEventDestroy(e);
      for (auto& e : pev)
        if (e) cudaEventDestroy(e);
    }
  } ev;
  // TKM_SWEEP_TRACE=<file>: one line per batch (round, batch, live columns, widest group, tiles, ms) -- a
  // tuning aid; it turns the poll events into timing events and changes nothing else.
  const char* trace_path = getenv("TKM_SWEEP_TRACE");
  FILE* trace = trace_path && *trace_path ? fopen(trace_path, "a") : nullptr;
  struct TraceGuard {
    FILE* f;
    ~TraceGuard() {
      if (f) fclose(f);
    }
  } trace_guard{trace};
  for (auto& e : ev.poll) TKM_CUDA(cudaEventCreateWithFlags(&e, trace ? cudaEventDefault : cudaEventDisableTiming));
  if (opts->profile) {
    ev.pev.assign((size_t)POLL_RING * nsamp * 4, nullptr);
    for (auto& e : ev.pev) TKM_CUDA(cudaEventCreate(&e));
  }
  auto pev = [&](int ring, int sidx, int q) -> cudaEvent_t { return ev.pev[((size_t)ring * nsamp + sidx) * 4 + q]; };
  DevBuf fam_cnt;
  if (opts->profile == 2) TKM_TRY(fam_cnt.alloc(4 * sizeof(unsigned long long), true, st, true));

  // GEMM problems: A = abar x (U Lam)^T, B = Zt x (U^T)^T
  GemmProblem prA, prB;
  prA.P = Abar.as<double>();
  prA.ldp = ldr;
  prA.p_group_rows = B;
  prA.p_total_rows = GB;
  prA.ldq = ldr;
  prA.G = G;
  prA.M = (int)n;
  prA.K = (int)r;
  prB.P = Zt.as<double>();
  prB.ldp = ldn;
  prB.p_group_rows = B;
  prB.p_total_rows = GB;
  prB.ldq = ldn;
  prB.G = G;
  prB.M = (int)r;
  prB.K = (int)n;
  // thin U with n >= KBLOCK_F64_MIN_K: the FP64 GEMM-B reads a K-blocked copy of U^T (its rows are n * 8 bytes
  // apart: every 128-byte piece of a stage would come from another page; profiles/r01f)
  // (K-blocked FP64 copies of BOTH operands for the full kernel at n >= 8192 were measured in round 2 and bought
  // nothing: 3452 against 3664 GB/s at n = 20000 with 14 live columns, profiles/r02_narrow_batch.md -- with rows
  // "only" 160 KB apart the 128-byte pieces of a stage are not what limits the stream; kblk64A stays off.)
  const bool kblk64 = n >= KBLOCK_F64_MIN_K && r < n, kblk64A = false;
  DevBuf utb[GEMM_MAX_GROUPS], ulb[GEMM_MAX_GROUPS];
  for (int g = 0; g < G; ++g) {
    prA.Q[g] = specs[g]->UL.as<double>();
    prB.Q[g] = specs[g]->Ut.as<double>();
    if (kblk64) {
      TKM_TRY(utb[g].alloc((size_t)ceil_div(n, (int64_t)TMA_BOX_K) * r * TMA_BOX_K * sizeof(double), false, st, true));
      TKM_TRY(kblock_f64(specs[g]->Ut.as<double>(), ldn, r, n, utb[g].as<double>(), st));
      prB.Q[g] = utb[g].as<double>();
    }
    if (kblk64A) {
      TKM_TRY(ulb[g].alloc((size_t)ceil_div(r, (int64_t)TMA_BOX_K) * n * TMA_BOX_K * sizeof(double), false, st, true));
      TKM_TRY(kblock_f64(specs[g]->UL.as<double>(), ldr, n, r, ulb[g].as<double>(), st));
      prA.Q[g] = ulb[g].as<double>();
    }
  }
  prB.q_blocked = kblk64;
  prA.q_blocked = kblk64A;
  GemmArgs argsA, argsB;
  GemmTile tileA{-1, 0, 0}, tileB{-1, 0, 0};

  const int restart = opts->restart ? 1 : 0;
  // sampled launches, by kernel family and contraction: [0] DMMA GEMM-A, [1] DMMA GEMM-B, [2] tcgen05 A, [3] tcgen05 B
  double prof_ms[4] = {0.0, 0.0, 0.0, 0.0}, prof_flops[4] = {0.0, 0.0, 0.0, 0.0};
  int64_t prof_launches[4] = {0, 0, 0, 0};
  std::vector<int> samp_kind((size_t)POLL_RING * nsamp * 2, -1);   // [ring][sampled iteration][A, B]: family or -1
  int ce_of[POLL_RING] = {};   // iterations of the batch in each ring slot (trace)
  // One smoothing round (S3-S7 until every participating column has met `rtol`) at level `smooth`; `active`
  // ([G*B] device, or NULL = all columns) selects the participating columns (outer control, reading G23).
  auto run_round = [&](int rnd, double smooth, double rtol, const int32_t* active) -> int {
    NvtxRange nvtx_round("tkm smoothing round");
    const double curv = curvature_of(loss, smooth);
    RoundArgs ra{(int)r, B, ldr, gp, curv, p0->col_lam.as<double>(), p0->col_nc.as<double>(), col_c.as<double>(),
                 col_s.as<double>(), A.as<double>(), Aprev.as<double>(), Abar.as<double>(), beta.as<double>(),
                 beta_prev.as<double>(), bbar.as<double>(), rk.as<double>(), done.as<int32_t>(),
                 iters_round.as<int32_t>(), col_of_slot.as<int32_t>(), nslots.as<int32_t>(), active};
    init_round_kernel<<<dim3(B, G), 256, 0, st>>>(ra);
    TKM_LAUNCH_CHECK();

    // Host view of the live-slot counts: an upper bound that lags the device by at most two batches.
    int bound[GEMM_MAX_GROUPS];
    for (int g = 0; g < G; ++g) bound[g] = B;
    if (active) {
      // columns outside the round leave the batch before its first iteration; the counts are read back once
      CompactArgs c0{B, (int)r, ldr, gp, nslots.as<int32_t>(), col_of_slot.as<int32_t>(), done.as<int32_t>(),
                     fin_list.as<int32_t>(), tail_list.as<int32_t>(), counts.as<int32_t>(), A.as<double>(),
                     Aprev.as<double>(), Abar.as<double>(), nullptr, nullptr, ldn, (int)n, nullptr, nullptr, nullptr,
                     nullptr, ldr32};
      compact_plan_kernel<<<G, 1024, 0, st>>>(c0);
      TKM_LAUNCH_CHECK();
      compact_apply_kernel<<<dim3(B, G), 256, 0, st>>>(c0);
      TKM_LAUNCH_CHECK();
      TKM_CUDA(cudaMemcpyAsync(h_ns.as<int32_t>(), nslots.p, GEMM_MAX_GROUPS * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
      TKM_CUDA(cudaStreamSynchronize(st));
      int tot = 0;
      for (int g = 0; g < G; ++g) tot += (bound[g] = h_ns.as<int32_t>()[g]);
      if (tot == 0) return TKM_OK;
    }
    int64_t batch = 0, done_polls = 0;
    bool finished = false;
    while (!finished) {
      const int ring = (int)(batch % POLL_RING);
      int nmax = 0;
      int64_t ntot = 0;
      for (int g = 0; g < G; ++g) {
        nmax = std::max(nmax, bound[g]);
        ntot += bound[g];
      }
      // tile configuration for this batch (tensor maps are rebuilt only when it changes)
      const GemmTile tA = gemm_f64_choose(bound, G, (int)n, (int)r), tB = gemm_f64_choose(bound, G, (int)r, (int)n);
      if (tA.cfg != tileA.cfg) {
        TKM_TRY(gemm_f64_make_args(prA, tA, &argsA));
        argsA.nslots = nslots.as<int32_t>();
        if (delta_f) {
          prA2 = prA;
          prA2.P = A.as<double>();
          TKM_TRY(gemm_f64_make_args(prA2, tA, &argsA2));
          argsA2.nslots = nslots.as<int32_t>();
        }
        tileA = tA;
      }
      if (tB.cfg != tileB.cfg) {
        TKM_TRY(gemm_f64_make_args(prB, tB, &argsB));
        argsB.nslots = nslots.as<int32_t>();
        tileB = tB;
      }
      argsA.N = argsB.N = argsA2.N = std::max(nmax, 1);
      if (delta) {
        const int want = 0;   // one tile shape: the maps are built once
        if (want != tcfg) {
          const int bn = TF32_PBOX;
          if (kblk) {
            const int64_t kb = ldn32 / 32;
            TKM_TRY(make_tmap_f32(&targs.p_hi, dz_hi.as<float>(), kb * GB, 32, 32, bn));
            TKM_TRY(make_tmap_f32(&targs.p_lo, dz_lo.as<float>(), kb * GB, 32, 32, bn));
            for (int g = 0; g < G; ++g) {
              TKM_TRY(make_tmap_f32(&targs.q_hi[g], ut_hi[g].as<float>(), kb * r, 32, 32, TF32_BM));
              TKM_TRY(make_tmap_f32(&targs.q_lo[g], ut_lo[g].as<float>(), kb * r, 32, 32, TF32_BM));
            }
            targs.kblocked = 3;
            targs.p_blk_rows = GB;
            targs.q_blk_rows = (int)r;
          } else {
            TKM_TRY(make_tmap_f32(&targs.p_hi, dz_hi.as<float>(), GB, n, ldn32, bn));
            TKM_TRY(make_tmap_f32(&targs.p_lo, dz_lo.as<float>(), GB, n, ldn32, bn));
            for (int g = 0; g < G; ++g) {
              TKM_TRY(make_tmap_f32(&targs.q_hi[g], ut_hi[g].as<float>(), r, n, ldn32, TF32_BM));
              TKM_TRY(make_tmap_f32(&targs.q_lo[g], ut_lo[g].as<float>(), r, n, ldn32, TF32_BM));
            }
          }
          targs.nslots = nslots.as<int32_t>();
          targs.p_group_rows = B;
          targs.M = (int)r;
          targs.K = (int)n;
          if (delta_f) {
            TKM_TRY(make_tmap_f32(&targsF.p_hi, da_hi.as<float>(), GB, r, ldr32, bn));
            TKM_TRY(make_tmap_f32(&targsF.p_lo, da_lo.as<float>(), GB, r, ldr32, bn));
            for (int g = 0; g < G; ++g) {
              if (kblk_f) {
                TKM_TRY(make_tmap_f32(&targsF.q_hi[g], ul_hi[g].as<float>(), (ldr32 / 32) * n, 32, 32, TF32_BM));
                TKM_TRY(make_tmap_f32(&targsF.q_lo[g], ul_lo[g].as<float>(), (ldr32 / 32) * n, 32, 32, TF32_BM));
              } else {
                TKM_TRY(make_tmap_f32(&targsF.q_hi[g], ul_hi[g].as<float>(), n, r, ldr32, TF32_BM));
                TKM_TRY(make_tmap_f32(&targsF.q_lo[g], ul_lo[g].as<float>(), n, r, ldr32, TF32_BM));
              }
            }
            targsF.kblocked = kblk_f ? 1 : 0;
            targsF.q_blk_rows = (int)n;
            targsF.nslots = nslots.as<int32_t>();
            targsF.p_group_rows = B;
            targsF.M = (int)n;
            targsF.K = (int)r;
          }
          tcfg = want;
        }
        targs.N = targsF.N = std::max(nmax, 1);
      }
      // K-split of GEMM-B: only when its output tiles cannot fill the SMs and the contraction is long
      int ksB = 1;
      if (ksplit_ok) {
        const int64_t mt = ceil_div((int64_t)r, (int64_t)tileB.BM);
        int64_t ctas = 0;
        for (int g = 0; g < G; ++g) ctas += mt * ceil_div((int64_t)bound[g], (int64_t)tileB.BN);
        const int64_t sm = 148;   // B200
        // FP64 kernel: two resident CTAs per SM at least
        if (ctas > 0 && 4 * ctas < 3 * sm) ksB = (int)std::min<int64_t>({(int64_t)KSPLIT_MAX, 2 * sm / ctas, (int64_t)n / 2048});
        ksB = std::max(ksB, 1);
      }
      argsB.ksplit = ksB;
      // The delta forms pay while the batch is wide; the narrow tail is latency-bound either way and its slow
      // columns converge in fewer iterations on exact contractions, so it runs all-FP64 (the live set only
      // shrinks within a round, and every round starts with an exact iteration).
      const bool dz_on = delta && ntot > dmin, df_on = delta_f && ntot > dmin;
      const int ce = (dz_on && ntot >= 4 * (int64_t)dmin) ? ce_max : check_every;   // iterations of this batch
      ce_of[ring] = ce;
      for (int k = 0; k < ce; ++k) {
        // FP64 GEMM-B: always without the delta form; with it, on the first iteration of a round (no zeta yet)
        // and on the last iteration of every batch, whose exact rho carries the stop test before the compaction
        const bool exact_it = !dz_on || (batch == 0 && k == 0) || k == ce - 1;
        // sampled launches: right after a compaction every slot is live, so the counted flops are all useful; the
        // delta form has its FP64 GEMM-B on the last iteration of the batch instead
        // first iteration after a compaction (every slot live) and, in the delta forms, the exact last iteration
        const int sidx = !opts->profile ? -1 : (opts->profile == 2 ? k : (k == 0 ? 0 : ((dz_on && k == ce - 1) ? 1 : -1)));
        if (k == 0) std::fill(samp_kind.begin() + (size_t)ring * nsamp * 2, samp_kind.begin() + (size_t)(ring + 1) * nsamp * 2, -1);
        int* sk = samp_kind.data() + ((size_t)ring * nsamp + std::max(sidx, 0)) * 2;
        int famA = 0, famB = 0;
        if (sidx >= 0) TKM_CUDA(cudaEventRecord(pev(ring, sidx, 0), st));
        int nblkA = (int)ceil_div(n, tileA.BM);
        if (df_on && !exact_it) {
          // F half: the product U Lam da on the tcgen05 tensor cores, then F+ = Fbar - U Lam da with the loss
          // derivative as an elementwise pass over all (slot, sample)
          ProdEpi pa{prodA.as<float>(), ldn32, B};
          TKM_TRY(gemm_tf32_launch(targsF, G, tsc, pa, st));
          if (sidx >= 0) TKM_CUDA(cudaEventRecord(pev(ring, sidx, 1), st));   // the contraction alone is the sampled span
          FLossArgs fa{(const double*)y, d_fold.as<int32_t>(), nslots.as<int32_t>(), col_of_slot.as<int32_t>(),
                       bbar.as<double>(), mu.as<double>(), p0->col_nc.as<double>(), p0->col_tau.as<double>(),
                       p0->col_v.as<int32_t>(), B, (int)loss, (int)n, smooth, smooth > 0.0 ? 1.0 / (2.0 * smooth) : 0.0,
                       prodA.as<float>(), ldn32, Fb.as<double>(), Fp.as<double>(), Zt.as<double>(), ldn,
                       dz_hi.as<float>(), dz_lo.as<float>(), ldn32, gpart.as<double>(), ldpart, dz_blk_rows};
          nblkA = (int)ceil_div(n, FLOSS_THREADS * FLOSS_EPT);
          floss_kernel<<<dim3((unsigned)std::max(nmax, 1), (unsigned)nblkA, (unsigned)G), FLOSS_THREADS, 0, st>>>(fa);
          TKM_LAUNCH_CHECK();
          famA = 2;
        } else {
          LossEpi le{(const double*)y, d_fold.as<int32_t>(), col_of_slot.as<int32_t>(), bbar.as<double>(),
                     p0->col_nc.as<double>(), p0->col_tau.as<double>(), p0->col_v.as<int32_t>(), B, (int)loss, smooth,
                     Zt.as<double>(), ldn, gpart.as<double>(), ldpart, dz_on ? dz_hi.as<float>() : nullptr,
                     dz_on ? dz_lo.as<float>() : nullptr, ldn32, df_on ? Fb.as<double>() : nullptr, dz_blk_rows};
          TKM_TRY(gemm_f64_launch(argsA, tileA, G, le, st));
          if (df_on) {   // exact iteration of the F half: also F = U Lam a, so that both recurrence states are exact
            // (shifting the old F by the correction of Fbar instead was tried: the drift it leaves in F - F_prev is
            // amplified by the momentum and tripled the iteration counts)
            StoreEpi fs{Fp.as<double>(), ldn, (int64_t)B * ldn, 1.0};   // its time counts for family 0
            TKM_TRY(gemm_f64_launch(argsA2, tileA, G, fs, st));
          }
        }
        if (sidx >= 0) {
          if (famA == 0) TKM_CUDA(cudaEventRecord(pev(ring, sidx, 1), st));
          sk[0] = famA + ((df_on && exact_it) ? 8 : 0);   // + 8: the timed span holds two FP64 GEMM-A launches
          TKM_CUDA(cudaEventRecord(pev(ring, sidx, 2), st));
        }
        if (exact_it) {
          // FP64 contraction; in delta form it also re-establishes zeta = U^T z exactly
          SpecEpi se{col_of_slot.as<int32_t>(), p0->col_lam.as<double>(), B, Abar.as<double>(), ldr, Rho.as<double>(),
                     dz_on ? Zeta.as<double>() : nullptr};
          if (ksB > 1) {
            PartEpi pe{B, ksB, ldr, split_stride, zpart.as<double>()};
            TKM_TRY(gemm_f64_launch(argsB, tileB, G, pe, st));
            spec_finalize_kernel<<<dim3((unsigned)ceil_div(r, 256), (unsigned)std::max(nmax, 1), (unsigned)G), 256, 0, st>>>(
                zpart.as<double>(), ksB, split_stride, nslots.as<int32_t>(), col_of_slot.as<int32_t>(),
                p0->col_lam.as<double>(), B, (int)r, ldr, Abar.as<double>(), dz_on ? Zeta.as<double>() : nullptr, 0,
                Rho.as<double>());
            TKM_LAUNCH_CHECK();
          } else {
            TKM_TRY(gemm_f64_launch(argsB, tileB, G, se, st));
          }
        } else {
          // delta form: the product U^T dz on the tcgen05 tensor cores; zeta += product and rho in update_kernel
          ProdEpi pb{prodB.as<float>(), ldr32, B};
          TKM_TRY(gemm_tf32_launch(targs, G, tsc, pb, st));
        }
        famB = exact_it ? 1 : 3;
        if (sidx >= 0) {
          TKM_CUDA(cudaEventRecord(pev(ring, sidx, 3), st));
          sk[1] = famB;
        }
        UpdateArgs ua{(int)r, (int)n, B, nblkA, restart, maxit, exact_it ? 1 : 0, ldr,
                      ldpart, rtol, gp, nslots.as<int32_t>(), col_of_slot.as<int32_t>(), p0->col_lam.as<double>(),
                      col_c.as<double>(), p0->col_nc.as<double>(), col_s.as<double>(), gpart.as<double>(),
                      Rho.as<double>(), A.as<double>(), Aprev.as<double>(),
                      Abar.as<double>(), beta.as<double>(), beta_prev.as<double>(), bbar.as<double>(), rk.as<double>(),
                      kkt.as<double>(), done.as<int32_t>(), iters.as<int32_t>(), iters_round.as<int32_t>(),
                      flags.as<int32_t>(), df_on ? da_hi.as<float>() : nullptr, df_on ? da_lo.as<float>() : nullptr,
                      ldr32, df_on ? mu.as<double>() : nullptr,
                      exact_it ? nullptr : prodB.as<float>(), ldr32, Zeta.as<double>(), Rho.as<double>(),
                      opts->profile == 2 ? fam_cnt.as<unsigned long long>() : nullptr, famA, famB};
        update_kernel<<<dim3(std::max(nmax, 1), G), 256, 0, st>>>(ua);
        TKM_LAUNCH_CHECK();
      }
      // compaction on the device; the new counts travel back asynchronously
      CompactArgs ca{B, (int)r, ldr, gp, nslots.as<int32_t>(), col_of_slot.as<int32_t>(), done.as<int32_t>(),
                     fin_list.as<int32_t>(), tail_list.as<int32_t>(), counts.as<int32_t>(), A.as<double>(),
                     Aprev.as<double>(), Abar.as<double>(), dz_on ? Zeta.as<double>() : nullptr,
                     dz_on ? Zt.as<double>() : nullptr, ldn, (int)n, df_on ? Fb.as<double>() : nullptr,
                     df_on ? Fp.as<double>() : nullptr, df_on ? da_hi.as<float>() : nullptr,
                     df_on ? da_lo.as<float>() : nullptr, ldr32};
      compact_plan_kernel<<<G, 1024, 0, st>>>(ca);
      TKM_LAUNCH_CHECK();
      compact_apply_kernel<<<dim3(std::max(nmax, 1), G), 256, 0, st>>>(ca);
      TKM_LAUNCH_CHECK();
      TKM_CUDA(cudaMemcpyAsync(h_ns.as<int32_t>() + ring * GEMM_MAX_GROUPS, nslots.p, GEMM_MAX_GROUPS * sizeof(int32_t),
                               cudaMemcpyDeviceToHost, st));
      TKM_CUDA(cudaEventRecord(ev.poll[ring], st));
      // Read back the polls of EARLIER batches while the GPU works on the ones just enqueued.  The host runs
      // one batch ahead while the live set is wide (fresh counts matter for the tile choice) and up to three
      // once it is narrow (batches of ~1 ms: slack against a descheduled host thread matters more).
      const int lag = ntot > 256 ? 2 : POLL_RING - 2;
      while (!finished && done_polls + lag <= batch) {
        const int64_t b = done_polls;
        const int cur = (int)(b % POLL_RING);
        TKM_CUDA(cudaEventSynchronize(ev.poll[cur]));
        const int32_t* hn = h_ns.as<int32_t>() + cur * GEMM_MAX_GROUPS;
        int live = 0;
        for (int g = 0; g < G; ++g) {
          bound[g] = hn[g];
          live += hn[g];
        }
        // live columns during batch b = the counts after the compaction of batch b-1 (all columns for b = 0)
        int live_then = GB, max_then = B;
        if (b >= 1) {
          const int32_t* h1 = h_ns.as<int32_t>() + (int)((b - 1) % POLL_RING) * GEMM_MAX_GROUPS;
          live_then = max_then = 0;
          for (int g = 0; g < G; ++g) {
            live_then += h1[g];
            max_then = std::max(max_then, h1[g]);
          }
        }
        if (opts->profile && live_then > 0) {
          // the sampled launches of batch b precede its poll event; flops = 2 n r (live columns) per launch
          for (int q = 0; q < 2 * nsamp; ++q) {
            int kind = samp_kind[(size_t)cur * nsamp * 2 + q];
            if (kind < 0) continue;
            const int twice = kind >= 8 ? 2 : 1;   // kernel roofline: both launches of the span did 2 n r live flops
            kind &= 7;
            float ms = 0.f;
            TKM_CUDA(cudaEventElapsedTime(&ms, pev(cur, q >> 1, 2 * (q & 1)), pev(cur, q >> 1, 2 * (q & 1) + 1)));
            prof_ms[kind] += ms;
            prof_flops[kind] += twice * 2.0 * (double)live_then * (double)n * (double)r;   // profile == 2: replaced below
            prof_launches[kind] += twice;
          }
        }
        if (trace && b >= 1) {
          float bms = 0.f;
          cudaEventElapsedTime(&bms, ev.poll[(b - 1) % POLL_RING], ev.poll[cur]);
          fprintf(trace, "%d %lld %d %d %d %d %.4f %d\n", rnd, (long long)b, live_then, max_then, tileA.cfg, tileB.cfg, bms,
                  ce_of[cur]);
        }
        ++done_polls;
        if (live == 0) finished = true;   // batches already enqueued beyond b find no live slot and do nothing
      }
      ++batch;
    }
    return TKM_OK;
  };

  // Smoothing schedule (S8).  gap_tol <= 0: the fixed schedule of reading G7.  gap_tol > 0: the
  // outer control of reading G23 -- after round k < R-1 a column whose iterate certifies a duality gap of the
  // non-smoothed problem <= gap_tol is finished at THIS level to `tol` (when the round stopped at warm_tol), tested
  // again on the converged point and, if certified, leaves the schedule with that level's minimiser.
  const bool outer = smoothed && rounds > 1 && opts->gap_tol > 0.0;
  DevBuf onsched, passed, level, d_gapP, d_gapV;
  if (smoothed) {
    TKM_TRY(level.alloc((size_t)GB * sizeof(int32_t), false, st, true));
    std::vector<int32_t> h_lv(GB, rounds - 1);
    TKM_CUDA(cudaMemcpyAsync(level.p, h_lv.data(), GB * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    TKM_CUDA(cudaStreamSynchronize(st));   // h_lv is a local
  }
  if (outer) {
    TKM_TRY(onsched.alloc((size_t)GB * sizeof(int32_t), false, st, true));
    TKM_TRY(passed.alloc((size_t)GB * sizeof(int32_t), true, st, true));
    TKM_TRY(d_gapP.alloc((size_t)GB * sizeof(double), false, st, true));
    TKM_TRY(d_gapV.alloc((size_t)GB * sizeof(double), false, st, true));
    TKM_CUDA(cudaMemsetAsync(onsched.p, 0x01, (size_t)GB * sizeof(int32_t), st));   // any non-zero value = on the schedule
  }
  auto gap_pass = [&](double smooth) -> int {   // d_gapV[gc] = gap of column gc at (a_out, beta) for level `smooth`
    for (int g = 0; g < G; ++g)
      TKM_TRY(path_gap_device(out[g], (const double*)y, d_fold.as<int32_t>(), beta.as<double>() + (size_t)g * B, smooth,
                              nullptr, d_gapP.as<double>() + (size_t)g * B, d_gapV.as<double>() + (size_t)g * B, st));
    return TKM_OK;
  };
  auto control = [&](int mode, int rnd) -> int {
    outer_control_kernel<<<(unsigned)ceil_div(GB, 256), 256, 0, st>>>(mode, GB, opts->gap_tol, rnd, d_gapV.as<double>(),
                                                                     onsched.as<int32_t>(), passed.as<int32_t>(),
                                                                     level.as<int32_t>(), flags.as<int32_t>());
    TKM_LAUNCH_CHECK();
    return TKM_OK;
  };
  double smooth = opts->smooth0;
  for (int rnd = 0; rnd < rounds; ++rnd) {
    if (smoothed && rnd > 0) smooth *= opts->eta;   // PAPER.md:220 (Alg.1 l.22)
    const bool last = rnd + 1 == rounds;
    const double rtol = (!last && opts->warm_tol > 0.0) ? opts->warm_tol : tol;
    TKM_TRY(run_round(rnd, smooth, rtol, outer ? onsched.as<int32_t>() : nullptr));
    if (!outer) continue;
    TKM_TRY(gap_pass(smooth));
    if (last) {
      TKM_TRY(control(2, rnd));
      break;
    }
    TKM_TRY(control(0, rnd));
    if (rtol > tol) {   // the warm iterate only screens
      TKM_TRY(run_round(rnd, smooth, tol, passed.as<int32_t>()));
      TKM_TRY(gap_pass(smooth));
    }
    TKM_TRY(control(1, rnd));
  }
  // results: beta0 per group, diagnostics to the host
  std::vector<double> hb(GB), hk(GB);
  std::vector<int32_t> hi(GB), hf(GB), hl(GB, 0);
  if (smoothed) TKM_CUDA(cudaMemcpyAsync(hl.data(), level.p, GB * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  for (int g = 0; g < G; ++g)
    TKM_CUDA(cudaMemcpyAsync(out[g]->beta0.p, beta.as<double>() + (size_t)g * B, (size_t)B * sizeof(double),
                             cudaMemcpyDeviceToDevice, st));
  TKM_CUDA(cudaMemcpyAsync(hb.data(), beta.p, GB * sizeof(double), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaMemcpyAsync(hk.data(), kkt.p, GB * sizeof(double), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaMemcpyAsync(hi.data(), iters.p, GB * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaMemcpyAsync(hf.data(), flags.p, GB * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  unsigned long long h_fam[4] = {0, 0, 0, 0};
  if (opts->profile == 2) TKM_CUDA(cudaMemcpyAsync(h_fam, fam_cnt.p, sizeof(h_fam), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaStreamSynchronize(st));
  if (opts->profile == 2)   // every launch was timed: the useful work is what the device counted, column by column
    for (int q = 0; q < 4; ++q) prof_flops[q] = 2.0 * (double)n * (double)r * (double)h_fam[q];
  bool notconv = false;
  for (int g = 0; g < G; ++g) {
    tkm_path* p = out[g];
    p->smooth_final = smoothed ? smooth : 0.0;
    p->h_beta0.assign(hb.begin() + (size_t)g * B, hb.begin() + (size_t)(g + 1) * B);
    p->h_kkt.assign(hk.begin() + (size_t)g * B, hk.begin() + (size_t)(g + 1) * B);
    p->h_iters.assign(hi.begin() + (size_t)g * B, hi.begin() + (size_t)(g + 1) * B);
    p->h_flags.assign(hf.begin() + (size_t)g * B, hf.begin() + (size_t)(g + 1) * B);
    p->h_level.assign(hl.begin() + (size_t)g * B, hl.begin() + (size_t)(g + 1) * B);
    p->h_smooth.assign(B, 0.0);
    if (smoothed) {
      for (int c = 0; c < B; ++c) p->h_smooth[c] = opts->smooth0 * std::pow(opts->eta, (double)p->h_level[c]);
      TKM_TRY(p->col_smooth.alloc((size_t)B * sizeof(double), false, st));
      TKM_CUDA(cudaMemcpy(p->col_smooth.p, p->h_smooth.data(), (size_t)B * sizeof(double), cudaMemcpyHostToDevice));
    }
    p->total_col_iters = 0;
    for (int c = 0; c < B; ++c) {
      p->total_col_iters += p->h_iters[c];
      notconv |= (p->h_flags[c] & 1) != 0;
    }
  }
  // sampled timings cover all groups of the shared launches: reported on the first path
  for (int q = 0; q < 4; ++q) {
    out[0]->prof_ms[q] = prof_ms[q];
    out[0]->prof_flops[q] = prof_flops[q];
    out[0]->prof_launches[q] = prof_launches[q];
  }
  guard.armed = false;
  if (notconv) return set_error(TKM_ENOTCONV, "tkm_fit_path: some columns hit maxit (see flags)");
  return TKM_OK;
}

extern "C" int tkm_fit_path(const tkm_spectral* s, const void* y, tkm_loss loss, const tkm_loss_opts* opts,
                            const double* lambdas, int32_t L, const int32_t* foldid, int32_t V, double tol,
                            int32_t maxit, const tkm_path* warm, tkm_path** out, void* stream) {
  if (!out) return set_error(TKM_EINVAL, "tkm_fit_path: out is NULL");
  *out = nullptr;
  if (!s) return set_error(TKM_EINVAL, "tkm_fit_path: NULL argument");
  return tkm_fit_path_multi(&s, 1, y, loss, opts, lambdas, L, foldid, V, tol, maxit, warm ? &warm : nullptr, out, stream);
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

extern "C" int tkm_path_shape(const tkm_path* p, int32_t* T, int32_t* L, int32_t* V, int64_t* n) {
  if (!p) return set_error(TKM_EINVAL, "tkm_path_shape: NULL handle");
  if (T) *T = p->T;
  if (L) *L = p->L;
  if (V) *V = p->V;
  if (n) *n = p->spec->n;
  return TKM_OK;
}

extern "C" int tkm_path_levels(const tkm_path* p, int32_t* level, double* smooth) {
  if (!p) return set_error(TKM_EINVAL, "tkm_path_levels: NULL handle");
  if (level) memcpy(level, p->h_level.data(), p->B * sizeof(int32_t));
  if (smooth) memcpy(smooth, p->h_smooth.data(), p->B * sizeof(double));
  return TKM_OK;
}

extern "C" int tkm_path_profile(const tkm_path* p, double* ms, double* flops, int64_t* launches) {
  if (!p) return set_error(TKM_EINVAL, "tkm_path_profile: NULL handle");
  for (int q = 0; q < 4; ++q) {
    if (ms) ms[q] = p->prof_ms[q];
    if (flops) flops[q] = p->prof_flops[q];
    if (launches) launches[q] = p->prof_launches[q];
  }
  return TKM_OK;
}

extern "C" int tkm_path_get_a(const tkm_path* p, double* a_out, void* stream) {
  if (!p || !a_out) return set_error(TKM_EINVAL, "tkm_path_get_a: NULL argument");
  const int64_t r = p->spec->r;
  TKM_CUDA(cudaMemcpy2DAsync(a_out, r * sizeof(double), p->a.p, p->spec->ldr * sizeof(double), r * sizeof(double),
                             p->B, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
  return TKM_OK;
}
