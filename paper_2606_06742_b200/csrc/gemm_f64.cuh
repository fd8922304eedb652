// gemm_f64.cuh -- FP64 tensor-core (DMMA.8x8x4) GEMM with fused epilogues for the sweep.
//
// Computes Dt[N][M] = P[N][K] * Q[M][K]^T  ("NT": both operands K-contiguous).
//   GEMM-A of the sweep:  P = abar (slots x r),  Q = U*Lam (n x r)  -> F^T (slots x n)
//   GEMM-B of the sweep (S6):                 P = Z^T  (slots x n),  Q = U^T   (r x n)  -> zeta^T (slots x r)
// The moving operand is stored one column of the paper's (lambda, fold) batch per ROW, so that a
// column's vector is contiguous (per-column reductions and compaction are row operations).
//
// The MMA "A" operand (row-major 8x4) is a P fragment, the MMA "B" operand (col-major 4x8) is a Q
// fragment, so the accumulator fragment of lane l holds Dt[n0 + l/4][m0 + 2(l%4) + {0,1}]: two
// consecutive m, i.e. 16-byte stores along the contiguous output dimension.
//
// Pipeline: STAGES-deep cp.async ring, one __syncthreads per K-step of 16.  Requirements checked by
// the host wrappers: P, Q 16-byte aligned and ldp, ldq even (16-byte row alignment).  Rows beyond
// N / M and the K tail are zero-filled through the cp.async src-size operand, so no padding of the
// operands is read.
#pragma once

#include "common.cuh"

namespace tkm {

constexpr int GEMM_BK = 16;            // K-step in doubles (128 bytes per row)
constexpr int GEMM_LDS = GEMM_BK + 4;  // padded smem row: (20 mod 16) = 4 => conflict-free LDS.64

struct GemmOperands {
  const double* P;
  int64_t ldp;
  const double* Q;
  int64_t ldq;
  int N, M, K;
};

template <int BN, int BM, int WARPS_N, int WARPS_M, int STAGES, class Epi>
__global__ void __launch_bounds__(WARPS_N* WARPS_M * 32)
    gemm_f64_nt_kernel(const GemmOperands g, const Epi epi) {
  constexpr int NT = WARPS_N * WARPS_M * 32;
  constexpr int WN = BN / WARPS_N, WM = BM / WARPS_M;
  constexpr int TN = WN / 8, TM = WM / 8;
  static_assert(WN % 8 == 0 && WM % 8 == 0, "warp tile must be a multiple of the 8x8 MMA tile");
  extern __shared__ __align__(16) double smem[];
  double* Ps = smem;                                   // [STAGES][BN][GEMM_LDS]
  double* Qs = smem + (size_t)STAGES * BN * GEMM_LDS;   // [STAGES][BM][GEMM_LDS]

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int warp_n = warp / WARPS_M, warp_m = warp % WARPS_M;
  const int m_blk0 = blockIdx.x * BM, n_blk0 = blockIdx.y * BN;
  if (n_blk0 >= g.N) return;   // grid may be sized for more slots than are still active
  const int KT = (g.K + GEMM_BK - 1) / GEMM_BK;

  auto load_stage = [&](int stage, int kt) {
    const int k0 = kt * GEMM_BK;
    double* ps = Ps + (size_t)stage * BN * GEMM_LDS;
    double* qs = Qs + (size_t)stage * BM * GEMM_LDS;
#pragma unroll
    for (int id = tid; id < BN * 8; id += NT) {
      const int row = id >> 3, ch = id & 7;
      const int kk = k0 + ch * 2;
      const int nb = ((n_blk0 + row) < g.N) ? min(max(g.K - kk, 0), 2) * 8 : 0;
      const double* src = nb ? g.P + (int64_t)(n_blk0 + row) * g.ldp + kk : g.P;
      cp_async_16(ps + row * GEMM_LDS + ch * 2, src, nb);
    }
#pragma unroll
    for (int id = tid; id < BM * 8; id += NT) {
      const int row = id >> 3, ch = id & 7;
      const int kk = k0 + ch * 2;
      const int nb = ((m_blk0 + row) < g.M) ? min(max(g.K - kk, 0), 2) * 8 : 0;
      const double* src = nb ? g.Q + (int64_t)(m_blk0 + row) * g.ldq + kk : g.Q;
      cp_async_16(qs + row * GEMM_LDS + ch * 2, src, nb);
    }
  };

  double acc[TN][TM][2];
#pragma unroll
  for (int i = 0; i < TN; ++i)
#pragma unroll
    for (int j = 0; j < TM; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

#pragma unroll
  for (int s = 0; s < STAGES - 1; ++s) {
    if (s < KT) load_stage(s, s);
    cp_async_commit();
  }

  const int frag_row = lane >> 2, frag_k = lane & 3;
  for (int kt = 0; kt < KT; ++kt) {
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    {
      const int nk = kt + STAGES - 1;
      if (nk < KT) load_stage(nk % STAGES, nk);
      cp_async_commit();
    }
    const double* ps = Ps + (size_t)(kt % STAGES) * BN * GEMM_LDS + (warp_n * WN + frag_row) * GEMM_LDS + frag_k;
    const double* qs = Qs + (size_t)(kt % STAGES) * BM * GEMM_LDS + (warp_m * WM + frag_row) * GEMM_LDS + frag_k;
#pragma unroll
    for (int kk = 0; kk < GEMM_BK; kk += 4) {
      double a[TN], b[TM];
#pragma unroll
      for (int i = 0; i < TN; ++i) a[i] = ps[i * 8 * GEMM_LDS + kk];
#pragma unroll
      for (int j = 0; j < TM; ++j) b[j] = qs[j * 8 * GEMM_LDS + kk];
#pragma unroll
      for (int i = 0; i < TN; ++i)
#pragma unroll
        for (int j = 0; j < TM; ++j) dmma_884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
    }
  }
  cp_async_wait<0>();
  __syncthreads();   // pipeline smem is now free: epilogues may use it as reduction scratch

  epi.template run<BN, BM, WARPS_N, WARPS_M, TN, TM>(acc, n_blk0, m_blk0, warp_n, warp_m, lane, g.N, g.M, smem);
}

template <int BN, int BM, int STAGES>
constexpr size_t gemm_f64_smem_bytes() {
  return (size_t)STAGES * (BN + BM) * GEMM_LDS * sizeof(double);
}

// Per-CTA deterministic column reduction helper used by the epilogues: `v[TN]` holds, per thread, a
// partial sum for the TN slot-rows n = n_blk0 + warp_n*WN + i*8 + lane/4.  Reduces over the quad
// (the 4 lanes sharing a row) and over the WARPS_M warps, then thread n_local < BN returns the CTA
// total for row n_local in `out` (valid only when the function returns true).
template <int BN, int WARPS_N, int WARPS_M, int TN>
__device__ __forceinline__ bool cta_row_reduce(double (&v)[TN], int warp_n, int warp_m, int lane,
                                               double* scratch, double& out) {
  constexpr int WN = BN / WARPS_N;
#pragma unroll
  for (int i = 0; i < TN; ++i) {
    v[i] += __shfl_xor_sync(0xffffffffu, v[i], 1);
    v[i] += __shfl_xor_sync(0xffffffffu, v[i], 2);
  }
  if ((lane & 3) == 0) {
#pragma unroll
    for (int i = 0; i < TN; ++i) scratch[warp_m * BN + warp_n * WN + i * 8 + (lane >> 2)] = v[i];
  }
  __syncthreads();
  const int t = threadIdx.x;
  bool have = t < BN;
  if (have) {
    double s = 0.0;
#pragma unroll
    for (int w = 0; w < WARPS_M; ++w) s += scratch[w * BN + t];
    out = s;
  }
  __syncthreads();   // scratch may be reused by the caller
  return have;
}

// ---- epilogue: plain store --------------------------------------------------------------------
struct StoreEpi {
  double* Dt;
  int64_t ldd;
  double alpha;   // Dt = alpha * acc
  template <int BN, int BM, int WARPS_N, int WARPS_M, int TN, int TM>
  __device__ __forceinline__ void run(double (&acc)[TN][TM][2], int n_blk0, int m_blk0, int warp_n,
                                      int warp_m, int lane, int N, int M, double*) const {
    constexpr int WN = BN / WARPS_N, WM = BM / WARPS_M;
#pragma unroll
    for (int i = 0; i < TN; ++i) {
      const int n = n_blk0 + warp_n * WN + i * 8 + (lane >> 2);
      if (n >= N) continue;
#pragma unroll
      for (int j = 0; j < TM; ++j) {
        const int m = m_blk0 + warp_m * WM + j * 8 + 2 * (lane & 3);
        double* d = Dt + (int64_t)n * ldd + m;
        if (m + 1 < M) {
          *reinterpret_cast<double2*>(d) = make_double2(alpha * acc[i][j][0], alpha * acc[i][j][1]);
        } else if (m < M) {
          d[0] = alpha * acc[i][j][0];
        }
      }
    }
  }
};

template <int BN, int BM, int WARPS_N, int WARPS_M, int STAGES, class Epi>
int launch_gemm_f64(const GemmOperands& g, const Epi& epi, cudaStream_t st) {
  auto kern = gemm_f64_nt_kernel<BN, BM, WARPS_N, WARPS_M, STAGES, Epi>;
  constexpr size_t smem = gemm_f64_smem_bytes<BN, BM, STAGES>();
  static bool configured = false;   // per template instantiation
  if (!configured) {
    TKM_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    configured = true;
  }
  dim3 grid((unsigned)ceil_div(g.M, BM), (unsigned)ceil_div(g.N, BN));
  kern<<<grid, WARPS_N * WARPS_M * 32, smem, st>>>(g, epi);
  TKM_LAUNCH_CHECK();
  return TKM_OK;
}

// Shape-based tile choice shared by all FP64 GEMM call sites.  The grid is (M tiles, N tiles); pick
// the largest tile whose CTA count still covers the 148 SMs about twice, else the smallest.
// gemm_f64_tile_bm() returns the BM of that choice (callers size per-M-block partial arrays by it).
inline int gemm_f64_config(int64_t N, int64_t M) {
  const int64_t t128 = ceil_div(M, 128) * ceil_div(N, 64);
  if (t128 >= 2 * 148) return 2;
  const int64_t t64 = ceil_div(M, 64) * ceil_div(N, 64);
  if (t64 >= 148 + 74) return 1;
  return 0;
}
inline int gemm_f64_tile_bm(int64_t N, int64_t M) { return gemm_f64_config(N, M) == 2 ? 128 : 64; }

template <class Epi>
int gemm_f64_dispatch(const GemmOperands& g, const Epi& epi, cudaStream_t st) {
  switch (gemm_f64_config(g.N, g.M)) {
    case 2: return launch_gemm_f64<64, 128, 2, 2, 3>(g, epi, st);
    case 1: return launch_gemm_f64<64, 64, 2, 2, 3>(g, epi, st);
    default: return launch_gemm_f64<32, 64, 1, 4, 4>(g, epi, st);
  }
}

}  // namespace tkm
