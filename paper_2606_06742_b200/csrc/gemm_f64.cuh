// gemm_f64.cuh -- FP64 tensor-core (DMMA.8x8x4) GEMM with fused epilogues: the two contractions of the
// sweep, the exact-CV scoring pass (S9) and the Nystrom setup products.
//
// Computes, for every group g < G (independent problems sharing one launch, e.g. the bandwidths of a
// sigma grid),   Dt_g[N_g][M] = P_g[N_g][K] * Q_g[M][K]^T   ("NT": both operands K-contiguous).
//   GEMM-A (S5):  P = Lam*abar (slots x r),  Q = U   ... stored as U*Lam (n x r)  -> F^T    (slots x n)
//   GEMM-B (S6):  P = Z^T      (slots x n),  Q = U^T (r x n)                      -> zeta^T (slots x r)
// The moving operand P holds one column of the paper's (lambda, fold) batch per ROW ("slot"); the
// groups' P matrices are stacked: row g * p_group_rows + slot of one array.  N_g (live slots) is read
// from device memory so that the host never has to synchronise to launch the next iteration.
//
// Blackwell mapping: tcgen05 has no FP64 kind, so the math is mma.sync m8n8k4 f64 (DMMA).  Operand
// tiles are staged by TMA (cp.async.bulk.tensor, 128-byte swizzle, box = rows x 16 doubles) into a
// STAGES-deep ring guarded by full/empty mbarriers; one producer warp issues the loads, WN x WM
// consumer warps run the MMAs and never meet at a CTA-wide barrier inside the K loop.
//
// Fragment addressing: with the 128-byte swizzle a tile row is 8 chunks of 16 B, chunk c of row R
// stored at chunk c ^ (R & 7).  The MMA k-slot j = lane & 3 of sub-step s is mapped to
// k = 8 (j >> 1) + 2 s + (j & 1)  (any bijection of the 16 k of a stage is a valid summation order,
// as long as both operands use the same one); then the 16 lanes of a half-warp touch 16 distinct
// 8-byte bank pairs -> conflict-free LDS.64 for both operands.
//
// Accumulator fragment of lane l: Dt[n0 + l/4][m0 + 2 (l%4) + {0,1}] per 8x8 sub-tile.
#pragma once

#include "tma.cuh"

namespace tkm {

constexpr int GEMM_MAX_GROUPS = 8;
constexpr int GEMM_ROW_BYTES = TMA_BOX_K * 8;   // 128

struct GemmArgs {
  CUtensorMap p_map;                    // [G * p_group_rows][K], box = BN x 16
  CUtensorMap q_map[GEMM_MAX_GROUPS];   // per group [M][K], box = BM x 16
  const int32_t* nslots;                // [G] device, live rows of each group; NULL => N for all
  int p_group_rows;                     // row offset between consecutive groups in P
  int N, M, K;                          // N: upper bound of the live rows (the grid covers it)
  int ksplit;                           // <= 1: one CTA contracts all of K; S > 1: blockIdx.x = split * n_tiles + n_tile,
                                        // split s contracts K-tiles [s KT/S, (s+1) KT/S) and the epilogue sees a partial sum
  int q_blk_rows;                       // 0: Q_g row-major [M][K]; > 0: Q_g K-blocked [K/16][q_blk_rows][16] (map over
                                        // [(K/16) q_blk_rows][16]): a stage's Q tile is one contiguous read (thin U, K = n large)
};

// K-split index of this CTA, for epilogues that store partial sums (ksplit as in GemmArgs / Tf32Args)
__device__ __forceinline__ int gemm_split_index(int ksplit) { return ksplit > 1 ? (int)(blockIdx.x / (gridDim.x / ksplit)) : 0; }
// Grid: x = (K-split, slot tile) -- fastest, so that the CTAs that share a Q tile (the same rows of U) are
// scheduled together and the tile is read from HBM once (ncu at n = 20000, 900 slots, with x = row tile: 48 GB of
// DRAM reads per launch against 3.3 GB algorithmic); y = row tile of the output (index of the per-tile partial sums
// the epilogues write); z = group.
__device__ __forceinline__ int gemm_m_block() { return (int)blockIdx.y; }

template <int TN_, int WN_, int TM_, int WM_, int STAGES_>
struct GemmCfg {
  static constexpr int TN = TN_, WN = WN_, TM = TM_, WM = WM_, STAGES = STAGES_;
  static constexpr int BN = TN * WN * 8, BM = TM * WM * 8;
  static constexpr int CONSUMERS = WN * WM * 32;
  static constexpr int THREADS = CONSUMERS + 32;
  static constexpr int STAGE_BYTES = (BN + BM) * GEMM_ROW_BYTES;
  static constexpr size_t SMEM = (size_t)STAGES * STAGE_BYTES + 1024;   // + alignment slack
  static_assert(BN <= 256 && BM <= 256, "TMA box dimension limit");
  static_assert(BN <= CONSUMERS, "epilogue row reductions assign one thread per tile row");
};

// consumer-only barrier (the producer warp has left the CTA-wide flow)
template <int COUNT>
__device__ __forceinline__ void consumer_sync() {
  asm volatile("bar.sync 1, %0;\n" ::"n"(COUNT) : "memory");
}

// Fragment load from a pipeline stage: an explicit shared-space load.  The stage base is an integer-aligned
// address, so a plain C++ dereference compiled to GENERIC loads (LD.E), whose reads of shared memory are not
// ordered with the mbarrier.arrive that hands the stage back to the TMA producer: with a starved ring (first wave of
// a launch on freshly mapped operands, two CTAs per SM) the refill of K-tile kt + STAGES landed before the last
// loads of K-tile kt had read the stage -- four elements of one fragment row wrong in a few hundred outputs per launch
// (found at n = 581 012 in the streamed Nystrom set-up; profiles/r02_host_stalls.md, second part).  LDS goes
// through the same in-order shared-memory pipe as the arrive; `volatile` keeps the loads between the wait and the
// arrive in program order.
__device__ __forceinline__ double lds_f64(uint32_t saddr) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];\n" : "=d"(v) : "r"(saddr));
  return v;
}

// K loop of one consumer warp with exactly NV live 8-row sub-tiles (compile time).
template <class Cfg, int NV>
__device__ __forceinline__ void gemm_k_body(double (&acc)[Cfg::TN][Cfg::TM][2], uint32_t p_base,
                                            uint32_t q_base, const uint32_t (&off)[4], uint64_t* full_bar,
                                            uint64_t* empty_bar, int KT, int lane) {
  constexpr int TM = Cfg::TM, STAGES = Cfg::STAGES;
  // with one or two accumulator tiles per warp the four MMAs of a stage would form one dependent chain:
  // alternate between two accumulator sets and add them at the end
  constexpr bool SPLIT = NV * TM <= 2;
  double acc2[SPLIT ? NV : 1][TM][2];
#pragma unroll
  for (int i = 0; i < (SPLIT ? NV : 1); ++i)
#pragma unroll
    for (int j = 0; j < TM; ++j) acc2[i][j][0] = acc2[i][j][1] = 0.0;
  // A stage is handed back to the producer ONE K-tile late, after the wait for the next tile: every MMA of the
  // finished tile has then issued, so its fragment loads have returned.  Arriving right after the loads were ISSUED
  // is not enough -- nothing orders an in-flight LDS before a later mbarrier.arrive of the same warp, and with a
  // starved ring the TMA refill of K-tile kt + STAGES overtook the last loads of K-tile kt (see lds_f64).
  int s = 0, s_prev = 0;
  uint32_t phase = 0;
  for (int kt = 0; kt < KT; ++kt) {
    mbar_wait(&full_bar[s], phase);
    if (kt > 0) {
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty_bar[s_prev]);
    }
    const uint32_t ps = p_base + (uint32_t)s * Cfg::STAGE_BYTES;   // shared-space byte addresses
    const uint32_t qs = q_base + (uint32_t)s * Cfg::STAGE_BYTES;
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
      double a[NV], b[TM];
#pragma unroll
      for (int j = 0; j < TM; ++j) b[j] = lds_f64(qs + j * 8 * GEMM_ROW_BYTES + off[ks]);
#pragma unroll
      for (int i = 0; i < NV; ++i) a[i] = lds_f64(ps + i * 8 * GEMM_ROW_BYTES + off[ks]);
#pragma unroll
      for (int i = 0; i < NV; ++i)
#pragma unroll
        for (int j = 0; j < TM; ++j) {
          if (SPLIT && (ks & 1))
            dmma_884(acc2[i][j][0], acc2[i][j][1], a[i], b[j]);
          else
            dmma_884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
    }
    s_prev = s;
    if (++s == STAGES) {
      s = 0;
      phase ^= 1;
    }
  }   // the last tile's stage is never refilled: no release needed
  if (SPLIT) {
#pragma unroll
    for (int i = 0; i < NV; ++i)
#pragma unroll
      for (int j = 0; j < TM; ++j) {
        acc[i][j][0] += acc2[i][j][0];
        acc[i][j][1] += acc2[i][j][1];
      }
  }
}
// a warp without live sub-tiles still has to release the stages
template <class Cfg>
__device__ __forceinline__ void gemm_k_idle(uint64_t* full_bar, uint64_t* empty_bar, int KT, int lane) {
  int s = 0;
  uint32_t phase = 0;
  for (int kt = 0; kt < KT; ++kt) {
    mbar_wait(&full_bar[s], phase);
    if (lane == 0) mbar_arrive(&empty_bar[s]);
    if (++s == Cfg::STAGES) {
      s = 0;
      phase ^= 1;
    }
  }
}
template <class Cfg, int NV>
__device__ __forceinline__ void gemm_k_loop(int nv, double (&acc)[Cfg::TN][Cfg::TM][2], uint32_t p_base,
                                            uint32_t q_base, const uint32_t (&off)[4], uint64_t* full_bar,
                                            uint64_t* empty_bar, int KT, int lane) {
  if constexpr (NV == 0) {
    gemm_k_idle<Cfg>(full_bar, empty_bar, KT, lane);
  } else {
    if (nv == NV)
      gemm_k_body<Cfg, NV>(acc, p_base, q_base, off, full_bar, empty_bar, KT, lane);
    else
      gemm_k_loop<Cfg, NV - 1>(nv, acc, p_base, q_base, off, full_bar, empty_bar, KT, lane);
  }
}

template <class Cfg, class Epi>
__global__ void __launch_bounds__(Cfg::THREADS)
    gemm_f64_tma_kernel(const __grid_constant__ GemmArgs g, const Epi epi) {
  constexpr int TN = Cfg::TN, WN = Cfg::WN, TM = Cfg::TM, WM = Cfg::WM, STAGES = Cfg::STAGES;
  constexpr int BN = Cfg::BN, BM = Cfg::BM;
  extern __shared__ uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t full_bar[STAGES];
  __shared__ __align__(8) uint64_t empty_bar[STAGES];
  __shared__ double scratch[WM * BN];

  const int grp = blockIdx.z;
  const int N = g.nslots ? min(g.nslots[grp], g.N) : g.N;
  const int S = max(g.ksplit, 1), ny = (int)gridDim.x / S, split = (int)blockIdx.x / ny;
  const int m_blk0 = blockIdx.y * BM, n_blk0 = ((int)blockIdx.x - split * ny) * BN;
  if (n_blk0 >= N) return;   // the grid is sized for an upper bound of the live slots
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int KT_all = (g.K + TMA_BOX_K - 1) / TMA_BOX_K;
  const int kt0 = (int)((int64_t)split * KT_all / S), KT = (int)((int64_t)(split + 1) * KT_all / S) - kt0;
  uint8_t* tiles = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(&full_bar[s], 1);
      mbar_init(&empty_bar[s], WN * WM);
    }
    mbar_fence_init();
  }
  __syncthreads();

  if (warp == WN * WM) {
    // ===== TMA producer =====
    if (lane == 0) {
      tma_prefetch_desc(&g.p_map);
      tma_prefetch_desc(&g.q_map[grp]);
      const int prow = grp * g.p_group_rows + n_blk0;
      int s = 0;
      uint32_t phase = 1;   // parity of the empty-barrier phase that frees stage s (first pass: no wait)
      for (int kt = 0; kt < KT; ++kt) {
        if (kt >= STAGES) mbar_wait(&empty_bar[s], phase);
        mbar_arrive_expect_tx(&full_bar[s], Cfg::STAGE_BYTES);
        uint8_t* ps = tiles + (size_t)s * Cfg::STAGE_BYTES;
        tma_load_2d(ps, &g.p_map, (kt0 + kt) * TMA_BOX_K, prow, &full_bar[s]);
        if (g.q_blk_rows)
          tma_load_2d(ps + BN * GEMM_ROW_BYTES, &g.q_map[grp], 0, (kt0 + kt) * g.q_blk_rows + m_blk0, &full_bar[s]);
        else
          tma_load_2d(ps + BN * GEMM_ROW_BYTES, &g.q_map[grp], (kt0 + kt) * TMA_BOX_K, m_blk0, &full_bar[s]);
        if (++s == STAGES) {
          s = 0;
          phase ^= 1;
        }
      }
    }
    return;
  }

  // ===== MMA consumers =====
  const int warp_n = warp / WM, warp_m = warp % WM;
  const int fr = lane >> 2, fj = lane & 3;
  // live 8-row sub-tiles of this warp (slots beyond N are neither multiplied nor stored)
  const int nv = min(TN, max(0, (N - (n_blk0 + warp_n * TN * 8) + 7) >> 3));
  uint32_t off[4];   // byte offset inside a 128-byte tile row of this lane's element at sub-step s
#pragma unroll
  for (int s = 0; s < 4; ++s) off[s] = (uint32_t)(((((fj >> 1) << 2) + s) ^ fr) << 4) | (uint32_t)((fj & 1) << 3);
  const uint32_t p_row = (uint32_t)((warp_n * TN * 8 + fr) * GEMM_ROW_BYTES);
  const uint32_t q_row = (uint32_t)(BN * GEMM_ROW_BYTES + (warp_m * TM * 8 + fr) * GEMM_ROW_BYTES);

  double acc[TN][TM][2];
#pragma unroll
  for (int i = 0; i < TN; ++i)
#pragma unroll
    for (int j = 0; j < TM; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  // The K loop is instantiated once per possible number of live sub-tiles so that every MMA and every
  // fragment load is unconditional (a ragged last N tile costs only the sub-tiles it has).
  const uint32_t p_base = smem_u32(tiles) + p_row;
  const uint32_t q_base = smem_u32(tiles) + q_row;
  gemm_k_loop<Cfg, TN>(nv, acc, p_base, q_base, off, full_bar, empty_bar, KT, lane);

  epi.template run<Cfg>(acc, n_blk0, m_blk0, warp_n, warp_m, lane, N, g.M, grp, scratch);
}

// Per-CTA deterministic row reduction used by the epilogues: `v[TN]` holds, per thread, a partial sum
// for the TN slot-rows n = n_blk0 + warp_n*TN*8 + i*8 + lane/4.  Reduces over the quad (the 4 lanes
// sharing a row) and over the WM warps in fixed order; thread t < BN then returns the CTA total of tile
// row t in `out` (valid only when the function returns true).  Consumer threads only.
template <class Cfg>
__device__ __forceinline__ bool cta_row_reduce(double (&v)[Cfg::TN], int warp_n, int warp_m, int lane,
                                               double* scratch, double& out) {
  constexpr int TN = Cfg::TN, BN = Cfg::BN, WM = Cfg::WM;
#pragma unroll
  for (int i = 0; i < TN; ++i) {
    v[i] += __shfl_xor_sync(0xffffffffu, v[i], 1);
    v[i] += __shfl_xor_sync(0xffffffffu, v[i], 2);
  }
  if ((lane & 3) == 0) {
#pragma unroll
    for (int i = 0; i < TN; ++i) scratch[warp_m * BN + warp_n * TN * 8 + i * 8 + (lane >> 2)] = v[i];
  }
  consumer_sync<Cfg::CONSUMERS>();
  const int t = threadIdx.x;
  const bool have = t < BN;
  if (have) {
    double s = 0.0;
#pragma unroll
    for (int w = 0; w < WM; ++w) s += scratch[w * BN + t];
    out = s;
  }
  consumer_sync<Cfg::CONSUMERS>();   // scratch may be reused by the caller
  return have;
}

// ---- epilogue: plain store  Dt = alpha * acc -------------------------------------------------------
struct StoreEpi {
  double* Dt;
  int64_t ldd;
  int64_t group_stride;   // elements between the groups' outputs
  double alpha;
  template <class Cfg>
  __device__ __forceinline__ void run(double (&acc)[Cfg::TN][Cfg::TM][2], int n_blk0, int m_blk0, int warp_n,
                                      int warp_m, int lane, int N, int M, int grp, double*) const {
    double* base = Dt + (int64_t)grp * group_stride;
#pragma unroll
    for (int i = 0; i < Cfg::TN; ++i) {
      const int n = n_blk0 + (warp_n * Cfg::TN + i) * 8 + (lane >> 2);
      if (n >= N) continue;
#pragma unroll
      for (int j = 0; j < Cfg::TM; ++j) {
        const int m = m_blk0 + (warp_m * Cfg::TM + j) * 8 + 2 * (lane & 3);
        double* d = base + (int64_t)n * ldd + m;
        if (m + 1 < M) {
          *reinterpret_cast<double2*>(d) = make_double2(alpha * acc[i][j][0], alpha * acc[i][j][1]);
        } else if (m < M) {
          d[0] = alpha * acc[i][j][0];
        }
      }
    }
  }
};

// ---- host side ---------------------------------------------------------------------------------------
// One GEMM problem set as the host sees it; tensor maps are built by gemm_f64_prepare.
struct GemmProblem {
  const double* P = nullptr;   // [G * p_group_rows][ldp]
  int64_t ldp = 0;
  int p_group_rows = 0;
  int64_t p_total_rows = 0;    // rows of the stacked P array that may be read (>= G * p_group_rows)
  const double* Q[GEMM_MAX_GROUPS] = {};
  int64_t ldq = 0;
  bool q_blocked = false;      // Q[g] is K-blocked: [ceil(K / 16)][M][16]
  int G = 1;
  int M = 0, K = 0;
};

// src [rows][lds] -> dst [ceil(cols / 16)][rows][16] (columns beyond `cols` zero): the K-blocked Q layout
int kblock_f64(const double* src, int64_t lds, int64_t rows, int64_t cols, double* dst, cudaStream_t st);

// Tile configurations.  The slot dimension is cut into BN = 8 TN WN rows, the output dimension into
// BM = 8 TM WM.  Wide batches use 64 x 128 tiles (each Q tile feeds 64 slots); narrower ones shrink TN so
// that the last N tile is not mostly padding, and shrink BM to put more CTAs in flight.
using GemmW8 = GemmCfg<8, 1, 2, 8, 6>;   // 64 x 128
using GemmW6 = GemmCfg<6, 1, 2, 8, 4>;   // 48 x 128
using GemmW4 = GemmCfg<4, 1, 2, 8, 5>;   // 32 x 128
using GemmS8 = GemmCfg<8, 1, 1, 8, 5>;   // 64 x 64
using GemmS5 = GemmCfg<5, 1, 1, 8, 5>;   // 40 x 64
using GemmS3 = GemmCfg<3, 1, 1, 8, 6>;   // 24 x 64
using GemmS2 = GemmCfg<2, 1, 1, 8, 7>;   // 16 x 64
using GemmS1 = GemmCfg<1, 1, 1, 8, 8>;   //  8 x 64
using GemmX4 = GemmCfg<4, 2, 2, 8, 6>;   // 64 x 128, 16 consumer warps
using GemmS4 = GemmCfg<4, 1, 1, 8, 5>;   // 32 x 64 (5 stages: 3 CTAs per SM)
constexpr int GEMM_NUM_CFG = 10;

struct GemmTile {
  int cfg, BN, BM;
};
struct GemmTileInfo {   // what the cost model of gemm_f64_choose needs to know about a configuration
  int BN, BM, stages, occ;   // occ: resident CTAs per SM (shared memory / register limit)
};
inline GemmTile gemm_f64_tile_of(int cfg) {
  switch (cfg) {
    case 0: return {0, GemmW8::BN, GemmW8::BM};
    case 1: return {1, GemmW6::BN, GemmW6::BM};
    case 2: return {2, GemmW4::BN, GemmW4::BM};
    case 3: return {3, GemmS8::BN, GemmS8::BM};
    case 4: return {4, GemmS5::BN, GemmS5::BM};
    case 5: return {5, GemmS3::BN, GemmS3::BM};
    case 6: return {6, GemmS2::BN, GemmS2::BM};
    case 7: return {7, GemmS1::BN, GemmS1::BM};
    case 8: return {8, GemmX4::BN, GemmX4::BM};
    default: return {9, GemmS4::BN, GemmS4::BM};
  }
}
// Shape-based choice by a small cost model (gemm_host.cu): nb[g] = (upper bound of the) live slots of group g.
GemmTile gemm_f64_choose(const int* nb, int G, int M, int K);
int gemm_f64_force_cfg(int cfg);   // tuning hook: >= 0 forces a configuration, -1 restores the heuristic

int gemm_f64_make_args(const GemmProblem& pr, const GemmTile& tile, GemmArgs* out);

template <class Cfg, class Epi>
int launch_gemm_f64(const GemmArgs& a, int G, const Epi& epi, cudaStream_t st) {
  auto kern = gemm_f64_tma_kernel<Cfg, Epi>;
  static std::atomic<unsigned long long> configured{0};   // per template instantiation, one bit per device
  if (first_use_on_device(configured))
    TKM_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM));
  if (ceil_div(a.M, Cfg::BM) > 65535) return set_error(TKM_EINVAL, "GEMM: more than 65535 row tiles");
  dim3 grid((unsigned)(ceil_div(std::max(a.N, 1), Cfg::BN) * std::max(a.ksplit, 1)), (unsigned)ceil_div(a.M, Cfg::BM),
            (unsigned)G);
  kern<<<grid, Cfg::THREADS, Cfg::SMEM, st>>>(a, epi);
  TKM_LAUNCH_CHECK();
  return TKM_OK;
}

// `a` must have been built by gemm_f64_make_args for `tile`; a.N / a.nslots are set by the caller.
template <class Epi>
int gemm_f64_launch(const GemmArgs& a, const GemmTile& tile, int G, const Epi& epi, cudaStream_t st) {
  switch (tile.cfg) {
    case 0: return launch_gemm_f64<GemmW8>(a, G, epi, st);
    case 1: return launch_gemm_f64<GemmW6>(a, G, epi, st);
    case 2: return launch_gemm_f64<GemmW4>(a, G, epi, st);
    case 3: return launch_gemm_f64<GemmS8>(a, G, epi, st);
    case 4: return launch_gemm_f64<GemmS5>(a, G, epi, st);
    case 5: return launch_gemm_f64<GemmS3>(a, G, epi, st);
    case 6: return launch_gemm_f64<GemmS2>(a, G, epi, st);
    case 7: return launch_gemm_f64<GemmS1>(a, G, epi, st);
    case 8: return launch_gemm_f64<GemmX4>(a, G, epi, st);
    default: return launch_gemm_f64<GemmS4>(a, G, epi, st);
  }
}

// Convenience for one-off single-group products (setup, exact CV): choose, build maps, launch.
template <class Epi>
int gemm_f64_once(const double* P, int64_t ldp, const double* Q, int64_t ldq, int N, int M, int K, const Epi& epi,
                  cudaStream_t st, GemmTile* used = nullptr) {
  GemmProblem pr;
  pr.P = P;
  pr.ldp = ldp;
  pr.p_group_rows = N;
  pr.p_total_rows = N;
  pr.Q[0] = Q;
  pr.ldq = ldq;
  pr.G = 1;
  pr.M = M;
  pr.K = K;
  const GemmTile tile = gemm_f64_choose(&N, 1, M, K);
  GemmArgs a;
  TKM_TRY(gemm_f64_make_args(pr, tile, &a));
  a.N = N;
  a.nslots = nullptr;
  if (used) *used = tile;
  return gemm_f64_launch(a, tile, 1, epi, st);
}

}  // namespace tkm
