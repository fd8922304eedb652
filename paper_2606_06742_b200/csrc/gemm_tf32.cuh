// gemm_tf32.cuh -- 3xTF32 contraction on the 5th-generation tensor cores (tcgen05.mma, accumulator in TMEM).
//
// Same product as gemm_f64.cuh,  Dt_g[N_g][M] = P_g[N_g][K] * Q_g[M][K]^T  ("NT", both K-contiguous), for the
// FP32 variant of the sweep (BASELINE.json north_star: "3xTF32 split").  Every FP32 operand is carried as a
// TF32-representable high part and a TF32-rounded remainder (x ~ hi + lo, about 21 mantissa bits); the product
// is accumulated in FP32 as  lo*hi + hi*lo + hi*hi  (the lo*lo term is below FP32 resolution).
//
// Mapping: the fixed operand Q (rows of U) is the UMMA "A" operand, M = 128 rows = the 128 TMEM lanes; the
// moving operand P (slots) is the UMMA "B" operand, N = BN slots = BN FP32 TMEM columns.  K advances 32
// floats (one 128-byte swizzle span) per pipeline stage = 4 UMMA K-steps of 8, 3 MMAs each.
// Warp roles (320 threads): warp 0 = TMA producer, warp 1 = MMA issuer (one elected thread), warps 2..9 =
// epilogue (warp w owns TMEM lanes 32 (w % 4) .. +31, i.e. 32 rows of the tile; the two warps of a lane quarter
// take alternate 16-column chunks -- FP64 epilogue arithmetic is latency-bound with one warp per scheduler);
// warp 2 allocates TMEM.
#pragma once

#include <algorithm>

#include "tcgen05.cuh"

namespace tkm {

constexpr int TF32_MAX_GROUPS = 8;
constexpr int TF32_BM = 128;          // UMMA M
constexpr int TF32_BK = 32;           // floats per stage row: 128 B
constexpr int TF32_A_BYTES = TF32_BM * 128;

struct Tf32Args {
  CUtensorMap p_hi, p_lo;                                  // [G * p_group_rows][K] floats, box = BN x 32
  CUtensorMap q_hi[TF32_MAX_GROUPS], q_lo[TF32_MAX_GROUPS];   // per group [M][K] floats, box = 128 x 32
  const int32_t* nslots;                                   // [G] device or NULL
  int p_group_rows;
  int N, M, K;
  int ksplit;   // as in GemmArgs: S > 1 => blockIdx.y = split * n_tiles + n_tile, K-tiles [s KT/S, (s+1) KT/S)
  // K-blocked operands (thin U, K = n ~ 10^5..10^6): P is stored [K/32][p_blk_rows][32] and every Q_g
  // [K/32][q_blk_rows][32], so a stage is two contiguous reads instead of one 128-byte piece from each of
  // several hundred rows that lie kilo- to megabytes apart.  The maps are then 2-D over [(K/32) blk_rows][32].
  // kblocked: bit 0 = Q blocked, bit 1 = P blocked.
  int kblocked, p_blk_rows, q_blk_rows;
};

template <int BN_, int STAGES_>
struct Tf32Cfg {
  static constexpr int BN = BN_, STAGES = STAGES_;
  static constexpr int B_BYTES = BN * 128;
  static constexpr int STAGE_BYTES = 2 * TF32_A_BYTES + 2 * B_BYTES;
  static constexpr size_t SMEM = (size_t)STAGES * STAGE_BYTES + 1024;
  static constexpr int THREADS = 320;
  static_assert(BN == 32 || BN == 64 || BN == 128 || BN == 256, "TMEM allocations are powers of two >= 32 columns");
};

template <class Cfg, class Epi>
__global__ void __launch_bounds__(Cfg::THREADS, 1) gemm_tf32x3_kernel(const __grid_constant__ Tf32Args g, const Epi epi) {
  constexpr int BN = Cfg::BN, STAGES = Cfg::STAGES;
  extern __shared__ uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t full_bar[STAGES];
  __shared__ __align__(8) uint64_t empty_bar[STAGES];
  __shared__ __align__(8) uint64_t accum_bar;
  __shared__ uint32_t tmem_slot;
  __shared__ double epi_red[Epi::kReduce ? 4 : 1][Epi::kReduce ? BN : 1];   // per-warp slot sums of a reducing epilogue

  const int grp = blockIdx.z;
  const int N = g.nslots ? min(g.nslots[grp], g.N) : g.N;
  const int S = max(g.ksplit, 1), ny = (int)gridDim.y / S, split = (int)blockIdx.y / ny;
  const int m_blk0 = blockIdx.x * TF32_BM, n_blk0 = ((int)blockIdx.y - split * ny) * BN;
  if (n_blk0 >= N) return;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int KT_all = (g.K + TF32_BK - 1) / TF32_BK;
  const int kt0 = (int)((int64_t)split * KT_all / S), KT = (int)((int64_t)(split + 1) * KT_all / S) - kt0;   // host: S <= KT_all
  uint8_t* tiles = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(&full_bar[s], 1);
      mbar_init(&empty_bar[s], 1);
    }
    mbar_init(&accum_bar, 1);
    mbar_fence_init();
  }
  if (warp == 2) tmem_alloc<BN>(&tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_slot;

  if (warp == 0) {
    if (lane == 0) {
      // ===== TMA producer =====
      const int prow = grp * g.p_group_rows + n_blk0;
      int s = 0;
      uint32_t phase = 1;
      for (int kt = 0; kt < KT; ++kt) {
        if (kt >= STAGES) mbar_wait(&empty_bar[s], phase);
        mbar_arrive_expect_tx(&full_bar[s], Cfg::STAGE_BYTES);
        uint8_t* st = tiles + (size_t)s * Cfg::STAGE_BYTES;
        const int x = (kt0 + kt) * TF32_BK;
        const bool qb = g.kblocked & 1, pb = g.kblocked & 2;
        const int xq = qb ? 0 : x, yq = qb ? (kt0 + kt) * g.q_blk_rows + m_blk0 : m_blk0;
        const int xp = pb ? 0 : x, yp = pb ? (kt0 + kt) * g.p_blk_rows + prow : prow;
        tma_load_2d(st, &g.q_hi[grp], xq, yq, &full_bar[s]);
        tma_load_2d(st + TF32_A_BYTES, &g.q_lo[grp], xq, yq, &full_bar[s]);
        tma_load_2d(st + 2 * TF32_A_BYTES, &g.p_hi, xp, yp, &full_bar[s]);
        tma_load_2d(st + 2 * TF32_A_BYTES + Cfg::B_BYTES, &g.p_lo, xp, yp, &full_bar[s]);
        if (++s == STAGES) {
          s = 0;
          phase ^= 1;
        }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      // ===== MMA issuer =====
      // a ragged last tile multiplies only the live slots (UMMA N is any multiple of 16)
      const uint32_t idesc = umma_idesc_tf32(TF32_BM, min(BN, ((N - n_blk0 + 15) >> 4) << 4));
      int s = 0;
      uint32_t phase = 0, acc = 0;
      for (int kt = 0; kt < KT; ++kt) {
        mbar_wait(&full_bar[s], phase);
        tc_fence_after();
        const uint8_t* st = tiles + (size_t)s * Cfg::STAGE_BYTES;
        const uint64_t a_hi = umma_smem_desc_sw128(st), a_lo = umma_smem_desc_sw128(st + TF32_A_BYTES);
        const uint64_t b_hi = umma_smem_desc_sw128(st + 2 * TF32_A_BYTES);
        const uint64_t b_lo = umma_smem_desc_sw128(st + 2 * TF32_A_BYTES + Cfg::B_BYTES);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const uint64_t o = (uint64_t)(k * 2);   // 8 floats = 32 B, in units of 16 B
          umma_tf32(tmem_base, a_lo + o, b_hi + o, idesc, acc);
          acc = 1;
          umma_tf32(tmem_base, a_hi + o, b_lo + o, idesc, 1);
          umma_tf32(tmem_base, a_hi + o, b_hi + o, idesc, 1);
        }
        umma_commit(&empty_bar[s]);   // frees the stage once these MMAs have read it
        if (++s == STAGES) {
          s = 0;
          phase ^= 1;
        }
      }
      umma_commit(&accum_bar);
    }
  } else {
    // ===== epilogue: TMEM -> registers -> Epi =====
    const int q = warp & 3, half = (warp - 2) >> 2;   // warps 2..5: even chunks, warps 6..9: odd chunks
    mbar_wait(&accum_bar, 0);
    tc_fence_after();
    const int m = m_blk0 + 32 * q + lane;
#pragma unroll 1
    for (int c0 = 16 * half; c0 < BN; c0 += 32) {
      if (n_blk0 + c0 >= N) break;   // warp-uniform
      float v[16];
      tmem_ld_32x16(tmem_base + ((uint32_t)(32 * q) << 16) + (uint32_t)c0, v);
      epi.chunk(v, m, n_blk0 + c0, N, g.M, grp, Epi::kReduce ? &epi_red[q][c0] : nullptr, lane);
    }
    if constexpr (Epi::kReduce) {
      // sum the four warps' per-slot sums in a fixed order: one thread per slot of the tile
      asm volatile("bar.sync 2, 256;\n" ::: "memory");
      for (int c = tid - 64; c < BN; c += 256)
        if (n_blk0 + c < N)
          epi.finish(n_blk0 + c, epi_red[0][c] + epi_red[1][c] + epi_red[2][c] + epi_red[3][c], (int)blockIdx.x, grp);
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc<BN>(tmem_base);
}

// plain store epilogue: Dt[n][m] = acc  (FP64 output array, one slot per row)
struct Tf32StoreEpi {
  static constexpr bool kReduce = false;
  double* Dt;
  int64_t ldd;
  int64_t group_stride;
  __device__ __forceinline__ void chunk(const float (&v)[16], int m, int n0, int N, int M, int grp, double*, int) const {
    if (m >= M) return;
    double* base = Dt + (int64_t)grp * group_stride + m;
#pragma unroll
    for (int i = 0; i < 16; ++i)
      if (n0 + i < N) base[(int64_t)(n0 + i) * ldd] = (double)v[i];
  }
};

// ---- host side (gemm_tf32.cu, gemm_host.cu) -------------------------------------------------------------
int make_tmap_f32(CUtensorMap* out, const float* base, int64_t rows, int64_t cols, int64_t ld, int box_rows);
int split_tf32(const double* src, int64_t lds, int64_t rows, int64_t cols, float* hi, float* lo, int64_t ldo,
               cudaStream_t st);   // x -> (tf32(x), tf32(x - hi))
// the same into the K-blocked layout [ceil(cols / 32)][rows][32] (columns beyond `cols` are written as zeros)
int split_tf32_kblocked(const double* src, int64_t lds, int64_t rows, int64_t cols, float* hi, float* lo, cudaStream_t st);
int tf32_bn_of(int cfg);           // slots per tile of configuration 0 / 1 / 2 = 64 / 128 / 256

template <class Cfg, class Epi>
int launch_gemm_tf32(const Tf32Args& a, int G, const Epi& epi, cudaStream_t st) {
  auto kern = gemm_tf32x3_kernel<Cfg, Epi>;
  static bool configured = false;
  if (!configured) {
    TKM_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM));
    configured = true;
  }
  dim3 grid((unsigned)ceil_div(a.M, TF32_BM), (unsigned)(ceil_div(std::max(a.N, 1), Cfg::BN) * std::max(a.ksplit, 1)),
            (unsigned)G);
  kern<<<grid, Cfg::THREADS, Cfg::SMEM, st>>>(a, epi);
  TKM_LAUNCH_CHECK();
  return TKM_OK;
}

using Tf32N64 = Tf32Cfg<64, 4>;     // 48 KB per stage
using Tf32N128 = Tf32Cfg<128, 3>;   // 64 KB per stage
using Tf32N256 = Tf32Cfg<256, 2>;   // 96 KB per stage

template <class Epi>
int gemm_tf32_launch(const Tf32Args& a, int cfg, int G, const Epi& epi, cudaStream_t st) {
  switch (cfg) {
    case 0: return launch_gemm_tf32<Tf32N64>(a, G, epi, st);
    case 1: return launch_gemm_tf32<Tf32N128>(a, G, epi, st);
    default: return launch_gemm_tf32<Tf32N256>(a, G, epi, st);
  }
}

}  // namespace tkm
