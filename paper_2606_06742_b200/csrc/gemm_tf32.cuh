// gemm_tf32.cuh -- 3xTF32 contraction on the 5th-generation tensor cores (tcgen05.mma, accumulator in TMEM):
// persistent CTA pairs (cta_group::2) with a stream-K partition of the work.
//
// Same product as gemm_f64.cuh,  Dt_g[N_g][M] = P_g[N_g][K] * Q_g[M][K]^T  ("NT", both K-contiguous), for the
// delta forms of the sweep (BASELINE.json north_star: "3xTF32 split").  Every operand is
// carried as a TF32-representable high part and a TF32-rounded remainder (x ~ hi + lo, about 21 mantissa bits);
// the product is accumulated in FP32 as  lo*hi + hi*lo + hi*hi  (the lo*lo term is below FP32 resolution).
//
// Tile.  The kernel is bound by the L2 -> shared-memory fill rate unless a tile is large (hi + lo operands weigh
// as much as FP64), so a tile is as large as tensor memory allows: a PAIR of CTAs on the two SMs of a TPC
// (cluster 2 x 1 x 1) owns 256 rows of the fixed operand Q (rows of U: 128 TMEM lanes in each CTA) times up to
// 512 slots of the moving operand P (two FP32 accumulators of <= 256 TMEM columns: all 512 columns of both SMs).
// Each CTA stages its own 128 Q rows and HALF of the P rows; tcgen05.mma.cta_group::2 (UMMA M = 256), issued by
// one thread of the leader CTA, reads both halves.
//
// Partition (stream-K).  Tiles of 256 x 512 never divide the 74 TPCs evenly (n = 2000 x 5 bandwidths: 40 tiles,
// n = 20000: 79 tiles), and the kernel's time is a chain of dependent MMAs along K.  So the launch is one wave of
// C <= 74 pairs and the linearised (tile, K-tile) space is cut into C equal ranges.  A pair whose range ends inside
// a tile is a HELPER for that tile: it contracts its K-range, stores the FP32 partial accumulator and raises a
// flag; the pair that holds the tile's last K-tile is its OWNER: it adds the helpers' partials in a fixed order
// (deterministic results) and runs the epilogue.  Every pair processes its helper segment FIRST, so an owner only
// ever waits for work that lower-numbered pairs start with: no cycle, and no dependence on co-residency.
//
// The number of live slots N_g of every group is read from device memory; slot tiles are padded to a multiple of
// 64 (each CTA's half to a multiple of 32 = one TMA box); the depth of the TMA -> MMA ring follows from the widest
// tile of the launch (2 stages at 512 slots, 5 at <= 64).  With Tf32Args.terms == 1 (single-TF32 products:
// tkm_loss_opts.tf32_delta = 3) a stage holds the hi tiles only: the ring is twice as deep (4 .. 8 stages), a launch
// streams half the bytes and the issuer sends one MMA per K-step instead of three.
//
// Warp roles (320 threads per CTA): warp 0 = TMA producer (its loads complete on the LEADER's full barrier),
// warp 1 = MMA issuer (leader CTA only), warps 2..9 = epilogue (warp w owns TMEM lanes 32 (w % 4) .. +31, i.e. 32
// rows of this CTA's 128; the two warps of a lane quarter take alternate 16-column chunks); warp 2 allocates
// TMEM (tcgen05.alloc.cta_group::2 in both CTAs).
#pragma once

#include <algorithm>
#include <cstdlib>

#include "tcgen05.cuh"

namespace tkm {

constexpr int TF32_MAX_GROUPS = 8;
constexpr int TF32_BM = 128;           // Q rows per CTA (UMMA M = 256 per pair)
constexpr int TF32_BK = 32;            // floats per stage row: 128 B
constexpr int TF32_BN = 512;           // slots per pair tile (two accumulators of 256 TMEM columns)
constexpr int TF32_PBOX = 32;          // P rows per TMA box
constexpr int TF32_A_BYTES = TF32_BM * 128;
constexpr int TF32_RED_BYTES = 4 * TF32_BN * 8;        // per-warp slot sums of a reducing epilogue
constexpr int TF32_TILE_SMEM = 208 * 1024;             // shared memory of the TMA -> MMA ring
constexpr size_t TF32_SMEM = TF32_TILE_SMEM + TF32_RED_BYTES + 1024;    // + alignment slack
constexpr int TF32_MAX_STAGES = 8;
constexpr int TF32_THREADS = 320;
constexpr int TF32_MIN_UNITS = 8;      // K-tiles below which a pair is not worth starting
// Smallest range of a pair, in K-tiles: at least half a tile's depth (a tile then has at most two helpers, whose
// partials the owner prefetches while it works), except that very deep contractions (thin U: K = n ~ 10^5) may be
// cut every 256 K-tiles -- there the exchange is small against the contraction.
__host__ __device__ inline int tf32_min_range(int KT) {
  const int h = (KT + 1) >> 1;
  const int w = h < 256 ? h : 256;
  return w > TF32_MIN_UNITS ? w : TF32_MIN_UNITS;
}
constexpr int TF32_MAX_PAIRS = 74;     // B200: 148 SMs
constexpr size_t TF32_PARTIAL_FLOATS = (size_t)TF32_BM * TF32_BN;   // one CTA's FP32 partial accumulator

struct Tf32Args {
  CUtensorMap p_hi, p_lo;                                  // [G * p_group_rows][K] floats, box = 32 x 32
  CUtensorMap q_hi[TF32_MAX_GROUPS], q_lo[TF32_MAX_GROUPS];   // per group [M][K] floats, box = 128 x 32
  const int32_t* nslots;                                   // [G] device or NULL
  int p_group_rows;
  int N, M, K;                                             // N: upper bound of the live slots of a group
  int G;                                                   // groups of this launch
  // K-blocked operands (thin U, K = n ~ 10^5..10^6): P is stored [K/32][p_blk_rows][32] and every Q_g
  // [K/32][q_blk_rows][32], so a stage is a few contiguous reads instead of one 128-byte piece from each of
  // several hundred rows that lie kilo- to megabytes apart.  The maps are then 2-D over [(K/32) blk_rows][32].
  // kblocked: bit 0 = Q blocked, bit 1 = P blocked.
  int kblocked, p_blk_rows, q_blk_rows;
  // stream-K exchange: FP32 partial accumulators [pairs][2][TF32_PARTIAL_FLOATS] and one flag per CTA; a flag
  // holds the `epoch` of the launch that wrote the partial (the host bumps it per launch, flags start at 0)
  float* partial;
  uint32_t* flags;
  uint32_t epoch;
  int min_range;   // smallest range of a pair in K-tiles (tf32_min_range, or the TKM_SK_MINRANGE tuning override)
  int terms;       // 3 (or 0): lo*hi + hi*lo + hi*hi, the 3xTF32 product; 1: hi*hi only -- a single TF32 product (11-bit
                   // operands): the lo tiles are neither loaded nor multiplied (half the bytes, a third of the MMAs)
  unsigned long long* dbg;   // tuning aid (TKM_SK_DEBUG): clock64 stamps of pair 0 [0..] MMA full-wait done, [4096..] producer issue
};

// slots of a pair tile after padding
__host__ __device__ inline int tf32_tile_pad(int nt) { return ((nt + 63) >> 6) << 6; }
// copies = 2: every operand as (hi, lo); 1: hi only (Tf32Args.terms == 1)
__host__ __device__ inline int tf32_stages_of(int half_rows, int copies) {
  const int s = TF32_TILE_SMEM / (copies * (TF32_A_BYTES + half_rows * 128));
  return s < TF32_MAX_STAGES ? s : TF32_MAX_STAGES;
}

// One segment of a pair's range: K-tiles [k0, k1) of one tile.
struct Tf32Seg {
  int grp, n_blk0, nlive, n0, n1, m_pair0;   // tile: group, first slot, live slots, accumulator widths, first Q row of the pair
  int k0, k1;
  int helper;                   // 1: store the partial and raise the flag; 0: owner (epilogue)
  int help_first, help_count;   // owner: pairs help_first .. help_first + help_count - 1 hold partials of this tile
};

// group tables of the plan live in shared memory (dynamic indexing would put them into local memory)
struct Tf32Groups {
  int tile_base[TF32_MAX_GROUPS + 1];   // first tile of each group in the linearised tile list
  int ng[TF32_MAX_GROUPS];              // live slots
  int bn[TF32_MAX_GROUPS];              // slot-tile width of the group (multiple of 64, <= 512)
};
struct Tf32Plan {
  int mp, KT, W, nseg, t_first, t_last, last_is_helper;
  long long a, b;
};

__device__ __forceinline__ void tf32_segment(const Tf32Plan& pl, const Tf32Groups& gr, int idx, Tf32Seg& s) {
  // processing order: the helper segment (the pair's last tile, if its range ends inside it) first
  int t;
  if (pl.last_is_helper) t = idx == 0 ? pl.t_last : pl.t_first + idx - 1;
  else t = pl.t_first + idx;
  const long long tb = (long long)t * pl.KT;
  s.k0 = (int)(max(pl.a, tb) - tb);
  s.k1 = (int)(min(pl.b, tb + pl.KT) - tb);
  s.helper = s.k1 < pl.KT;
  int g = 0;
  while (t >= gr.tile_base[g + 1]) ++g;
  const int local = t - gr.tile_base[g];
  s.grp = g;
  s.n_blk0 = (local / pl.mp) * gr.bn[g];
  s.m_pair0 = (local % pl.mp) * 2 * TF32_BM;
  s.nlive = min(gr.bn[g], gr.ng[g] - s.n_blk0);
  const int pad = tf32_tile_pad(s.nlive);
  s.n0 = min(pad, 256);
  s.n1 = pad - s.n0;
  s.help_first = (int)(tb / pl.W);
  s.help_count = s.helper ? 0 : (int)((tb + pl.KT - 1) / pl.W) - s.help_first;
}

template <class Epi>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(TF32_THREADS, 1)
    gemm_tf32x3_kernel(const __grid_constant__ Tf32Args g, const Epi epi) {
  extern __shared__ uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t full_bar[TF32_MAX_STAGES];
  __shared__ __align__(8) uint64_t empty_bar[TF32_MAX_STAGES];
  __shared__ __align__(8) uint64_t accum_bar;       // MMA -> epilogue: the accumulator of a segment is complete
  __shared__ __align__(8) uint64_t tmem_free_bar;   // epilogue (both CTAs) -> MMA issuer: tensor memory drained
  __shared__ uint32_t tmem_slot;
  __shared__ Tf32Groups gr;
  __shared__ int s_half_max;

  // ---- the plan: identical in every CTA of the launch ----
  Tf32Plan pl;
  pl.mp = (g.M + 2 * TF32_BM - 1) / (2 * TF32_BM);
  pl.KT = (g.K + TF32_BK - 1) / TF32_BK;
  if (threadIdx.x == 0) {
    // Slot tiles are as wide as tensor memory allows (512 slots); stream-K balances the pairs along K.  (Cutting
    // the slots of a group into narrower tiles so that every pair also gets a share of the epilogue was tried when
    // the FP64 state updates were still fused into this kernel; with the product-only epilogue it only costs
    // MMA efficiency: 57 ns per MMA at 128 slots against 87 ns at 256.)
    gr.tile_base[0] = 0;
    int hm = 0;
    for (int i = 0; i < g.G; ++i) {
      const int n = max(0, g.nslots ? min(g.nslots[i], g.N) : g.N);
      const int split = (n + TF32_BN - 1) / TF32_BN;
      const int bn = n > 0 ? tf32_tile_pad((n + split - 1) / split) : 64;
      gr.ng[i] = n;
      gr.bn[i] = bn;
      gr.tile_base[i + 1] = gr.tile_base[i] + pl.mp * ((n + bn - 1) / bn);
      hm = max(hm, tf32_tile_pad(min(n, bn)) >> 1);
    }
    for (int i = g.G; i < TF32_MAX_GROUPS; ++i) gr.tile_base[i + 1] = gr.tile_base[g.G];
    s_half_max = hm;
  }
  __syncthreads();
  const int half_max = s_half_max;
  const long long total = (long long)gr.tile_base[g.G] * pl.KT;
  if (total == 0) return;
  const int pairs = (int)min((long long)(gridDim.x >> 1), max(1LL, total / g.min_range));
  pl.W = (int)((total + pairs - 1) / pairs);
  const int pair = (int)blockIdx.x >> 1;
  pl.a = (long long)pair * pl.W;
  if (pl.a >= total) return;   // the same decision in both CTAs of the pair
  pl.b = min(total, pl.a + pl.W);
  pl.t_first = (int)(pl.a / pl.KT);
  pl.t_last = (int)((pl.b - 1) / pl.KT);
  pl.nseg = pl.t_last - pl.t_first + 1;
  pl.last_is_helper = pl.b < (long long)(pl.t_last + 1) * pl.KT;

  const uint32_t rank = cluster_ctarank();            // 0 = leader
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nt = g.terms == 1 ? 1 : 2;                                // operand copies per stage
  const int stage_bytes = nt * (TF32_A_BYTES + half_max * 128);      // one layout for the launch: Q hi | (Q lo) | P hi | (P lo)
  const int STAGES = tf32_stages_of(half_max, nt);
  uint8_t* tiles = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  double* epi_red = reinterpret_cast<double*>(tiles + TF32_TILE_SMEM);   // [4][TF32_BN]

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < TF32_MAX_STAGES; ++s) {
      mbar_init(&full_bar[s], 1);    // leader: one arrive.expect_tx per use; completes when both CTAs' loads landed
      mbar_init(&empty_bar[s], 1);   // one multicast tcgen05.commit per use
    }
    mbar_init(&accum_bar, 1);
    mbar_init(&tmem_free_bar, 16);   // 8 epilogue warps of each CTA
    mbar_fence_init();
  }
  if (warp == 2) tmem_alloc_pair<512>(&tmem_slot);
  tc_fence_before();
  cluster_sync();          // barriers initialised and TMEM allocated in both CTAs before any remote arrive
  tc_fence_after();
  const uint32_t tmem_base = tmem_slot;

  if (warp == 0) {
    // ===== TMA producer (both CTAs): own Q rows, own half of the P rows; bytes complete on the leader's barrier.
    // The whole warp runs the loop (uniform operands), one elected lane issues. =====
    if (elect_one()) tma_prefetch_desc(&g.p_hi);
    const bool qb = g.kblocked & 1, pb = g.kblocked & 2;
    int s = 0, filled = 0;
    uint32_t phase = 1;
    for (int si = 0; si < pl.nseg; ++si) {
      Tf32Seg sg;
      tf32_segment(pl, gr, si, sg);
      const int m_blk0 = sg.m_pair0 + (int)rank * TF32_BM;
      const int prow = sg.grp * g.p_group_rows + sg.n_blk0;
      const int p0 = prow + (int)rank * (sg.n0 >> 1);              // first slot row of this CTA's half of range 0
      const int p1 = prow + sg.n0 + (int)rank * (sg.n1 >> 1);      // ... of range 1
      const int half = (sg.n0 + sg.n1) >> 1;
      const uint32_t seg_bytes = 2u * (uint32_t)(nt * (TF32_A_BYTES + half * 128));   // both CTAs
      const CUtensorMap* qh = &g.q_hi[sg.grp];
      const CUtensorMap* ql = &g.q_lo[sg.grp];
      for (int kt = sg.k0; kt < sg.k1; ++kt) {
        if (filled >= STAGES) mbar_wait(&empty_bar[s], phase);
        ++filled;
        uint8_t* st = tiles + (size_t)s * stage_bytes;
        const uint32_t lead_bar = mapa_u32(smem_u32(&full_bar[s]), 0);
        const int x = kt * TF32_BK;
        const int xq = qb ? 0 : x, yq = qb ? kt * g.q_blk_rows + m_blk0 : m_blk0;
        const int xp = pb ? 0 : x, yoff = pb ? kt * g.p_blk_rows : 0;
        if (elect_one()) {
          if (g.dbg && pair == 0 && rank == 0 && kt - sg.k0 < 2048) g.dbg[4096 + kt - sg.k0] = clock64();
          if (rank == 0) mbar_arrive_expect_tx(&full_bar[s], seg_bytes);
          tma_load_2d_pair(st, qh, xq, yq, lead_bar);
          if (nt == 2) tma_load_2d_pair(st + TF32_A_BYTES, ql, xq, yq, lead_bar);
          uint8_t* ph = st + nt * TF32_A_BYTES;
          uint8_t* plo = ph + half_max * 128;
          for (int b = 0; b < half; b += TF32_PBOX) {
            const int row = (b < (sg.n0 >> 1) ? p0 + b : p1 + (b - (sg.n0 >> 1))) + yoff;
            tma_load_2d_pair(ph + b * 128, &g.p_hi, xp, row, lead_bar);
            if (nt == 2) tma_load_2d_pair(plo + b * 128, &g.p_lo, xp, row, lead_bar);
          }
        }
        __syncwarp();
        if (++s == STAGES) {
          s = 0;
          phase ^= 1;
        }
      }
    }
  } else if (warp == 1) {
    if (rank == 0) {
      // ===== MMA issuer (leader CTA): UMMA M = 256 over both CTAs, N = n0 (+ n1) slots.  Whole warp, one elected
      // lane issues (always the same lane: tcgen05.commit tracks the MMAs of the committing thread). =====
      int s = 0;
      uint32_t phase = 0;
      for (int si = 0; si < pl.nseg; ++si) {
        Tf32Seg sg;
        tf32_segment(pl, gr, si, sg);
        const uint32_t idesc0 = umma_idesc_tf32(256, sg.n0), idesc1 = umma_idesc_tf32(256, max(sg.n1, 16));
        const uint32_t b1_off = (uint32_t)((sg.n0 >> 1) * 128) >> 4;   // range 1 inside a CTA's P half, in 16-byte units
        const bool two = sg.n1 > 0;
        if (si > 0) {   // the previous segment's accumulator has been drained by both CTAs' epilogue warps
          mbar_wait(&tmem_free_bar, (uint32_t)((si - 1) & 1));
          tc_fence_after();
        }
        for (int kt = sg.k0; kt < sg.k1; ++kt) {
          mbar_wait(&full_bar[s], phase);
          tc_fence_after();
          const uint8_t* st = tiles + (size_t)s * stage_bytes;
          const uint64_t a_hi = umma_smem_desc_sw128(st), a_lo = umma_smem_desc_sw128(st + TF32_A_BYTES);
          const uint64_t b_hi = umma_smem_desc_sw128(st + nt * TF32_A_BYTES);
          const uint64_t b_lo = umma_smem_desc_sw128(st + nt * TF32_A_BYTES + half_max * 128);   // nt == 2 only
          const uint32_t acc0 = kt == sg.k0 ? 0u : 1u;
          if (elect_one()) {
            if (g.dbg && pair == 0 && kt - sg.k0 < 2048) g.dbg[kt - sg.k0] = clock64();
            if (g.terms == 1) {
#pragma unroll
              for (int k = 0; k < 4; ++k) {
                const uint64_t o = (uint64_t)(k * 2);
                umma_tf32_pair(tmem_base, a_hi + o, b_hi + o, idesc0, k == 0 ? acc0 : 1u);
                if (two) umma_tf32_pair(tmem_base + 256, a_hi + o, b_hi + b1_off + o, idesc1, k == 0 ? acc0 : 1u);
              }
            } else if (!two) {
#pragma unroll
              for (int k = 0; k < 4; ++k) {
                const uint64_t o = (uint64_t)(k * 2);   // 8 floats = 32 B, in units of 16 B
                umma_tf32_pair(tmem_base, a_lo + o, b_hi + o, idesc0, k == 0 ? acc0 : 1u);
                umma_tf32_pair(tmem_base, a_hi + o, b_lo + o, idesc0, 1);
                umma_tf32_pair(tmem_base, a_hi + o, b_hi + o, idesc0, 1);
              }
            } else {
#pragma unroll
              for (int k = 0; k < 4; ++k) {
                const uint64_t o = (uint64_t)(k * 2);
                umma_tf32_pair(tmem_base, a_lo + o, b_hi + o, idesc0, k == 0 ? acc0 : 1u);
                umma_tf32_pair(tmem_base + 256, a_lo + o, b_hi + b1_off + o, idesc1, k == 0 ? acc0 : 1u);
                umma_tf32_pair(tmem_base, a_hi + o, b_lo + o, idesc0, 1);
                umma_tf32_pair(tmem_base + 256, a_hi + o, b_lo + b1_off + o, idesc1, 1);
                umma_tf32_pair(tmem_base, a_hi + o, b_hi + o, idesc0, 1);
                umma_tf32_pair(tmem_base + 256, a_hi + o, b_hi + b1_off + o, idesc1, 1);
              }
            }
            umma_commit_pair(&empty_bar[s]);   // frees the stage in BOTH CTAs once these MMAs have read it
          }
          __syncwarp();
          if (++s == STAGES) {
            s = 0;
            phase ^= 1;
          }
        }
        if (elect_one()) umma_commit_pair(&accum_bar);
        __syncwarp();
      }
    }
  } else {
    // ===== epilogue (both CTAs): TMEM -> registers -> partial store (helper) or Epi (owner) =====
    const int q = warp & 3, hsel = (warp - 2) >> 2;   // warps 2..5: even chunks, warps 6..9: odd chunks
    const int row = 32 * q + lane;                    // this thread's TMEM lane = row of the CTA's 128
    const uint32_t free_bar = mapa_u32(smem_u32(&tmem_free_bar), 0);
    for (int si = 0; si < pl.nseg; ++si) {
      Tf32Seg sg;
      tf32_segment(pl, gr, si, sg);
      mbar_wait(&accum_bar, (uint32_t)(si & 1));
      tc_fence_after();
      const int m = sg.m_pair0 + (int)rank * TF32_BM + row;
      if (sg.helper) {
        // FP32 partial, layout [chunk of 16 slots][128 rows][16]: a warp stores 2 KB contiguously
        float* dst = g.partial + ((size_t)pair * 2 + rank) * TF32_PARTIAL_FLOATS;
#pragma unroll 1
        for (int c0 = 16 * hsel; c0 < sg.nlive; c0 += 32) {
          float v[16];
          tmem_ld_32x16(tmem_base + ((uint32_t)(32 * q) << 16) + (uint32_t)c0, v);
          float4* d4 = reinterpret_cast<float4*>(dst + ((size_t)(c0 >> 4) * TF32_BM + row) * 16);
#pragma unroll
          for (int i = 0; i < 4; ++i) d4[i] = make_float4(v[4 * i], v[4 * i + 1], v[4 * i + 2], v[4 * i + 3]);
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(free_bar);
        __threadfence();
        asm volatile("bar.sync 2, 256;\n" ::: "memory");
        if (tid == 64) st_release_gpu(g.flags + pair * 2 + rank, g.epoch);
      } else {
        if (sg.help_count > 0) {
          // wait for the helpers' partials (they are the first thing those pairs compute)
          if (lane == 0) {
            const long long t0 = clock64();
            for (int h = 0; h < sg.help_count; ++h)
              while (ld_acquire_gpu(g.flags + (sg.help_first + h) * 2 + rank) != g.epoch)
                if (clock64() - t0 > 20000000000LL) __trap();   // ~10 s: a lost helper must not hang the device
          }
          __syncwarp();
        }
        const float* src = g.partial + ((size_t)sg.help_first * 2 + rank) * TF32_PARTIAL_FLOATS;
        auto part_ptr = [&](int h, int c0) {
          return reinterpret_cast<const float4*>(src + (size_t)h * 2 * TF32_PARTIAL_FLOATS + ((size_t)(c0 >> 4) * TF32_BM + row) * 16);
        };
        // the first helpers' partials of the NEXT chunk are in flight while the current chunk's epilogue runs
        constexpr int HP = Epi::kReduce ? 1 : 2;   // (the reducing epilogue is short of registers)
        float4 pre[HP][4];
        const int hp = min(sg.help_count, HP);
        auto prefetch = [&](int c0) {
#pragma unroll
          for (int h = 0; h < HP; ++h)
            if (h < hp) {
              const float4* s4 = part_ptr(h, c0);
#pragma unroll
              for (int i = 0; i < 4; ++i) pre[h][i] = __ldcg(s4 + i);
            }
        };
        if (16 * hsel < sg.nlive) prefetch(16 * hsel);
#pragma unroll 1
        for (int c0 = 16 * hsel; c0 < sg.nlive; c0 += 32) {
          float v[16];
          tmem_ld_32x16(tmem_base + ((uint32_t)(32 * q) << 16) + (uint32_t)c0, v);
          // helpers in a fixed order: deterministic sums
#pragma unroll
          for (int h = 0; h < HP; ++h)
            if (h < hp) {
#pragma unroll
              for (int i = 0; i < 4; ++i) {
                v[4 * i] += pre[h][i].x;
                v[4 * i + 1] += pre[h][i].y;
                v[4 * i + 2] += pre[h][i].z;
                v[4 * i + 3] += pre[h][i].w;
              }
            }
          for (int h = HP; h < sg.help_count; ++h) {
            const float4* s4 = part_ptr(h, c0);
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const float4 t = __ldcg(s4 + i);
              v[4 * i] += t.x;
              v[4 * i + 1] += t.y;
              v[4 * i + 2] += t.z;
              v[4 * i + 3] += t.w;
            }
          }
          if (c0 + 32 < sg.nlive) prefetch(c0 + 32);
          if (c0 + 32 >= sg.nlive) {   // this warp's last chunk has left tensor memory
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(free_bar);
          }
          epi.chunk(v, m, sg.n_blk0 + c0, gr.ng[sg.grp], g.M, sg.grp, Epi::kReduce ? epi_red + q * TF32_BN + c0 : nullptr, lane);
        }
        if (16 * hsel >= sg.nlive) {   // a warp without chunks still has to report
          __syncwarp();
          if (lane == 0) mbar_arrive_cluster(free_bar);
        }
        if constexpr (Epi::kReduce) {
          // sum the four warps' per-slot sums in a fixed order: one thread per slot of the tile
          asm volatile("bar.sync 2, 256;\n" ::: "memory");
          for (int c = tid - 64; c < sg.nlive; c += 256)
            epi.finish(sg.n_blk0 + c, epi_red[c] + epi_red[TF32_BN + c] + epi_red[2 * TF32_BN + c] + epi_red[3 * TF32_BN + c],
                       (sg.m_pair0 / TF32_BM) + (int)rank, sg.grp);
          asm volatile("bar.sync 2, 256;\n" ::: "memory");   // epi_red is reused by the next segment
        }
      }
    }
  }
  __syncwarp();
  tc_fence_before();
  cluster_sync();          // both CTAs have drained their TMEM half; no load or commit is still in flight
  if (warp == 2) tmem_dealloc_pair<512>(tmem_base);
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

// stream-K exchange buffers of one stream of launches (the sweep owns one; launches on it are serialised)
struct Tf32Scratch {
  DevBuf partial, flags, dbg;
  uint32_t epoch = 0;
  int alloc(cudaStream_t st) {
    if (getenv("TKM_SK_DEBUG")) TKM_TRY(dbg.alloc(8192 * sizeof(unsigned long long), true, st, false));
    TKM_TRY(partial.alloc((size_t)TF32_MAX_PAIRS * 2 * TF32_PARTIAL_FLOATS * sizeof(float), false, st, true));
    TKM_TRY(flags.alloc((size_t)TF32_MAX_PAIRS * 2 * sizeof(uint32_t), true, st, true));
    epoch = 0;
    return TKM_OK;
  }
};

// `a` without the exchange fields; `upper[g]` = host-side upper bounds of the live slots (sizes the grid)
template <class Epi>
int gemm_tf32_launch(Tf32Args a, int G, Tf32Scratch& sc, const Epi& epi, cudaStream_t st) {
  auto kern = gemm_tf32x3_kernel<Epi>;
  static std::atomic<unsigned long long> configured{0};   // per template instantiation, one bit per device
  if (first_use_on_device(configured))
    TKM_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TF32_SMEM));
  a.G = G;
  a.partial = sc.partial.as<float>();
  a.flags = sc.flags.as<uint32_t>();
  a.epoch = ++sc.epoch;
  const int64_t units = (int64_t)G * ceil_div(a.M, 2 * TF32_BM) * ceil_div(std::max(a.N, 1), TF32_BN) * ceil_div(a.K, TF32_BK);
  a.dbg = sc.dbg.p ? sc.dbg.as<unsigned long long>() : nullptr;
  if (a.terms != 1) a.terms = 3;
  const char* mr = getenv("TKM_SK_MINRANGE");
  a.min_range = mr && *mr ? std::max(1, atoi(mr)) : tf32_min_range((int)ceil_div(a.K, TF32_BK));
  const int pairs = (int)std::max<int64_t>(1, std::min<int64_t>(TF32_MAX_PAIRS, units / a.min_range));
  kern<<<dim3(2 * pairs), TF32_THREADS, TF32_SMEM, st>>>(a, epi);
  TKM_LAUNCH_CHECK();
  return TKM_OK;
}

}  // namespace tkm
