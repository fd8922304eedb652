// gemm_host.cu -- host side of the FP64 DMMA GEMM (gemm_f64.cuh): tensor-map encoding through the
// driver entry point, tile choice, and the calibration probes of the C ABI (tkm_dgemm_nt,
// tkm_gemm_probe).
#include <algorithm>
#include <mutex>

#include "gemm_f64.cuh"

namespace tkm {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  static std::once_flag once;
  std::call_once(once, [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
    else
      cudaGetLastError();
  });
  return fn;
}

int make_tmap_f64(CUtensorMap* out, const double* base, int64_t rows, int64_t cols, int64_t ld, int box_rows) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return set_error(TKM_ECUDA, "cuTensorMapEncodeTiled is not available from this driver");
  if ((reinterpret_cast<uintptr_t>(base) & 15) || (ld & 1) || rows < 1 || cols < 1 || ld < cols || box_rows < 1 ||
      box_rows > 256)
    return set_error(TKM_EINVAL, "GEMM operand needs a 16-byte aligned base and an even leading dimension >= cols");
  const cuuint64_t gdim[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
  const cuuint64_t gstride[1] = {(cuuint64_t)ld * sizeof(double)};
  const cuuint32_t box[2] = {(cuuint32_t)TMA_BOX_K, (cuuint32_t)box_rows};
  const cuuint32_t estr[2] = {1, 1};
  CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<double*>(base), gdim, gstride, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return set_error(TKM_ECUDA, "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
  return TKM_OK;
}

static int g_forced_cfg = -1;
int gemm_f64_force_cfg(int cfg) {
  const int old = g_forced_cfg;
  g_forced_cfg = (cfg >= 0 && cfg < GEMM_NUM_CFG) ? cfg : -1;
  return old;
}

GemmTile gemm_f64_choose(int nmax, int64_t ntot, int G, int M) {
  if (g_forced_cfg >= 0) return gemm_f64_tile_of(g_forced_cfg);
  (void)ntot;
  const int S = std::max(1, (nmax + 7) / 8);   // live 8-row sub-tiles of the widest group
  const int nt = (S + 7) / 8;                  // N tiles at the largest TN
  const int tn = (S + nt - 1) / nt;            // balanced TN
  const int64_t ctas_wide = ceil_div(M, 128) * (int64_t)G * nt;
  if (ctas_wide >= 148) {
    if (tn <= 4) return gemm_f64_tile_of(2);
    if (tn <= 6) return gemm_f64_tile_of(1);
    return gemm_f64_tile_of(0);
  }
  if (tn <= 1) return gemm_f64_tile_of(7);
  if (tn <= 2) return gemm_f64_tile_of(6);
  if (tn <= 3) return gemm_f64_tile_of(5);
  if (tn <= 5) return gemm_f64_tile_of(4);
  return gemm_f64_tile_of(3);
}

int gemm_f64_make_args(const GemmProblem& pr, const GemmTile& tile, GemmArgs* out) {
  if (pr.G < 1 || pr.G > GEMM_MAX_GROUPS) return set_error(TKM_EINVAL, "GEMM: 1..%d groups", GEMM_MAX_GROUPS);
  memset(out, 0, sizeof(*out));
  TKM_TRY(make_tmap_f64(&out->p_map, pr.P, std::max<int64_t>(pr.p_total_rows, 1), pr.K, pr.ldp, tile.BN));
  for (int g = 0; g < pr.G; ++g) TKM_TRY(make_tmap_f64(&out->q_map[g], pr.Q[g], pr.M, pr.K, pr.ldq, tile.BM));
  out->p_group_rows = pr.p_group_rows;
  out->M = pr.M;
  out->K = pr.K;
  out->N = 0;
  out->nslots = nullptr;
  return TKM_OK;
}

}  // namespace tkm

using namespace tkm;

extern "C" int tkm_dgemm_nt(const double* P, int64_t ldp, const double* Q, int64_t ldq, double* Dt, int64_t ldd,
                            int64_t N, int64_t M, int64_t K, void* stream) {
  if (!P || !Q || !Dt || N < 1 || M < 1 || K < 1 || ldp < K || ldq < K || ldd < M || (ldp & 1) || (ldq & 1) || (ldd & 1) ||
      N > (1 << 24) || M > (1 << 24) || K > (1 << 24))
    return set_error(TKM_EINVAL, "tkm_dgemm_nt: bad arguments");
  TKM_TRY(device_check());
  StoreEpi epi{Dt, ldd, 0, 1.0};
  return gemm_f64_once(P, ldp, Q, ldq, (int)N, (int)M, (int)K, epi, (cudaStream_t)stream);
}

// Calibration probe: G independent products Dt_g[N][M] = P_g[N][K] Q_g[M][K]^T on library-owned buffers
// filled with a fixed pattern, `iters` back-to-back launches of tile configuration `cfg` (-1: the
// heuristic's choice) timed with CUDA events on `stream`; *ms = average per launch.
extern "C" int tkm_gemm_probe(int32_t cfg, int32_t G, int32_t N, int32_t M, int32_t K, int32_t iters, float* ms,
                              void* stream) {
  if (G < 1 || G > GEMM_MAX_GROUPS || N < 1 || M < 1 || K < 1 || iters < 1 || !ms || cfg >= GEMM_NUM_CFG)
    return set_error(TKM_EINVAL, "tkm_gemm_probe: bad arguments");
  TKM_TRY(device_check());
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t ldk = round_up(K, 16), ldm = round_up(M, 16);
  DevBuf P, Q, D;
  TKM_TRY(P.alloc((size_t)G * N * ldk * sizeof(double), true, st));
  TKM_TRY(Q.alloc((size_t)G * M * ldk * sizeof(double), true, st));
  TKM_TRY(D.alloc((size_t)G * N * ldm * sizeof(double), true, st));
  TKM_CUDA(cudaMemsetAsync(P.p, 0x3f, (size_t)G * N * ldk * sizeof(double), st));   // finite pattern
  TKM_CUDA(cudaMemsetAsync(Q.p, 0x3f, (size_t)G * M * ldk * sizeof(double), st));
  GemmProblem pr;
  pr.P = P.as<double>();
  pr.ldp = ldk;
  pr.p_group_rows = N;
  pr.p_total_rows = (int64_t)G * N;
  for (int g = 0; g < G; ++g) pr.Q[g] = Q.as<double>() + (size_t)g * M * ldk;
  pr.ldq = ldk;
  pr.G = G;
  pr.M = M;
  pr.K = K;
  const GemmTile tile = cfg >= 0 ? gemm_f64_tile_of(cfg) : gemm_f64_choose(N, (int64_t)N * G, G, M);
  GemmArgs a;
  TKM_TRY(gemm_f64_make_args(pr, tile, &a));
  a.N = N;
  StoreEpi epi{D.as<double>(), ldm, (int64_t)N * ldm, 1.0};
  cudaEvent_t e0, e1;
  TKM_CUDA(cudaEventCreate(&e0));
  TKM_CUDA(cudaEventCreate(&e1));
  int rc = gemm_f64_launch(a, tile, G, epi, st);   // warm-up
  if (rc == TKM_OK) {
    cudaEventRecord(e0, st);
    for (int i = 0; i < iters && rc == TKM_OK; ++i) rc = gemm_f64_launch(a, tile, G, epi, st);
    cudaEventRecord(e1, st);
    cudaError_t e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) rc = set_error(TKM_ECUDA, "tkm_gemm_probe: %s", cudaGetErrorString(e));
    else {
      cudaEventElapsedTime(ms, e0, e1);
      *ms /= (float)iters;
    }
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return rc;
}
