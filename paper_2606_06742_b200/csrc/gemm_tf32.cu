// gemm_tf32.cu -- host side of the 3xTF32 tcgen05 contraction (gemm_tf32.cuh): FP32 tensor maps, the
// FP64 -> (hi, lo) TF32 split, and the C-ABI entry points tkm_tf32x3_gemm_nt / tkm_tf32x3_probe.
#include <algorithm>

#include "gemm_tf32.cuh"

namespace tkm {

int make_tmap_f32(CUtensorMap* out, const float* base, int64_t rows, int64_t cols, int64_t ld, int box_rows);

// x -> hi = tf32(x), lo = tf32(x - hi); both stored as FP32 bit patterns with the low 13 mantissa bits zero
__global__ void split_tf32_kernel(const double* __restrict__ src, int64_t lds, int rows, int cols, float* __restrict__ hi,
                                  float* __restrict__ lo, int64_t ldo) {
  const int r = blockIdx.y;
  for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < cols; c += gridDim.x * blockDim.x) {
    const double v = src[(int64_t)r * lds + c];
    const float h = to_tf32((float)v);
    const float l = to_tf32((float)(v - (double)h));
    hi[(int64_t)r * ldo + c] = h;
    lo[(int64_t)r * ldo + c] = l;
  }
  (void)rows;
}

int split_tf32(const double* src, int64_t lds, int64_t rows, int64_t cols, float* hi, float* lo, int64_t ldo,
               cudaStream_t st) {
  dim3 grid((unsigned)std::min<int64_t>(ceil_div(cols, 256), 64), (unsigned)rows);
  split_tf32_kernel<<<grid, 256, 0, st>>>(src, lds, (int)rows, (int)cols, hi, lo, ldo);
  TKM_LAUNCH_CHECK();
  return TKM_OK;
}

template <class Cfg, class Epi>
int launch_gemm_tf32(const Tf32Args& a, int G, const Epi& epi, cudaStream_t st) {
  auto kern = gemm_tf32x3_kernel<Cfg, Epi>;
  static bool configured = false;
  if (!configured) {
    TKM_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM));
    configured = true;
  }
  dim3 grid((unsigned)ceil_div(a.M, TF32_BM), (unsigned)ceil_div(std::max(a.N, 1), Cfg::BN), (unsigned)G);
  kern<<<grid, Cfg::THREADS, Cfg::SMEM, st>>>(a, epi);
  TKM_LAUNCH_CHECK();
  return TKM_OK;
}

using Tf32N64 = Tf32Cfg<64, 4>;     // 48 KB per stage
using Tf32N128 = Tf32Cfg<128, 3>;   // 64 KB per stage
using Tf32N256 = Tf32Cfg<256, 2>;   // 96 KB per stage

int tf32_bn_of(int cfg) { return cfg == 0 ? 64 : (cfg == 1 ? 128 : 256); }

template <class Epi>
int gemm_tf32_launch(const Tf32Args& a, int cfg, int G, const Epi& epi, cudaStream_t st) {
  switch (cfg) {
    case 0: return launch_gemm_tf32<Tf32N64>(a, G, epi, st);
    case 1: return launch_gemm_tf32<Tf32N128>(a, G, epi, st);
    default: return launch_gemm_tf32<Tf32N256>(a, G, epi, st);
  }
}

}  // namespace tkm

using namespace tkm;

// Dt[N][M] (FP64) = P[N][K] Q[M][K]^T with both FP64 inputs split into TF32 (hi, lo) pairs on the fly and the
// product formed by the 3xTF32 tcgen05 kernel (FP32 accumulation).  cfg: 0/1/2 = 64/128/256 slots per tile,
// -1 = by N.  Test / calibration entry; ms [host] may be NULL, else the kernel time of `iters` launches.
extern "C" int tkm_tf32x3_gemm_nt(const double* P, int64_t ldp, const double* Q, int64_t ldq, double* Dt, int64_t ldd,
                                  int64_t N, int64_t M, int64_t K, int32_t cfg, int32_t iters, float* ms, void* stream) {
  if (!P || !Q || !Dt || N < 1 || M < 1 || K < 1 || ldp < K || ldq < K || ldd < M || N > (1 << 24) || M > (1 << 24) ||
      K > (1 << 24) || cfg > 2)
    return set_error(TKM_EINVAL, "tkm_tf32x3_gemm_nt: bad arguments");
  TKM_TRY(device_check());
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t ldk = round_up(K, 32);
  DevBuf ph, pl, qh, ql;
  TKM_TRY(ph.alloc((size_t)N * ldk * sizeof(float), true, st));
  TKM_TRY(pl.alloc((size_t)N * ldk * sizeof(float), true, st));
  TKM_TRY(qh.alloc((size_t)M * ldk * sizeof(float), true, st));
  TKM_TRY(ql.alloc((size_t)M * ldk * sizeof(float), true, st));
  TKM_TRY(split_tf32(P, ldp, N, K, ph.as<float>(), pl.as<float>(), ldk, st));
  TKM_TRY(split_tf32(Q, ldq, M, K, qh.as<float>(), ql.as<float>(), ldk, st));
  if (cfg < 0) cfg = N <= 64 ? 0 : (N <= 128 ? 1 : 2);
  const int bn = tf32_bn_of(cfg);
  Tf32Args a;
  memset(&a, 0, sizeof(a));
  TKM_TRY(make_tmap_f32(&a.p_hi, ph.as<float>(), N, K, ldk, bn));
  TKM_TRY(make_tmap_f32(&a.p_lo, pl.as<float>(), N, K, ldk, bn));
  TKM_TRY(make_tmap_f32(&a.q_hi[0], qh.as<float>(), M, K, ldk, TF32_BM));
  TKM_TRY(make_tmap_f32(&a.q_lo[0], ql.as<float>(), M, K, ldk, TF32_BM));
  a.nslots = nullptr;
  a.p_group_rows = (int)N;
  a.N = (int)N;
  a.M = (int)M;
  a.K = (int)K;
  Tf32StoreEpi epi{Dt, ldd, 0};
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (ms) {
    TKM_CUDA(cudaEventCreate(&e0));
    TKM_CUDA(cudaEventCreate(&e1));
  }
  int rc = gemm_tf32_launch(a, cfg, 1, epi, st);
  if (ms && rc == TKM_OK) {
    cudaEventRecord(e0, st);
    for (int i = 0; i < std::max(iters, 1) && rc == TKM_OK; ++i) rc = gemm_tf32_launch(a, cfg, 1, epi, st);
    cudaEventRecord(e1, st);
  }
  cudaError_t e = cudaStreamSynchronize(st);   // the split buffers are freed on return
  if (e != cudaSuccess) rc = set_error(TKM_ECUDA, "tkm_tf32x3_gemm_nt: %s", cudaGetErrorString(e));
  if (ms) {
    if (rc == TKM_OK) {
      cudaEventElapsedTime(ms, e0, e1);
      *ms /= (float)std::max(iters, 1);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
  }
  return rc;
}
