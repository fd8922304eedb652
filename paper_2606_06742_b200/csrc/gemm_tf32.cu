// gemm_tf32.cu -- host side of the 3xTF32 tcgen05 contraction (gemm_tf32.cuh): FP32 tensor maps, the
// FP64 -> (hi, lo) TF32 split, and the C-ABI entry points tkm_tf32x3_gemm_nt / tkm_tf32x3_probe.
#include <algorithm>

#include "gemm_tf32.cuh"

namespace tkm {

// x -> hi = tf32(x), lo = tf32(x - hi); both stored as FP32 bit patterns with the low 13 mantissa bits zero
__global__ void split_tf32_kernel(const double* __restrict__ src, int64_t lds, int rows, int cols, float* __restrict__ hi,
                                  float* __restrict__ lo, int64_t ldo) {
  const int r = blockIdx.x;   // rows on grid.x: no 65535 limit
  for (int c = blockIdx.y * blockDim.x + threadIdx.x; c < cols; c += gridDim.y * blockDim.x) {
    const double v = src[(int64_t)r * lds + c];
    const float h = to_tf32((float)v);
    const float l = to_tf32((float)(v - (double)h));
    hi[(int64_t)r * ldo + c] = h;
    lo[(int64_t)r * ldo + c] = l;
  }
  (void)rows;
}

__global__ void split_tf32_kblocked_kernel(const double* __restrict__ src, int64_t lds, int rows, int cols,
                                           float* __restrict__ hi, float* __restrict__ lo) {
  const int r = blockIdx.x;
  const int cpad = ((cols + 31) >> 5) << 5;
  for (int c = blockIdx.y * blockDim.x + threadIdx.x; c < cpad; c += gridDim.y * blockDim.x) {
    float h = 0.0f, l = 0.0f;
    if (c < cols) {
      const double v = src[(int64_t)r * lds + c];
      h = to_tf32((float)v);
      l = to_tf32((float)(v - (double)h));
    }
    const int64_t o = ((int64_t)(c >> 5) * rows + r) * 32 + (c & 31);
    hi[o] = h;
    lo[o] = l;
  }
}

int split_tf32(const double* src, int64_t lds, int64_t rows, int64_t cols, float* hi, float* lo, int64_t ldo,
               cudaStream_t st) {
  dim3 grid((unsigned)rows, (unsigned)std::min<int64_t>(ceil_div(cols, 256), 64));
  split_tf32_kernel<<<grid, 256, 0, st>>>(src, lds, (int)rows, (int)cols, hi, lo, ldo);
  TKM_LAUNCH_CHECK();
  return TKM_OK;
}

int split_tf32_kblocked(const double* src, int64_t lds, int64_t rows, int64_t cols, float* hi, float* lo, cudaStream_t st) {
  dim3 grid((unsigned)rows, (unsigned)std::min<int64_t>(ceil_div(cols, 256), 64));
  split_tf32_kblocked_kernel<<<grid, 256, 0, st>>>(src, lds, (int)rows, (int)cols, hi, lo);
  TKM_LAUNCH_CHECK();
  return TKM_OK;
}

}  // namespace tkm

using namespace tkm;

// Dt[N][M] (FP64) = P[N][K] Q[M][K]^T with both FP64 inputs split into TF32 (hi, lo) pairs on the fly and the
// product formed by the 3xTF32 tcgen05 kernel (FP32 accumulation).  cfg is ignored (kept for ABI stability: the
// pair kernel has one tile shape).  Test / calibration entry; ms [host] may be NULL, else the kernel time of
// `iters` launches.
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
  Tf32Args a;
  memset(&a, 0, sizeof(a));
  TKM_TRY(make_tmap_f32(&a.p_hi, ph.as<float>(), N, K, ldk, TF32_PBOX));
  TKM_TRY(make_tmap_f32(&a.p_lo, pl.as<float>(), N, K, ldk, TF32_PBOX));
  TKM_TRY(make_tmap_f32(&a.q_hi[0], qh.as<float>(), M, K, ldk, TF32_BM));
  TKM_TRY(make_tmap_f32(&a.q_lo[0], ql.as<float>(), M, K, ldk, TF32_BM));
  Tf32Scratch sc;
  TKM_TRY(sc.alloc(st));
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
  int rc = gemm_tf32_launch(a, 1, sc, epi, st);
  if (ms && rc == TKM_OK) {
    cudaEventRecord(e0, st);
    for (int i = 0; i < std::max(iters, 1) && rc == TKM_OK; ++i) rc = gemm_tf32_launch(a, 1, sc, epi, st);
    cudaEventRecord(e1, st);
  }
  cudaError_t e = cudaStreamSynchronize(st);   // the split buffers are freed on return
  if (sc.dbg.p) {   // TKM_SK_DEBUG: intervals of pair 0's last launch
    std::vector<unsigned long long> h(8192);
    cudaMemcpy(h.data(), sc.dbg.p, 8192 * sizeof(unsigned long long), cudaMemcpyDeviceToHost);
    fprintf(stderr, "mma full-wait stamps (delta clk): ");
    for (int i = 1; i < 64 && h[i]; ++i) fprintf(stderr, "%llu ", h[i] - h[i - 1]);
    fprintf(stderr, "\nproducer issue stamps (delta clk): ");
    for (int i = 1; i < 64 && h[4096 + i]; ++i) fprintf(stderr, "%llu ", h[4096 + i] - h[4096 + i - 1]);
    fprintf(stderr, "\nproducer[0] -> mma[0]: %lld clk\n", (long long)(h[0] - h[4096]));
  }
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
