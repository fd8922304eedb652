// gram.cu -- S1: RBF Gram matrix, FP64 (PAPER.md:69 kernel="rbf"; reading G12).
//
// K[i][j] = exp(-sum_k (x_ik - x'_jk)^2 / (2 sigma^2)) by direct differences (bit-exactly symmetric:
// (a-b)^2 == (b-a)^2 and the k-order is the same for (i,j) and (j,i)).  64x64 output tile per CTA,
// 4x4 outputs per thread, p consumed in chunks of 16 through shared memory.  For the symmetric case
// only tiles with bj >= bi are computed; the tile is staged through shared memory and written twice
// (as is, and transposed) with coalesced rows.  The matrix is written to HBM exactly once.
#include "common.cuh"

namespace tkm {

constexpr int GT = 64;   // tile edge
constexpr int GK = 16;   // feature chunk

constexpr int GRAM_MAX_SIGMAS = 8;
template <typename OutT>
struct GramOut {
  OutT* K[GRAM_MAX_SIGMAS];          // one output matrix per bandwidth
  double neg_inv_2s2[GRAM_MAX_SIGMAS];
  int G;
};

template <typename OutT>
__global__ void __launch_bounds__(256)
    gram_rbf_kernel(const double* __restrict__ X, int64_t ldx, int n, const double* __restrict__ Y,
                    int64_t ldy, int n2, int p, const GramOut<OutT> out, int64_t ldk, int symmetric, int nb) {
  int bi = blockIdx.y, bj = blockIdx.x;
  if (symmetric) {
    // enumerate the upper triangle: blockIdx.x runs over the nb(nb+1)/2 tiles with bj >= bi
    int t = blockIdx.x;
    bi = 0;
    while (t >= nb - bi) {
      t -= nb - bi;
      ++bi;
    }
    bj = bi + t;
  }
  // Ts (the finished tile) aliases the operand chunks, which are dead once the k-loop has ended.
  __shared__ __align__(16) double sbuf[GT * (GT + 1)];
  double (*Xs)[GT + 4] = reinterpret_cast<double (*)[GT + 4]>(sbuf);
  double (*Ys)[GT + 4] = reinterpret_cast<double (*)[GT + 4]>(sbuf + GK * (GT + 4));
  double (*Ts)[GT + 1] = reinterpret_cast<double (*)[GT + 1]>(sbuf);
  static_assert(2 * GK * (GT + 4) <= GT * (GT + 1), "operand chunks must fit inside the tile buffer");
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  const int i0 = bi * GT, j0 = bj * GT;
  double acc[4][4];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) acc[a][b] = 0.0;

  for (int k0 = 0; k0 < p; k0 += GK) {
    // 64 rows x 16 features per operand; thread t loads (row = t/4 .. , 4 consecutive k)
#pragma unroll
    for (int it = 0; it < 4; ++it) {
      const int id = tid + it * 256;      // 0..1023
      const int row = id >> 4, k = id & 15;
      const int gi = i0 + row, gj = j0 + row, gk = k0 + k;
      Xs[k][row] = (gi < n && gk < p) ? X[(int64_t)gi * ldx + gk] : 0.0;
      Ys[k][row] = (gj < n2 && gk < p) ? Y[(int64_t)gj * ldy + gk] : 0.0;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < GK; ++k) {
      double xv[4], yv[4];
#pragma unroll
      for (int a = 0; a < 4; ++a) xv[a] = Xs[k][ty * 4 + a];
#pragma unroll
      for (int b = 0; b < 4; ++b) yv[b] = Ys[k][tx * 4 + b];
#pragma unroll
      for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) {
          const double d = xv[a] - yv[b];
          acc[a][b] = fma(d, d, acc[a][b]);
        }
    }
    __syncthreads();
  }
  // the squared distances are shared by every bandwidth: one exp + one coalesced write (and its mirror) each
  for (int g = 0; g < out.G; ++g) {
    const double c = out.neg_inv_2s2[g];
    OutT* __restrict__ K = out.K[g];
    if (g > 0) __syncthreads();   // the previous bandwidth's tile has been written out
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
      for (int b = 0; b < 4; ++b) Ts[ty * 4 + a][tx * 4 + b] = exp(acc[a][b] * c);
    __syncthreads();
    for (int id = tid; id < GT * GT; id += 256) {
      const int r = id >> 6, cc = id & 63;
      const int gi = i0 + r, gj = j0 + cc;
      if (gi < n && gj < n2) K[(int64_t)gi * ldk + gj] = (OutT)Ts[r][cc];
    }
    if (symmetric && bi != bj) {
      for (int id = tid; id < GT * GT; id += 256) {
        const int r = id >> 6, cc = id & 63;   // write K[j0 + r][i0 + c] = T[c][r]
        const int gi = j0 + r, gj = i0 + cc;
        if (gi < n && gj < n2) K[(int64_t)gi * ldk + gj] = (OutT)Ts[cc][r];
      }
    }
  }
}

}  // namespace tkm

static int gram_launch(const void* X, int64_t n, int64_t p, int64_t ldx, const void* X2, int64_t n2, int64_t ldx2,
                       const double* sigmas, int G, tkm_dtype out_dt, void* const* Ks, int64_t ldk, cudaStream_t st) {
  using namespace tkm;
  if (!X || !Ks || !sigmas) return set_error(TKM_EINVAL, "tkm_gram: X, K and sigma must be non-NULL");
  if (G < 1 || G > GRAM_MAX_SIGMAS) return set_error(TKM_EINVAL, "tkm_gram_multi: 1..%d bandwidths", GRAM_MAX_SIGMAS);
  for (int g = 0; g < G; ++g) {
    if (!Ks[g]) return set_error(TKM_EINVAL, "tkm_gram: K must be non-NULL");
    if (!(sigmas[g] > 0.0)) return set_error(TKM_EINVAL, "tkm_gram: sigma must be > 0 (got %g)", sigmas[g]);
  }
  if (n <= 0 || p <= 0 || n > (1 << 30) || p > (1 << 24))
    return set_error(TKM_EINVAL, "tkm_gram: n=%lld p=%lld out of range", (long long)n, (long long)p);
  if (ldx < p) return set_error(TKM_EINVAL, "tkm_gram: ldx < p");
  const bool sym = (X2 == nullptr);
  if (sym) {
    X2 = X;
    n2 = n;
    ldx2 = ldx;
  } else if (n2 <= 0 || ldx2 < p || n2 > (1 << 30)) {
    return set_error(TKM_EINVAL, "tkm_gram: bad n2 / ldx2");
  }
  if (ldk < n2) return set_error(TKM_EINVAL, "tkm_gram: ldk < n2");
  if (out_dt != TKM_F64 && out_dt != TKM_F32) return set_error(TKM_EINVAL, "tkm_gram: bad out_dt");
  TKM_TRY(device_check());
  const int nbi = (int)ceil_div(n, GT), nbj = (int)ceil_div(n2, GT);
  const dim3 grid = sym ? dim3((unsigned)((int64_t)nbi * (nbi + 1) / 2), 1) : dim3(nbj, nbi);
  if (out_dt == TKM_F64) {
    GramOut<double> o;
    o.G = G;
    for (int g = 0; g < G; ++g) {
      o.K[g] = (double*)Ks[g];
      o.neg_inv_2s2[g] = -1.0 / (2.0 * sigmas[g] * sigmas[g]);
    }
    gram_rbf_kernel<double><<<grid, 256, 0, st>>>((const double*)X, ldx, (int)n, (const double*)X2, ldx2, (int)n2,
                                                  (int)p, o, ldk, sym ? 1 : 0, nbi);
  } else {
    GramOut<float> o;
    o.G = G;
    for (int g = 0; g < G; ++g) {
      o.K[g] = (float*)Ks[g];
      o.neg_inv_2s2[g] = -1.0 / (2.0 * sigmas[g] * sigmas[g]);
    }
    gram_rbf_kernel<float><<<grid, 256, 0, st>>>((const double*)X, ldx, (int)n, (const double*)X2, ldx2, (int)n2,
                                                 (int)p, o, ldk, sym ? 1 : 0, nbi);
  }
  TKM_LAUNCH_CHECK();
  return TKM_OK;
}

extern "C" int tkm_gram(const void* X, int64_t n, int64_t p, int64_t ldx, const void* X2, int64_t n2,
                        int64_t ldx2, double sigma, tkm_dtype out_dt, void* K, int64_t ldk, void* stream) {
  void* Ks[1] = {K};
  return gram_launch(X, n, p, ldx, X2, n2, ldx2, &sigma, 1, out_dt, Ks, ldk, (cudaStream_t)stream);
}

extern "C" int tkm_gram_multi(const void* X, int64_t n, int64_t p, int64_t ldx, const void* X2, int64_t n2,
                              int64_t ldx2, const double* sigmas, int32_t G, tkm_dtype out_dt, void* const* Ks,
                              int64_t ldk, void* stream) {
  tkm::NvtxRange nvtx_range("tkm_gram");
  return gram_launch(X, n, p, ldx, X2, n2, ldx2, sigmas, G, out_dt, Ks, ldk, (cudaStream_t)stream);
}
