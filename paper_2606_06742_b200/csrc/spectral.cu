// spectral.cu -- S2: one-time spectral setup K = U Lam U^T (Alg.1 l.3, 226; readings
// G11 Nystrom, G16 eigenvalue clamp, G19 one decomposition shared by all folds).
//
// The eigendecomposition itself is cuSOLVER Dsyevd (allowed as setup by BASELINE.json north_star and
// timed separately from the sweep).  Everything else -- transposes, scalings, u1 = U^T 1, and the
// Nystrom products -- is this library's own kernels (the products use the DMMA GEMM of gemm_f64.cuh).
#include <cusolverDn.h>

#include <algorithm>
#include <cmath>
#include <condition_variable>
#include <functional>
#include <mutex>
#include <new>
#include <string>
#include <thread>

#include "gemm_f64.cuh"
#include "handles.cuh"

namespace tkm {

// dst[c][r] = src[r][c] * (row_scale ? row_scale[r] : 1): 32x32 shared-memory tile transpose.
__global__ void transpose_scale_kernel(const double* __restrict__ src, int64_t lds, int rows, int cols,
                                       const double* __restrict__ row_scale, double* __restrict__ dst,
                                       int64_t ldd) {
  __shared__ double tile[32][33];
  const int r0 = blockIdx.y * 32, c0 = blockIdx.x * 32;
  for (int i = threadIdx.y; i < 32; i += blockDim.y) {
    const int r = r0 + i, c = c0 + threadIdx.x;
    double v = 0.0;
    if (r < rows && c < cols) v = src[(int64_t)r * lds + c] * (row_scale ? row_scale[r] : 1.0);
    tile[i][threadIdx.x] = v;
  }
  __syncthreads();
  for (int i = threadIdx.y; i < 32; i += blockDim.y) {
    const int c = c0 + i, r = r0 + threadIdx.x;
    if (r < rows && c < cols) dst[(int64_t)c * ldd + r] = tile[threadIdx.x][i];
  }
}

int transpose_scale_f64(const double* src, int64_t lds, int64_t rows, int64_t cols, const double* row_scale,
                        double* dst, int64_t ldd, cudaStream_t st) {
  dim3 grid((unsigned)ceil_div(cols, 32), (unsigned)ceil_div(rows, 32));
  transpose_scale_kernel<<<grid, dim3(32, 8), 0, st>>>(src, lds, (int)rows, (int)cols, row_scale, dst, ldd);
  TKM_LAUNCH_CHECK();
  return TKM_OK;
}

// rows[j][0..cols) *= scale[j]
__global__ void row_scale_kernel(double* __restrict__ A, int64_t lda, int rows, int cols,
                                 const double* __restrict__ scale) {
  const int j = blockIdx.x;
  const double s = scale[j];
  for (int i = threadIdx.x; i < cols; i += blockDim.x) A[(int64_t)j * lda + i] *= s;
}

// out[j] = sum_i A[j][i]  (one CTA per row, fixed-order reduction => deterministic)
__global__ void row_sum_kernel(const double* __restrict__ A, int64_t lda, int cols, double* __restrict__ out) {
  __shared__ double red[32];
  const int j = blockIdx.x;
  double s = 0.0;
  for (int i = threadIdx.x; i < cols; i += blockDim.x) s += A[(int64_t)j * lda + i];
  s = block_sum(s, red);
  if (threadIdx.x == 0) out[j] = s;
}

// v[i] = op(v[i]): 0 clamp to >= 0, 1 -> 1/sqrt(v), 2 -> sqrt(v)
__global__ void vec_op_kernel(double* v, int n, int op) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double x = v[i];
  v[i] = op == 0 ? fmax(x, 0.0) : (op == 1 ? 1.0 / sqrt(x) : sqrt(x));
}

// cuSOLVER handles are expensive to create: keep finished ones in a pool (one is taken per running
// decomposition, so concurrent setups on different streams each get their own).
struct Solver {
  cusolverDnHandle_t h = nullptr;
  static std::mutex& mu() {
    static std::mutex m;
    return m;
  }
  static std::vector<cusolverDnHandle_t>& pool() {
    static std::vector<cusolverDnHandle_t> p;
    return p;
  }
  // a persistent set-up worker (below) keeps one handle of its own: the handle then always sees the same thread
  // and the same stream
  static cusolverDnHandle_t& thread_handle() {
    static thread_local cusolverDnHandle_t h = nullptr;
    return h;
  }
  static bool& thread_keeps_handle() {
    static thread_local bool k = false;
    return k;
  }
  int acquire() {
    if (thread_keeps_handle() && thread_handle()) {
      h = thread_handle();
      return TKM_OK;
    }
    {
      std::lock_guard<std::mutex> lk(mu());
      if (!pool().empty()) {
        h = pool().back();
        pool().pop_back();
        return TKM_OK;
      }
    }
    if (cusolverDnCreate(&h) != CUSOLVER_STATUS_SUCCESS) {
      h = nullptr;
      return set_error(TKM_ESOLVER, "cusolverDnCreate failed");
    }
    return TKM_OK;
  }
  ~Solver() {
    if (!h) return;
    if (thread_keeps_handle()) {
      thread_handle() = h;
      return;
    }
    std::lock_guard<std::mutex> lk(mu());
    if (pool().size() < 16)
      pool().push_back(h);
    else
      cusolverDnDestroy(h);
  }
};

// In-place symmetric eigendecomposition of the n x n matrix in A (column-major, lda): on return
// column j of A (= row j of the row-major view) is eigenvector j, W ascending.
static int syevd_inplace(double* A, int64_t lda, int64_t n, double* W, cudaStream_t st) {
  Solver sv;
  TKM_TRY(sv.acquire());
  if (cusolverDnSetStream(sv.h, st) != CUSOLVER_STATUS_SUCCESS) return set_error(TKM_ESOLVER, "cusolverDnSetStream failed");
  int lwork = 0;
  cusolverStatus_t cs = cusolverDnDsyevd_bufferSize(sv.h, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER,
                                                    (int)n, A, (int)lda, W, &lwork);
  if (cs != CUSOLVER_STATUS_SUCCESS) return set_error(TKM_ESOLVER, "Dsyevd_bufferSize failed (%d)", (int)cs);
  // stream-ordered temporaries from the library's pool (64 MB of workspace at n = 2000): cudaFree would synchronise
  // the whole device and stall the other setups of a tkm_spectral_setup_multi call, and the device's DEFAULT pool
  // (release threshold 0) hands its memory back to the driver at every synchronisation -- a kernel-mode allocation
  // per decomposition per step, which on shared boxes stalled for 0.1-1.6 s at random (profiles/r02_host_stalls.md)
  DevBuf work, info;
  TKM_TRY(work.alloc((size_t)std::max(lwork, 1) * sizeof(double), false, st, true));
  TKM_TRY(info.alloc(sizeof(int), false, st, true));
  TKM_CUDA(cudaMemsetAsync(info.p, 0, sizeof(int), st));
  cs = cusolverDnDsyevd(sv.h, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, (int)n, A, (int)lda, W,
                        (double*)work.p, lwork, (int*)info.p);
  if (cs != CUSOLVER_STATUS_SUCCESS) return set_error(TKM_ESOLVER, "cusolverDnDsyevd failed (%d)", (int)cs);
  int h_info = 0;
  TKM_CUDA(cudaMemcpyAsync(&h_info, info.p, sizeof(int), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaStreamSynchronize(st));
  if (h_info != 0) return set_error(TKM_ESOLVER, "Dsyevd: info = %d", h_info);
  return TKM_OK;
}

static int dgemm_nt(const double* P, int64_t ldp, const double* Q, int64_t ldq, double* Dt, int64_t ldd,
                    int64_t N, int64_t M, int64_t K, cudaStream_t st) {
  if ((ldd & 1) || ((uintptr_t)Dt & 15))
    return set_error(TKM_EINVAL, "dgemm_nt: output must be 16-byte aligned with an even leading dimension");
  StoreEpi epi{Dt, ldd, 0, 1.0};
  return gemm_f64_once(P, ldp, Q, ldq, (int)N, (int)M, (int)K, epi, st);
}

// Finish a handle whose Ut ([r][ldn], rows = orthonormal eigenvectors) and lam are in place.
static int finish_spectral(tkm_spectral* s, cudaStream_t st) {
  const int64_t n = s->n, r = s->r;
  vec_op_kernel<<<(unsigned)ceil_div(r, 256), 256, 0, st>>>(s->lam.as<double>(), (int)r, 0);   // clamp (G16)
  TKM_LAUNCH_CHECK();
  row_sum_kernel<<<(unsigned)r, 256, 0, st>>>(s->Ut.as<double>(), s->ldn, (int)n, s->u1.as<double>());
  TKM_LAUNCH_CHECK();
  if (!s->UL.p) TKM_TRY(s->UL.alloc((size_t)n * s->ldr * sizeof(double), true, st));
  TKM_TRY(transpose_scale_f64(s->Ut.as<double>(), s->ldn, r, n, s->lam.as<double>(), s->UL.as<double>(), s->ldr, st));
  s->h_lam.resize(r);
  s->h_u1.resize(r);
  TKM_CUDA(cudaMemcpyAsync(s->h_lam.data(), s->lam.p, r * sizeof(double), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaMemcpyAsync(s->h_u1.data(), s->u1.p, r * sizeof(double), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaStreamSynchronize(st));
  if (s->r == s->n) {
    s->thin = 0.0;   // ||U^T 1||^2 = n exactly for an orthogonal U (reading G1)
  } else {
    long double acc = 0.0L;
    for (int64_t i = 0; i < r; ++i) acc += (long double)s->h_u1[i] * s->h_u1[i];
    s->thin = (double)((long double)n - acc);
    if (s->thin < 0.0) s->thin = 0.0;
  }
  return TKM_OK;
}

// Allocations of a full-kernel handle, separated from the arithmetic so that tkm_spectral_setup_multi can make
// them before its worker threads start (cudaMalloc serialises with work of the other streams).
static int alloc_full(int64_t n, tkm_spectral* s, cudaStream_t st) {
  s->n = s->r = n;
  s->ldn = s->ldr = round_up(n, 16);
  TKM_TRY(s->Ut.alloc((size_t)n * s->ldn * sizeof(double), true, st));
  TKM_TRY(s->lam.alloc((size_t)s->ldr * sizeof(double), true, st));
  TKM_TRY(s->u1.alloc((size_t)s->ldr * sizeof(double), true, st));
  TKM_TRY(s->UL.alloc((size_t)n * s->ldr * sizeof(double), true, st));
  return TKM_OK;
}
static int compute_full(const double* K, int64_t n, int64_t ldk, tkm_spectral* s, cudaStream_t st) {
  TKM_CUDA(cudaMemcpy2DAsync(s->Ut.p, s->ldn * sizeof(double), K, ldk * sizeof(double), n * sizeof(double), n,
                             cudaMemcpyDeviceToDevice, st));
  TKM_TRY(syevd_inplace(s->Ut.as<double>(), s->ldn, n, s->lam.as<double>(), st));
  return finish_spectral(s, st);
}
static int setup_full(const double* K, int64_t n, int64_t ldk, tkm_spectral* s, cudaStream_t st) {
  TKM_TRY(alloc_full(n, s, st));
  return compute_full(K, n, ldk, s, st);
}

constexpr double NYS_RANK_TOL = 1e-12;

// Where the rows of K_nm come from: a resident matrix, or X itself -- then K_nm is produced `block_rows` rows
// at a time by the Gram kernel and never exists as a whole (n ~ 10^6 rows).
struct NysSource {
  const double* K_nm = nullptr;   // resident [n][ld_nm]
  int64_t ld_nm = 0;
  const double* X = nullptr;      // streamed: [n][ldx] training matrix, Xl [m][ldxl] its landmark rows
  int64_t p = 0, ldx = 0;
  const double* Xl = nullptr;
  int64_t ldxl = 0;
  double sigma = 0.0;
  int64_t block_rows = 0;         // 0 = default
};

constexpr int64_t NYS_BLOCK_ROWS = 32768;

__global__ void gather_rows_kernel(const double* __restrict__ X, int64_t ldx, const int64_t* __restrict__ idx, int p,
                                   double* __restrict__ out, int64_t ldo) {
  const double* src = X + idx[blockIdx.x] * ldx;
  for (int c = threadIdx.x; c < p; c += blockDim.x) out[(int64_t)blockIdx.x * ldo + c] = src[c];
}

// Peak device memory beyond the inputs: one [rp][ldn] array (Phi^T, overwritten block by block with U^T), the
// [n][ldr] array U Lam, and three blocks of block_rows rows.
static int setup_nystrom(int64_t n, int64_t m, const double* K_mm, int64_t ld_mm, const int64_t* landmark_idx,
                         const NysSource& src, tkm_spectral* s, cudaStream_t st) {
  const int64_t ldm = round_up(m, 16);
  s->n = n;
  s->m = m;
  s->ldm = ldm;
  s->ldn = round_up(n, 16);
  const int64_t nb_max = std::min<int64_t>(round_up(src.block_rows > 0 ? src.block_rows : NYS_BLOCK_ROWS, 16), s->ldn);
  // 1. K_mm = W Theta W^T
  DevBuf Wv, theta;
  TKM_TRY(Wv.alloc((size_t)m * ldm * sizeof(double), true, st));
  TKM_TRY(theta.alloc((size_t)ldm * sizeof(double), true, st));
  TKM_CUDA(cudaMemcpy2DAsync(Wv.p, ldm * sizeof(double), K_mm, ld_mm * sizeof(double), m * sizeof(double), m,
                             cudaMemcpyDeviceToDevice, st));
  TKM_TRY(syevd_inplace(Wv.as<double>(), ldm, m, theta.as<double>(), st));
  std::vector<double> h_theta(m);
  TKM_CUDA(cudaMemcpyAsync(h_theta.data(), theta.p, m * sizeof(double), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaStreamSynchronize(st));
  int64_t k0 = 0;   // eigenvalues ascend: keep the suffix above the rank tolerance
  while (k0 < m && !(h_theta[k0] > NYS_RANK_TOL * h_theta[m - 1])) ++k0;
  const int64_t rp = m - k0;
  if (rp <= 0) return set_error(TKM_ESOLVER, "nystrom: K_mm has no positive eigenvalue");
  const int64_t ldrp = round_up(rp, 16);
  double* Wts = Wv.as<double>() + k0 * ldm;   // [rp][ldm]; rows become w_k / sqrt(theta_k)
  vec_op_kernel<<<(unsigned)ceil_div(rp, 256), 256, 0, st>>>(theta.as<double>() + k0, (int)rp, 1);
  TKM_LAUNCH_CHECK();
  row_scale_kernel<<<(unsigned)rp, 256, 0, st>>>(Wts, ldm, (int)rp, (int)m, theta.as<double>() + k0);
  TKM_LAUNCH_CHECK();
  // 2. Phi^T [rp][ldn] = Wts K_nm^T, one block of rows of K_nm at a time
  DevBuf PhiT, Kblk;
  TKM_TRY(PhiT.alloc((size_t)rp * s->ldn * sizeof(double), true, st));
  if (!src.K_nm) TKM_TRY(Kblk.alloc((size_t)nb_max * ldm * sizeof(double), true, st));
  for (int64_t b0 = 0; b0 < n; b0 += nb_max) {
    const int64_t nb = std::min(nb_max, n - b0);
    const double* Kb = src.K_nm ? src.K_nm + b0 * src.ld_nm : Kblk.as<double>();
    if (!src.K_nm)
      TKM_TRY(tkm_gram(src.X + b0 * src.ldx, nb, src.p, src.ldx, src.Xl, m, src.ldxl, src.sigma, TKM_F64, Kblk.p, ldm, st));
    TKM_TRY(dgemm_nt(Wts, ldm, Kb, src.K_nm ? src.ld_nm : ldm, PhiT.as<double>() + b0, s->ldn, rp, nb, m, st));
  }
  // 3. G = Phi^T Phi = Q Lam Q^T
  DevBuf G, lamv;
  TKM_TRY(G.alloc((size_t)rp * ldrp * sizeof(double), true, st));
  TKM_TRY(lamv.alloc((size_t)ldrp * sizeof(double), true, st));
  TKM_TRY(dgemm_nt(PhiT.as<double>(), s->ldn, PhiT.as<double>(), s->ldn, G.as<double>(), ldrp, rp, rp, n, st));
  TKM_TRY(syevd_inplace(G.as<double>(), ldrp, rp, lamv.as<double>(), st));
  std::vector<double> h_l(rp);
  TKM_CUDA(cudaMemcpyAsync(h_l.data(), lamv.p, rp * sizeof(double), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaStreamSynchronize(st));
  int64_t j0 = 0;
  while (j0 < rp && !(h_l[j0] > NYS_RANK_TOL * h_l[rp - 1])) ++j0;
  const int64_t r = rp - j0;
  if (r <= 0) return set_error(TKM_ESOLVER, "nystrom: Phi^T Phi has no positive eigenvalue");
  s->r = r;
  s->ldr = round_up(r, 16);
  const double* Qe = G.as<double>() + j0 * ldrp;   // [r][ldrp], rows = eigenvectors
  // 4. U^T [r][ldn] = Lam^-1/2 Qe Phi^T, block by block over Phi^T's own storage (r <= rp rows of it)
  TKM_TRY(s->lam.alloc((size_t)s->ldr * sizeof(double), true, st));
  TKM_TRY(s->u1.alloc((size_t)s->ldr * sizeof(double), true, st));
  TKM_CUDA(cudaMemcpyAsync(s->lam.p, lamv.as<double>() + j0, r * sizeof(double), cudaMemcpyDeviceToDevice, st));
  DevBuf isq, Phib;
  TKM_TRY(isq.alloc((size_t)r * sizeof(double), false, st));
  TKM_CUDA(cudaMemcpyAsync(isq.p, s->lam.p, r * sizeof(double), cudaMemcpyDeviceToDevice, st));
  vec_op_kernel<<<(unsigned)ceil_div(r, 256), 256, 0, st>>>(isq.as<double>(), (int)r, 1);
  TKM_LAUNCH_CHECK();
  TKM_TRY(Phib.alloc((size_t)nb_max * ldrp * sizeof(double), true, st));   // [nb][ldrp]: a block of Phi
  for (int64_t b0 = 0; b0 < n; b0 += nb_max) {
    const int64_t nb = std::min(nb_max, n - b0);
    TKM_TRY(transpose_scale_f64(PhiT.as<double>() + b0, s->ldn, rp, nb, nullptr, Phib.as<double>(), ldrp, st));
    TKM_TRY(dgemm_nt(Qe, ldrp, Phib.as<double>(), ldrp, PhiT.as<double>() + b0, s->ldn, r, nb, rp, st));
  }
  s->Ut.take(PhiT);
  row_scale_kernel<<<(unsigned)r, 256, 0, st>>>(s->Ut.as<double>(), s->ldn, (int)r, (int)n, isq.as<double>());
  TKM_LAUNCH_CHECK();
  // 5. landmark map: lmap_t[j][l] = sqrt(Lam_j) sum_k Qe[j][k] Wts[k][l]
  DevBuf WtsT;
  TKM_TRY(WtsT.alloc((size_t)m * ldrp * sizeof(double), true, st));
  TKM_TRY(transpose_scale_f64(Wts, ldm, rp, m, nullptr, WtsT.as<double>(), ldrp, st));
  TKM_TRY(s->lmap_t.alloc((size_t)r * ldm * sizeof(double), true, st));
  TKM_TRY(dgemm_nt(Qe, ldrp, WtsT.as<double>(), ldrp, s->lmap_t.as<double>(), ldm, r, m, rp, st));
  TKM_CUDA(cudaMemcpyAsync(isq.p, s->lam.p, r * sizeof(double), cudaMemcpyDeviceToDevice, st));   // -> sqrt(Lam)
  vec_op_kernel<<<(unsigned)ceil_div(r, 256), 256, 0, st>>>(isq.as<double>(), (int)r, 2);
  TKM_LAUNCH_CHECK();
  row_scale_kernel<<<(unsigned)r, 256, 0, st>>>(s->lmap_t.as<double>(), ldm, (int)r, (int)m, isq.as<double>());
  TKM_LAUNCH_CHECK();
  s->landmark_idx.assign(landmark_idx, landmark_idx + m);
  TKM_TRY(s->d_landmark_idx.alloc((size_t)m * sizeof(int64_t), false, st));
  TKM_CUDA(cudaMemcpyAsync(s->d_landmark_idx.p, s->landmark_idx.data(), m * sizeof(int64_t), cudaMemcpyHostToDevice, st));
  TKM_TRY(finish_spectral(s, st));   // synchronises: the temporaries above may now be freed
  return TKM_OK;
}

static int nystrom_x_impl(const double* X, int64_t n, int64_t p, int64_t ldx, double sigma, const int64_t* landmark_idx,
                          int64_t m, int64_t block_rows, tkm_spectral* s, cudaStream_t st) {
  const int64_t ldm = round_up(m, 16), ldxl = round_up(p, 2);
  DevBuf d_idx, Xl, Kmm;
  TKM_TRY(d_idx.alloc((size_t)m * sizeof(int64_t), false, st));
  TKM_TRY(Xl.alloc((size_t)m * ldxl * sizeof(double), true, st));
  TKM_TRY(Kmm.alloc((size_t)m * ldm * sizeof(double), true, st));
  TKM_CUDA(cudaMemcpyAsync(d_idx.p, landmark_idx, m * sizeof(int64_t), cudaMemcpyHostToDevice, st));
  gather_rows_kernel<<<(unsigned)m, 128, 0, st>>>(X, ldx, d_idx.as<int64_t>(), (int)p, Xl.as<double>(), ldxl);
  TKM_LAUNCH_CHECK();
  TKM_TRY(tkm_gram(Xl.p, m, p, ldxl, nullptr, 0, 0, sigma, TKM_F64, Kmm.p, ldm, st));
  NysSource src;
  src.X = X;
  src.p = p;
  src.ldx = ldx;
  src.Xl = Xl.as<double>();
  src.ldxl = ldxl;
  src.sigma = sigma;
  src.block_rows = block_rows;
  return setup_nystrom(n, m, Kmm.as<double>(), ldm, landmark_idx, src, s, st);   // synchronises before returning
}

}  // namespace tkm

extern "C" int tkm_spectral_setup(const void* K, int64_t n, int64_t ldk, const tkm_nystrom* ny,
                                  tkm_spectral** out, void* stream) {
  tkm::NvtxRange nvtx_range("tkm_spectral_setup");
  using namespace tkm;
  if (!out) return set_error(TKM_EINVAL, "tkm_spectral_setup: out is NULL");
  *out = nullptr;
  if (n <= 1 || n > (1 << 30)) return set_error(TKM_EINVAL, "tkm_spectral_setup: n out of range");
  if (!ny && (!K || ldk < n)) return set_error(TKM_EINVAL, "tkm_spectral_setup: K NULL or ldk < n");
  if (ny && (!ny->K_nm || !ny->K_mm || ny->m < 1 || ny->m > n || ny->ld_nm < ny->m || ny->ld_mm < ny->m ||
             !ny->landmark_idx))
    return set_error(TKM_EINVAL, "tkm_spectral_setup: bad tkm_nystrom fields");
  if (ny) {
    if ((ny->ld_nm & 1) || (ny->ld_mm & 1))
      return set_error(TKM_EINVAL, "tkm_spectral_setup: ld_nm and ld_mm must be even (the TMA operands need 16-byte aligned rows); "
                                   "pad K_nm / K_mm to an even leading dimension");
    for (int64_t j = 0; j < ny->m; ++j)
      if (ny->landmark_idx[j] < 0 || ny->landmark_idx[j] >= n)
        return set_error(TKM_EINVAL, "tkm_spectral_setup: landmark_idx[%lld] = %lld is outside [0, n)", (long long)j,
                         (long long)ny->landmark_idx[j]);
  }
  TKM_TRY(device_check());
  cudaStream_t st = (cudaStream_t)stream;
  tkm_spectral* s = new (std::nothrow) tkm_spectral();
  if (!s) return set_error(TKM_ENOMEM, "out of host memory");
  int rc;
  if (ny) {
    NysSource src;
    src.K_nm = ny->K_nm;
    src.ld_nm = ny->ld_nm;
    rc = setup_nystrom(n, ny->m, ny->K_mm, ny->ld_mm, ny->landmark_idx, src, s, st);
  } else {
    rc = setup_full((const double*)K, n, ldk, s, st);
  }
  if (rc != TKM_OK) {
    cudaStreamSynchronize(st);
    delete s;
    return rc;
  }
  *out = s;
  return TKM_OK;
}

// Nystrom setup straight from the training matrix: the landmark rows are gathered, K_mm is formed, and K_nm is
// produced and consumed block_rows rows at a time (never resident).
extern "C" int tkm_spectral_setup_nystrom_x(const void* X, int64_t n, int64_t p, int64_t ldx, double sigma,
                                            const int64_t* landmark_idx, int64_t m, int64_t block_rows,
                                            tkm_spectral** out, void* stream) {
  tkm::NvtxRange nvtx_range("tkm_spectral_setup_nystrom_x");
  using namespace tkm;
  if (!out) return set_error(TKM_EINVAL, "tkm_spectral_setup_nystrom_x: out is NULL");
  *out = nullptr;
  if (!X || !landmark_idx || n <= 1 || n > (1 << 30) || p < 1 || p > (1 << 24) || ldx < p || m < 1 || m > n ||
      !(sigma > 0.0) || block_rows < 0)
    return set_error(TKM_EINVAL, "tkm_spectral_setup_nystrom_x: bad arguments");
  for (int64_t i = 0; i < m; ++i)
    if (landmark_idx[i] < 0 || landmark_idx[i] >= n)
      return set_error(TKM_EINVAL, "tkm_spectral_setup_nystrom_x: landmark index out of range");
  TKM_TRY(device_check());
  cudaStream_t st = (cudaStream_t)stream;
  tkm_spectral* s = new (std::nothrow) tkm_spectral();
  if (!s) return set_error(TKM_ENOMEM, "out of host memory");
  int rc = nystrom_x_impl((const double*)X, n, p, ldx, sigma, landmark_idx, m, block_rows, s, st);
  if (rc != TKM_OK) {
    cudaStreamSynchronize(st);
    delete s;
    return rc;
  }
  *out = s;
  return TKM_OK;
}

namespace tkm {
// Persistent set-up workers: one host thread per (device, index), created on first use and kept for the life of the
// process, each with its own non-blocking stream and its own cuSOLVER handle.  Starting a thread per decomposition
// and binding it to the device cost nothing on average but stalled for 0.1-1 s in one call out of five on shared
// boxes (profiles/r02_host_stalls.md); a parked thread that is woken by a condition variable does not.
class SetupWorker {
 public:
  SetupWorker(int dev, int idx) : dev_(dev), idx_(idx) {
    std::thread([this] { run(); }).detach();
  }
  void submit(std::function<void(cudaStream_t)> f) {
    std::lock_guard<std::mutex> lk(mu_);
    job_ = std::move(f);
    state_ = 1;
    cv_.notify_all();
  }
  void wait() {
    std::unique_lock<std::mutex> lk(mu_);
    cv_.wait(lk, [&] { return state_ == 0; });
  }

 private:
  void run() {
    Solver::thread_keeps_handle() = true;
    bool ok = cudaSetDevice(dev_) == cudaSuccess;
    cudaStream_t st = ok ? lib_worker_stream(idx_) : nullptr;
    for (;;) {
      std::unique_lock<std::mutex> lk(mu_);
      cv_.wait(lk, [&] { return state_ == 1; });
      std::function<void(cudaStream_t)> f = std::move(job_);
      lk.unlock();
      f(st);   // st == NULL: the job reports the failure
      lk.lock();
      state_ = 0;
      cv_.notify_all();
    }
  }
  int dev_, idx_;
  std::mutex mu_;
  std::condition_variable cv_;
  std::function<void(cudaStream_t)> job_;
  int state_ = 0;   // 0 idle, 1 job pending or running
};

// the workers of the current device (never destroyed: their threads are parked in run()); `call_mu` serialises
// concurrent tkm_spectral_setup_multi calls on one device
struct SetupWorkers {
  std::mutex call_mu;
  SetupWorker* w[64] = {};
};
static SetupWorkers* setup_workers(int dev) {
  static std::mutex mu;
  static SetupWorkers* per_dev[64] = {};
  if (dev < 0 || dev >= 64) return nullptr;
  std::lock_guard<std::mutex> lk(mu);
  if (!per_dev[dev]) per_dev[dev] = new (std::nothrow) SetupWorkers();
  return per_dev[dev];
}
}  // namespace tkm

// G full-kernel setups side by side: a dense symmetric eigensolver spends much of its time in phases that
// cannot fill the device (panel factorisations, the divide-and-conquer merge tree), so G decompositions
// on G streams, driven by G host threads, overlap almost perfectly.
extern "C" int tkm_spectral_setup_multi(const void* const* Ks, int32_t G, int64_t n, int64_t ldk,
                                        tkm_spectral** out, void* stream) {
  tkm::NvtxRange nvtx_range("tkm_spectral_setup_multi");
  using namespace tkm;
  if (!out || !Ks || G < 1 || G > 64) return set_error(TKM_EINVAL, "tkm_spectral_setup_multi: bad arguments");
  for (int g = 0; g < G; ++g) out[g] = nullptr;
  TKM_TRY(device_check());
  int dev = 0;
  TKM_CUDA(cudaGetDevice(&dev));
  cudaStream_t st = (cudaStream_t)stream;
  cudaEvent_t ready;
  TKM_CUDA(cudaEventCreateWithFlags(&ready, cudaEventDisableTiming));
  std::vector<int> rc(G, TKM_OK);
  std::vector<std::string> msg(G);
  std::vector<int64_t> launches(G, 0);
  if (n <= 1 || n > (1 << 30) || ldk < n) {
    cudaEventDestroy(ready);
    return set_error(TKM_EINVAL, "tkm_spectral_setup_multi: bad n / ldk");
  }
  for (int g = 0; g < G; ++g) {   // every allocation happens here, before the concurrent part
    out[g] = new (std::nothrow) tkm_spectral();
    int a = out[g] && Ks[g] ? alloc_full(n, out[g], st) : set_error(TKM_EINVAL, "tkm_spectral_setup_multi: NULL matrix");
    if (a != TKM_OK) {
      for (int h = 0; h <= g; ++h) {
        delete out[h];
        out[h] = nullptr;
      }
      cudaEventDestroy(ready);
      return a;
    }
  }
  cudaEventRecord(ready, st);   // K ready and the zero fills of the new buffers done
  SetupWorkers* sw = setup_workers(dev);
  if (!sw) {
    cudaEventDestroy(ready);
    for (int g = 0; g < G; ++g) {
      delete out[g];
      out[g] = nullptr;
    }
    return set_error(TKM_ECUDA, "tkm_spectral_setup_multi: device ordinal %d outside 0..63", dev);
  }
  {
    std::lock_guard<std::mutex> call_lock(sw->call_mu);
    for (int g = 0; g < G; ++g) {
      if (!sw->w[g]) sw->w[g] = new SetupWorker(dev, g);
      sw->w[g]->submit([&, g](cudaStream_t s2) {
        if (!s2) {
          rc[g] = TKM_ECUDA;
          msg[g] = "tkm_spectral_setup_multi: could not create a stream";
          return;
        }
        const int64_t before = launch_counter();
        cudaStreamWaitEvent(s2, ready, 0);
        rc[g] = compute_full((const double*)Ks[g], n, ldk, out[g], s2);   // synchronises s2
        if (rc[g] != TKM_OK) msg[g] = err_buf();
        launches[g] = launch_counter() - before;
      });
    }
    for (int g = 0; g < G; ++g) sw->w[g]->wait();
  }
  cudaEventDestroy(ready);
  int bad = TKM_OK;
  for (int g = 0; g < G; ++g) {
    count_launch(launches[g]);
    if (rc[g] != TKM_OK && bad == TKM_OK) bad = set_error(rc[g], "%s", msg[g].c_str());
  }
  if (bad != TKM_OK)
    for (int g = 0; g < G; ++g) {
      delete out[g];
      out[g] = nullptr;
    }
  return bad;
}

extern "C" void tkm_spectral_free(tkm_spectral* s) { delete s; }

extern "C" int tkm_spectral_info(const tkm_spectral* s, int64_t* n, int64_t* r, double* lam, double* u1) {
  using namespace tkm;
  if (!s) return set_error(TKM_EINVAL, "tkm_spectral_info: NULL handle");
  if (n) *n = s->n;
  if (r) *r = s->r;
  if (lam) memcpy(lam, s->h_lam.data(), s->r * sizeof(double));
  if (u1) memcpy(u1, s->h_u1.data(), s->r * sizeof(double));
  return TKM_OK;
}

extern "C" int tkm_spectral_get_u(const tkm_spectral* s, double* U_out, void* stream) {
  using namespace tkm;
  if (!s || !U_out) return set_error(TKM_EINVAL, "tkm_spectral_get_u: NULL argument");
  return transpose_scale_f64(s->Ut.as<double>(), s->ldn, s->r, s->n, nullptr, U_out, s->r, (cudaStream_t)stream);
}

