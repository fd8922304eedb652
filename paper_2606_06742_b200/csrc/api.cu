// api.cu -- library-wide plumbing of the C ABI: error string, launch counter, device check, the
// integer-only fold generator and the whole-pipeline host entry point.
#include <cstdarg>
#include <new>

#include "handles.cuh"

namespace tkm {

char* err_buf() {
  static thread_local char buf[512] = {0};
  return buf;
}

int set_error(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(err_buf(), 512, fmt, ap);
  va_end(ap);
  return code;
}

int64_t& launch_counter() {
  static thread_local int64_t c = 0;
  return c;
}

cudaMemPool_t lib_pool() {
  static std::mutex mu;
  static cudaMemPool_t pools[64] = {};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) {
    cudaGetLastError();
    return nullptr;
  }
  std::lock_guard<std::mutex> lock(mu);
  if (!pools[dev]) {
    cudaMemPoolProps props = {};
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = dev;
    cudaMemPool_t mp = nullptr;
    if (cudaMemPoolCreate(&mp, &props) != cudaSuccess) {
      cudaGetLastError();
      return nullptr;
    }
    uint64_t keep = 8ull << 30;
    cudaMemPoolSetAttribute(mp, cudaMemPoolAttrReleaseThreshold, &keep);
    pools[dev] = mp;
  }
  return pools[dev];
}

cudaStream_t lib_worker_stream(int i) {
  static std::mutex mu;
  static cudaStream_t streams[64][64] = {};
  int dev = 0;
  if (i < 0 || i >= 64 || cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) {
    cudaGetLastError();
    return nullptr;
  }
  std::lock_guard<std::mutex> lock(mu);
  if (!streams[dev][i] && cudaStreamCreateWithFlags(&streams[dev][i], cudaStreamNonBlocking) != cudaSuccess) {
    cudaGetLastError();
    streams[dev][i] = nullptr;
  }
  return streams[dev][i];
}

int device_check() {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) {
    cudaGetLastError();
    return set_error(TKM_ECUDA, "no CUDA device: %s (libtkm has no CPU fallback)", cudaGetErrorString(e));
  }
  static thread_local int checked_dev = -1;
  if (checked_dev == dev) return TKM_OK;
  int major = 0;
  e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
  if (e != cudaSuccess) return set_error(TKM_ECUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
  if (major != 10)
    return set_error(TKM_ECUDA, "libtkm is built for sm_100a only; device %d has compute capability %d.x", dev, major);
  checked_dev = dev;
  return TKM_OK;
}

}  // namespace tkm

using namespace tkm;

extern "C" int tkm_version(void) { return TKM_VERSION_MAJOR * 100 + TKM_VERSION_MINOR; }
extern "C" const char* tkm_last_error(void) { return err_buf(); }
extern "C" int64_t tkm_launch_count(void) { return launch_counter(); }
extern "C" void tkm_launch_count_reset(void) { launch_counter() = 0; }

// SplitMix64 (Steele, Lea, Flood 2014) -> Fisher-Yates -> round-robin fold labels (reading G13).
extern "C" int tkm_make_folds(int64_t n, int32_t V, uint64_t seed, int32_t* foldid) {
  if (!foldid) return set_error(TKM_EINVAL, "tkm_make_folds: foldid is NULL");
  if (V < 2 || (int64_t)V > n) return set_error(TKM_EINVAL, "tkm_make_folds: need 2 <= V <= n");
  std::vector<int64_t> pi((size_t)n);
  for (int64_t i = 0; i < n; ++i) pi[i] = i;
  uint64_t x = seed;
  for (int64_t i = n - 1; i >= 1; --i) {
    x += 0x9E3779B97F4A7C15ull;
    uint64_t z = x;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    z ^= z >> 31;
    const int64_t j = (int64_t)(z % (uint64_t)(i + 1));
    std::swap(pi[i], pi[j]);
  }
  for (int64_t i = 0; i < n; ++i) foldid[pi[i]] = (int32_t)(i % V);
  return TKM_OK;
}

// fold sizes of a fold assignment (integer-only host helper; the weights of tkm_cv_select)
extern "C" int tkm_fold_sizes(const int32_t* foldid, int64_t n, int32_t V, double* sizes) {
  if (!foldid || !sizes || n < 1 || V < 1) return set_error(TKM_EINVAL, "tkm_fold_sizes: bad arguments");
  for (int v = 0; v < V; ++v) sizes[v] = 0.0;
  for (int64_t j = 0; j < n; ++j) {
    if (foldid[j] < 0 || foldid[j] >= V) return set_error(TKM_EINVAL, "tkm_fold_sizes: foldid[%lld] out of range", (long long)j);
    sizes[foldid[j]] += 1.0;
  }
  return TKM_OK;
}

extern "C" int tkm_train_tune_host(const double* X, int64_t n, int64_t p, const double* y, const double* sigmas,
                                   int32_t G, tkm_loss loss, const tkm_loss_opts* opts, const double* lambdas,
                                   int32_t L, const int32_t* foldid, int32_t V, double tol, int32_t maxit,
                                   double* cv_loss, int64_t* cv_err, double* cv_mean,
                                   int32_t* best_l, double* alpha_best, double* beta0_best, float* stage_ms,
                                   void* stream) {
  if (!X || !y || !sigmas || !opts || !lambdas || !foldid || !cv_loss || !cv_mean || !best_l)
    return set_error(TKM_EINVAL, "tkm_train_tune_host: NULL argument");
  if (n <= 1 || p <= 0 || G < 1 || G > 8 || L < 1 || V < 2) return set_error(TKM_EINVAL, "tkm_train_tune_host: bad n / p / G / L / V");
  TKM_TRY(device_check());
  cudaStream_t st = (cudaStream_t)stream;
  cudaEvent_t ev[6];
  for (auto& e : ev) TKM_CUDA(cudaEventCreate(&e));
  struct Owner {   // everything that must be released on every exit path
    cudaEvent_t* e;
    tkm_spectral* spec[8] = {};
    tkm_path* path[8] = {};
    ~Owner() {
      for (int i = 0; i < 6; ++i) cudaEventDestroy(e[i]);
      for (auto* q : path) tkm_path_free(q);
      for (auto* q : spec) tkm_spectral_free(q);
    }
  } own{ev};
  const int T = loss == TKM_LOSS_QUANTILE ? (opts->T > 0 ? opts->T : 1) : 1;
  DevBuf dX, dy, dK, dalpha;
  TKM_CUDA(cudaEventRecord(ev[0], st));
  TKM_TRY(dX.alloc((size_t)n * p * sizeof(double), false, st));
  TKM_TRY(dy.alloc((size_t)n * sizeof(double), false, st));
  TKM_TRY(dK.alloc((size_t)G * n * n * sizeof(double), false, st));
  TKM_CUDA(cudaMemcpyAsync(dX.p, X, (size_t)n * p * sizeof(double), cudaMemcpyHostToDevice, st));
  TKM_CUDA(cudaMemcpyAsync(dy.p, y, (size_t)n * sizeof(double), cudaMemcpyHostToDevice, st));
  TKM_CUDA(cudaEventRecord(ev[1], st));
  const void* Ks[8];
  void* Kw[8];
  for (int g = 0; g < G; ++g) Ks[g] = Kw[g] = dK.as<double>() + (size_t)g * n * n;
  TKM_TRY(tkm_gram_multi(dX.p, n, p, p, nullptr, 0, 0, sigmas, G, TKM_F64, Kw, n, st));
  TKM_CUDA(cudaEventRecord(ev[2], st));
  TKM_TRY(tkm_spectral_setup_multi(Ks, G, n, n, own.spec, st));   // the G decompositions overlap
  dK.release();
  TKM_CUDA(cudaEventRecord(ev[3], st));
  int rc = tkm_fit_path_multi(own.spec, G, dy.p, loss, opts, lambdas, L, foldid, V, tol, maxit, nullptr, own.path, st);
  if (rc != TKM_OK && rc != TKM_ENOTCONV) return rc;
  TKM_CUDA(cudaEventRecord(ev[4], st));
  if (alpha_best) TKM_TRY(dalpha.alloc((size_t)G * n * sizeof(double), false, st));
  for (int g = 0; g < G; ++g) {
    const size_t o3 = (size_t)g * T * L * V, o2 = (size_t)g * T * L, o1 = (size_t)g * T;
    TKM_TRY(tkm_exact_cv(own.path[g], dy.p, foldid, cv_loss + o3, cv_err ? cv_err + o3 : nullptr, cv_mean + o2,
                         best_l + o1, st));
    if (alpha_best)
      TKM_TRY(tkm_path_coef(own.path[g], 0, best_l[o1], V, dalpha.as<double>() + (size_t)g * n,
                            beta0_best ? beta0_best + g : nullptr, st));
  }
  if (alpha_best)
    TKM_CUDA(cudaMemcpyAsync(alpha_best, dalpha.p, (size_t)G * n * sizeof(double), cudaMemcpyDeviceToHost, st));
  TKM_CUDA(cudaEventRecord(ev[5], st));
  TKM_CUDA(cudaStreamSynchronize(st));
  if (stage_ms)
    for (int i = 0; i < 5; ++i) cudaEventElapsedTime(&stage_ms[i], ev[i], ev[i + 1]);
  return rc;
}
