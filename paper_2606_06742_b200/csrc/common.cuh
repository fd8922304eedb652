// common.cuh -- shared host/device helpers of libtkm (error handling, launch counting, PTX wrappers).
#pragma once

#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>
#include <cstdarg>
#include <cstdint>
#include <cstdlib>
#include <cstdio>
#include <cstring>
#include <atomic>
#include <mutex>
#include <vector>

#include "../../include/tkm.h"

namespace tkm {

// ---- thread-local error string + launch counter (tkm_last_error / tkm_launch_count) ----------
char* err_buf();
int set_error(int code, const char* fmt, ...);
int64_t& launch_counter();
inline void count_launch(int64_t k = 1) { launch_counter() += k; }

#define TKM_CUDA(expr)                                                                       \
  do {                                                                                       \
    cudaError_t _e = (expr);                                                                 \
    if (_e != cudaSuccess)                                                                   \
      return ::tkm::set_error(_e == cudaErrorMemoryAllocation ? TKM_ENOMEM : TKM_ECUDA,      \
                              "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e),        \
                              __FILE__, __LINE__);                                           \
  } while (0)

#define TKM_LAUNCH_CHECK()                                                                   \
  do {                                                                                       \
    ::tkm::count_launch();                                                                   \
    cudaError_t _e = cudaGetLastError();                                                     \
    if (_e != cudaSuccess)                                                                   \
      return ::tkm::set_error(TKM_ECUDA, "kernel launch failed: %s (%s:%d)",                 \
                              cudaGetErrorString(_e), __FILE__, __LINE__);                   \
  } while (0)

#define TKM_TRY(expr)                 \
  do {                                \
    int _s = (expr);                  \
    if (_s != TKM_OK) return _s;      \
  } while (0)

// NVTX range of one pipeline stage (visible to nsys / ncu --nvtx; a no-op without a tool attached)
struct NvtxRange {
  explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
  ~NvtxRange() { nvtxRangePop(); }
  NvtxRange(const NvtxRange&) = delete;
  NvtxRange& operator=(const NvtxRange&) = delete;
};

inline int64_t round_up(int64_t x, int64_t m) { return (x + m - 1) / m * m; }
inline int64_t ceil_div(int64_t x, int64_t m) { return (x + m - 1) / m; }

// The library's own stream-ordered memory pool of the current device (created on first use; the device's default
// pool is never touched).  It keeps up to 8 GiB of freed allocations, so that the temporaries of one sweep are
// handed to the next without a trip through the driver's page tables.  NULL on failure.
cudaMemPool_t lib_pool();

// Worker stream `i` (0..63) of the current device: non-blocking streams the library creates once per device and keeps
// (tkm_spectral_setup_multi runs its G decompositions on them).  NULL on failure.
cudaStream_t lib_worker_stream(int i);

// RAII device buffer, zero-initialised on request.  All memory comes from the library's pool (lib_pool), so that
// after the first step no allocation or free goes through the kernel-mode driver (on shared boxes those calls stall
// for 0.3-0.8 s at random: profiles/r02_host_stalls.md).  Two lifetimes:
//   pool = true  : a temporary of ONE stream -- stream-ordered cudaFreeAsync on the allocating stream;
//   pool = false : memory of a handle (tkm_spectral, tkm_path) or of a call that synchronises before it returns --
//                  released at an arbitrary later time from an arbitrary thread, so release() first waits for the
//                  device (what cudaFree does implicitly) and then returns the block to the pool.  The memory is
//                  valid in stream order of the allocating stream `st`: other streams must depend on `st` (they do:
//                  every producer of a handle runs on the call's stream or waits for an event recorded on it).
// Without a pool (cudaMemPoolCreate failed) it falls back to cudaMalloc / cudaFree.
struct DevBuf {
  void* p = nullptr;
  size_t bytes = 0;
  bool pooled = false;       // stream-ordered temporary
  bool from_pool = false;    // handle lifetime, but allocated from the pool
  int dev = -1;
  cudaStream_t pool_st = nullptr;
  DevBuf() = default;
  DevBuf(const DevBuf&) = delete;
  DevBuf& operator=(const DevBuf&) = delete;
  ~DevBuf() { release(); }
  void release() {
    if (p) {
      if (pooled) {
        cudaFreeAsync(p, pool_st);
      } else if (from_pool) {
        int cur = -1;
        cudaGetDevice(&cur);
        if (cur != dev && dev >= 0) cudaSetDevice(dev);
        cudaDeviceSynchronize();
        if (cudaFreeAsync(p, (cudaStream_t)0) != cudaSuccess) cudaGetLastError();
        if (cur != dev && cur >= 0) cudaSetDevice(cur);
      } else {
        cudaFree(p);
      }
    }
    p = nullptr;
    bytes = 0;
    pooled = from_pool = false;
  }
  int alloc(size_t nbytes, bool zero, cudaStream_t st, bool pool = false) {
    release();
    if (nbytes == 0) nbytes = 16;
    cudaMemPool_t mp = lib_pool();
    cudaError_t e;
    if (pool)
      e = mp ? cudaMallocFromPoolAsync(&p, nbytes, mp, st) : cudaMallocAsync(&p, nbytes, st);
    else
      e = mp ? cudaMallocFromPoolAsync(&p, nbytes, mp, st) : cudaMalloc(&p, nbytes);
    if (e != cudaSuccess) {
      p = nullptr;
      return set_error(TKM_ENOMEM, "device allocation of %zu bytes failed: %s", nbytes, cudaGetErrorString(e));
    }
    bytes = nbytes;
    pooled = pool;
    from_pool = !pool && mp != nullptr;
    pool_st = st;
    cudaGetDevice(&dev);
    if (zero) {
      e = cudaMemsetAsync(p, 0, nbytes, st);
      if (e != cudaSuccess) return set_error(TKM_ECUDA, "cudaMemsetAsync failed: %s", cudaGetErrorString(e));
    }
    return TKM_OK;
  }
  void take(DevBuf& o) {   // move o's allocation here
    release();
    p = o.p;
    bytes = o.bytes;
    pooled = o.pooled;
    from_pool = o.from_pool;
    dev = o.dev;
    pool_st = o.pool_st;
    o.p = nullptr;
    o.bytes = 0;
    o.pooled = o.from_pool = false;
  }
  template <class T>
  T* as() const { return reinterpret_cast<T*>(p); }
};

// Pinned host buffer.
struct PinBuf {
  void* p = nullptr;
  ~PinBuf() {
    if (p) cudaFreeHost(p);
  }
  int alloc(size_t nbytes) {
    if (p) cudaFreeHost(p);
    p = nullptr;
    cudaError_t e = cudaMallocHost(&p, nbytes ? nbytes : 16);
    if (e != cudaSuccess) {
      p = nullptr;
      return set_error(TKM_ENOMEM, "cudaMallocHost(%zu) failed: %s", nbytes, cudaGetErrorString(e));
    }
    return TKM_OK;
  }
  template <class T>
  T* as() const { return reinterpret_cast<T*>(p); }
};

int device_check();   // TKM_OK when a CUDA device of compute capability 10.x is current

// true the first time it is called for (this flag word, the current device): per-device one-time kernel setup
// (cudaFuncSetAttribute) without a process-wide "configured" bool
inline bool first_use_on_device(std::atomic<unsigned long long>& done) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return true;
  const unsigned long long bit = 1ull << dev;
  return (done.fetch_or(bit) & bit) == 0;
}

#ifdef __CUDACC__
// ---- device-side PTX wrappers ------------------------------------------------------------------
// 16-byte async copy; only the first `src_bytes` (0, 8 or 16) are read, the rest is zero-filled.
__device__ __forceinline__ void cp_async_16(void* smem_dst, const void* gmem_src, int src_bytes) {
  unsigned s = static_cast<unsigned>(__cvta_generic_to_shared(smem_dst));
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem_src), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}

// D(8x8) += A(8x4, row) * B(4x8, col), FP64 tensor core (SASS: DMMA.8x8x4).
__device__ __forceinline__ void dmma_884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Block-wide sum (all threads get the result); `red` holds >= 32 doubles of shared memory.
__device__ __forceinline__ double block_sum(double v, double* red) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  v = warp_sum(v);
  __syncthreads();   // protect `red` from a previous use
  if (lane == 0) red[w] = v;
  __syncthreads();
  double t = (lane < nw) ? red[lane] : 0.0;
  t = warp_sum(t);
  return t;
}
#endif  // __CUDACC__

}  // namespace tkm
