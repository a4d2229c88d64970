// lst_index_static.cu -- lst_index_hits_static (include/lst_static.h): step a0 (hits grouped by sensor
// in canonical order) for callers that may not allocate GPU memory.
//
// The regular a0 kernels (k_common.cu: k_hist / k_scatter / k_rank) keep their intermediate arrays in
// the slot workspace that lst_bind_workspace is given.  The kernels here do the same three steps with
// the same fp32 key arithmetic, but their intermediates sit in ONE fixed array that is part of the
// library image, so the call needs no workspace, no context and no allocation.  Nothing in this file
// is used by, or changes, the regular path.
//
// Rules of the fixed array (repeated for whoever edits this file):
//   * in HOST code the name `lst_static_scratch` is only a handle.  It is not a device address; a
//     kernel handed `lst_static_scratch` from the host would fault (or scribble over host memory on
//     a system with unified addressing).  The host obtains the real address once per GPU with
//     cudaGetSymbolAddress, with that GPU current, and passes the returned pointer to the kernels.
//   * the array holds whatever the previous call left; the counter block is cleared at the start of
//     every call, the other blocks are fully overwritten before they are read.
//   * all calls on a GPU share it: calls that overlap on the GPU race (documented in lst_static.h).
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "../../include/lst_static.h"

namespace {

constexpr uint32_t kMaxHits = LST_STATIC_MAX_HITS;
constexpr uint32_t kMaxDets = LST_STATIC_MAX_DETS;
// word layout of the array: [counters: one per sensor | ticket of the last-block scan | padding]
// [arrival rank per hit] [caller index per unordered position] [azimuth key per unordered position]
constexpr uint32_t kTicketWord = kMaxDets;
constexpr uint32_t kZeroWords = kMaxDets + 64;          // cleared by every call (counters + ticket)
constexpr uint32_t kRankWord0 = kZeroWords;
constexpr uint32_t kOrigWord0 = kRankWord0 + kMaxHits;
constexpr uint32_t kKeyWord0 = kOrigWord0 + kMaxHits;
constexpr uint32_t kScratchWords = kKeyWord0 + kMaxHits;  // 852 032 words = 3.25 MiB
static_assert(kZeroWords % 64 == 0 && kMaxHits % 64 == 0, "every block of the array starts 256-byte aligned");

static __device__ __align__(256) uint32_t lst_static_scratch[kScratchWords];

constexpr int kHistThreads = 1024, kThreads = 256;
constexpr float kTwoPi = 6.2831853071795864769f, kInvTwoPi = 0.15915494309189533577f;

__device__ __forceinline__ uint32_t warp_excl(uint32_t v, uint32_t *total) {
  const int lane = threadIdx.x & 31;
  uint32_t x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
    if (lane >= o) x += y;
  }
  *total = __shfl_sync(0xffffffffu, x, 31);
  return x - v;
}

// Step 1: every hit takes the next free place inside its sensor (arrival order; step 3 makes the
// order canonical).  The block that finishes last turns the counters into det_off.
__global__ void __launch_bounds__(kHistThreads) k_static_hist(uint32_t *scratch, const uint32_t *det, uint32_t n,
                                                               uint32_t n_dets, uint32_t *det_off, uint32_t *n_rejected) {
  __shared__ uint32_t sh_warp[32];
  __shared__ bool sh_last;
  uint32_t *cnt = scratch, *rank = scratch + kRankWord0;
  for (uint32_t h = blockIdx.x * blockDim.x + threadIdx.x; h < n; h += gridDim.x * blockDim.x) {
    const uint32_t d = det[h];
    if (d >= n_dets) { atomicAdd(n_rejected, 1u); continue; }
    rank[h] = atomicAdd(&cnt[d], 1u);
  }
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) sh_last = atomicAdd(&scratch[kTicketWord], 1u) == gridDim.x - 1u;
  __syncthreads();
  if (!sh_last) return;
  __threadfence();
  // exclusive scan of cnt[0 .. n_dets): thread t owns a contiguous run of `chunk` counters
  const uint32_t chunk = (n_dets + blockDim.x - 1) / blockDim.x;
  const uint32_t b0 = min(n_dets, threadIdx.x * chunk), b1 = min(n_dets, b0 + chunk);
  uint32_t sum = 0;
  for (uint32_t i = b0; i < b1; ++i) sum += __ldcg(&cnt[i]);
  uint32_t wtot;
  uint32_t e = warp_excl(sum, &wtot);
  if ((threadIdx.x & 31) == 31) sh_warp[threadIdx.x >> 5] = wtot;
  __syncthreads();
  if (threadIdx.x < 32) {
    uint32_t t;
    const uint32_t v = threadIdx.x < (blockDim.x >> 5) ? sh_warp[threadIdx.x] : 0u;
    sh_warp[threadIdx.x] = warp_excl(v, &t);
  }
  __syncthreads();
  e += sh_warp[threadIdx.x >> 5];
  for (uint32_t i = b0; i < b1; ++i) { det_off[i] = e; e += __ldcg(&cnt[i]); }
  if (b0 < n_dets && b1 == n_dets) det_off[n_dets] = e;
  if (n_dets == 0 && threadIdx.x == 0) det_off[0] = 0;
}

// Step 2: unordered copy (caller index + azimuth key) into the sensor's range.
__global__ void __launch_bounds__(kThreads) k_static_scatter(uint32_t *scratch, const float *x, const float *y,
                                                              const uint32_t *det, const float *phic, uint32_t n,
                                                              uint32_t n_dets, const uint32_t *det_off) {
  const uint32_t *rank = scratch + kRankWord0;
  uint32_t *orig = scratch + kOrigWord0;
  float *key = reinterpret_cast<float *>(scratch + kKeyWord0);
  for (uint32_t h = blockIdx.x * blockDim.x + threadIdx.x; h < n; h += gridDim.x * blockDim.x) {
    const uint32_t d = det[h];
    if (d >= n_dets) continue;
    const uint32_t p = det_off[d] + rank[h];
    orig[p] = h;
    const float dphi = atan2f(y[h], x[h]) - phic[d >> 1];
    const float k = dphi - kTwoPi * rintf(dphi * kInvTwoPi);
    key[p] = k == k ? k : 0.0f;
  }
}

// Step 3: position of a hit inside its sensor = hits of the sensor with a smaller (key, caller index).
__global__ void __launch_bounds__(kThreads) k_static_rank(const uint32_t *scratch, const float *x, const float *y,
                                                           const float *z, const uint32_t *det, uint32_t n_dets,
                                                           const uint32_t *det_off, uint32_t *hit_orig, float4 *hit_xyzr) {
  const uint32_t *orig = scratch + kOrigWord0;
  const float *key = reinterpret_cast<const float *>(scratch + kKeyWord0);
  const uint32_t n = det_off[n_dets];
  for (uint32_t p = blockIdx.x * blockDim.x + threadIdx.x; p < n; p += gridDim.x * blockDim.x) {
    const uint32_t h = orig[p];
    const uint32_t d = det[h];
    const uint32_t b = det_off[d], e = det_off[d + 1];
    const float k = key[p];
    uint32_t r = 0;
    for (uint32_t q = b; q < e; ++q) {
      const float kq = key[q];
      r += (kq < k || (kq == k && orig[q] < h));
    }
    const float hx = x[h], hy = y[h], hz = z[h];
    hit_xyzr[b + r] = make_float4(hx, hy, hz, sqrtf(hx * hx + hy * hy));
    hit_orig[b + r] = h;
  }
}

// ---- per-GPU set-up: device address of the array and the SM count, looked up on the first call
constexpr int kMaxGpus = 64;
struct PerGpu {
  uint32_t *scratch = nullptr;
  int n_sm = 0;
};
std::mutex g_mu;
PerGpu g_gpu[kMaxGpus];

int fail(int status, char *errbuf, size_t len, const char *fmt, ...) {
  if (errbuf && len) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(errbuf, len, fmt, ap);
    va_end(ap);
  }
  return status;
}

int setup_current_gpu(PerGpu *out, char *errbuf, size_t len) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(LST_ECUDA, errbuf, len, "lst_index_hits_static: cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= kMaxGpus) return fail(LST_EINVAL, errbuf, len, "lst_index_hits_static: device ordinal %d not supported (< %d)", dev, kMaxGpus);
  std::lock_guard<std::mutex> lock(g_mu);
  PerGpu &g = g_gpu[dev];
  if (!g.scratch) {
    // the symbol is a host-side handle: ask the runtime where the array lives on THIS gpu
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, lst_static_scratch);
    if (e != cudaSuccess || !p)
      return fail(LST_ECUDA, errbuf, len, "lst_index_hits_static: cudaGetSymbolAddress on device %d: %s", dev, cudaGetErrorString(e));
    int n_sm = 0;
    e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess || n_sm <= 0)
      return fail(LST_ECUDA, errbuf, len, "lst_index_hits_static: SM count of device %d: %s", dev, cudaGetErrorString(e));
    g.n_sm = n_sm;
    g.scratch = static_cast<uint32_t *>(p);
  }
  *out = g;
  return LST_OK;
}

int blocks_for(uint32_t n, int threads, int max_blocks) {
  long b = ((long)n + threads - 1) / threads;
  if (b < 1) b = 1;
  return (int)(b > max_blocks ? max_blocks : b);
}

}  // namespace

extern "C" int lst_index_hits_static(const float *x, const float *y, const float *z, const uint32_t *det, uint32_t n_hits,
                                     const float *phic, uint32_t n_dets, uint32_t *det_off, uint32_t *hit_orig,
                                     float *hit_xyzr, uint32_t *n_rejected, void *cuda_stream, char *errbuf,
                                     size_t errbuf_len) {
  if (n_hits > kMaxHits)
    return fail(LST_EINVAL, errbuf, errbuf_len,
                "lst_index_hits_static: %u hits exceed LST_STATIC_MAX_HITS = %u (the fixed scratch array cannot grow; use "
                "lst_create / lst_bind_workspace for larger events)", n_hits, kMaxHits);
  if (n_dets > kMaxDets)
    return fail(LST_EINVAL, errbuf, errbuf_len,
                "lst_index_hits_static: %u sensors exceed LST_STATIC_MAX_DETS = %u (the fixed scratch array cannot grow)",
                n_dets, kMaxDets);
  if (n_dets & 1u) return fail(LST_EINVAL, errbuf, errbuf_len, "lst_index_hits_static: n_dets = %u is odd (2 sensors per module)", n_dets);
  if (!det_off || !n_rejected || (n_dets && !phic))
    return fail(LST_EINVAL, errbuf, errbuf_len, "lst_index_hits_static: null det_off, n_rejected or phic");
  if (n_hits && (!x || !y || !z || !det || !hit_orig || !hit_xyzr))
    return fail(LST_EINVAL, errbuf, errbuf_len, "lst_index_hits_static: null hit array with n_hits = %u", n_hits);
  if (reinterpret_cast<uintptr_t>(hit_xyzr) & 15u)
    return fail(LST_EINVAL, errbuf, errbuf_len, "lst_index_hits_static: hit_xyzr is not 16-byte aligned");
  PerGpu g;
  const int rc = setup_current_gpu(&g, errbuf, errbuf_len);
  if (rc != LST_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  cudaError_t e = cudaMemsetAsync(g.scratch, 0, sizeof(uint32_t) * kZeroWords, st);
  if (e == cudaSuccess) e = cudaMemsetAsync(n_rejected, 0, sizeof(uint32_t), st);
  if (e != cudaSuccess) return fail(LST_ECUDA, errbuf, errbuf_len, "lst_index_hits_static: cudaMemsetAsync: %s", cudaGetErrorString(e));
  k_static_hist<<<blocks_for(n_hits, kHistThreads, g.n_sm * 2), kHistThreads, 0, st>>>(g.scratch, det, n_hits, n_dets, det_off,
                                                                                      n_rejected);
  const int nb = blocks_for(n_hits, kThreads, g.n_sm * 8);
  k_static_scatter<<<nb, kThreads, 0, st>>>(g.scratch, x, y, det, phic, n_hits, n_dets, det_off);
  k_static_rank<<<nb, kThreads, 0, st>>>(g.scratch, x, y, z, det, n_dets, det_off, hit_orig,
                                         reinterpret_cast<float4 *>(hit_xyzr));
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(LST_ECUDA, errbuf, errbuf_len, "lst_index_hits_static: kernel launch: %s", cudaGetErrorString(e));
  return LST_OK;
}
