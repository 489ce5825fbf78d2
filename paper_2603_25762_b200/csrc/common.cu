// libqhap: error text, device check, exclusive scan.
#include "common.cuh"

#include <stdarg.h>

#include <atomic>

namespace qhap {

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}

static std::atomic<uint64_t> g_launches{0};
void count_launches(uint64_t n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

// Per-device cache (a process may drive several devices): state 0 unknown, 1 sm_100 ok, -1 other architecture.
constexpr int kMaxDevices = 64;
struct DevInfo {
  std::atomic<int> state{0};
  std::atomic<int> sms{0};
};
static DevInfo g_dev[kMaxDevices];

static cudaError_t probe_device(int* dev_out, int* major, int* minor, int* sms) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(major, cudaDevAttrComputeCapabilityMajor, dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(minor, cudaDevAttrComputeCapabilityMinor, dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(sms, cudaDevAttrMultiProcessorCount, dev);
  *dev_out = dev;
  return e;
}

qhap_status require_device() {
  int dev = 0, major = 0, minor = 0, sms = 0;
  if (cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < kMaxDevices && g_dev[dev].state.load(std::memory_order_acquire) == 1)
    return QHAP_OK;
  const cudaError_t e = probe_device(&dev, &major, &minor, &sms);
  if (e != cudaSuccess) {
    set_error("no CUDA device: %s (libqhap has no CPU fallback)", cudaGetErrorString(e));
    (void)cudaGetLastError();
    return QHAP_ERR_CUDA;
  }
  if (major != 10) {
    set_error("device %d is sm_%d%d; libqhap is built for sm_100a only", dev, major, minor);
    return QHAP_ERR_CUDA;
  }
  if (dev >= 0 && dev < kMaxDevices) {
    g_dev[dev].sms.store(sms, std::memory_order_relaxed);
    g_dev[dev].state.store(1, std::memory_order_release);
  }
  return QHAP_OK;
}

int sm_count() {
  int dev = 0, major = 0, minor = 0, sms = 0;
  if (cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < kMaxDevices) {
    const int c = g_dev[dev].sms.load(std::memory_order_relaxed);
    if (c > 0) return c;
  }
  if (probe_device(&dev, &major, &minor, &sms) == cudaSuccess && sms > 0) {
    if (dev >= 0 && dev < kMaxDevices) g_dev[dev].sms.store(sms, std::memory_order_relaxed);
    return sms;
  }
  (void)cudaGetLastError();
  return 148;          // no device (size queries on a box without a GPU): B200's count, planning only
}

// ------------------------------------------------------------------------------------------------ scan
// One CTA of 1024 threads walks the array in tiles of 4096 counts, carrying the running total.
__global__ void __launch_bounds__(1024) scan_i32_kernel(const int32_t* __restrict__ in, int32_t* __restrict__ out,
                                                        int64_t n, int64_t* total_dev, int32_t* overflow_dev) {
  __shared__ int64_t warp_tot[32];
  __shared__ int64_t carry_s;
  const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
  if (t == 0) carry_s = 0;
  __syncthreads();
  for (int64_t base = 0; base < n; base += 4096) {
    int64_t i0 = base + int64_t(t) * 4;
    int32_t v[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) v[k] = (i0 + k < n) ? in[i0 + k] : 0;
    int64_t s = int64_t(v[0]) + v[1] + v[2] + v[3];
    int64_t incl = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int64_t u = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += u;
    }
    if (lane == 31) warp_tot[wid] = incl;
    __syncthreads();
    if (wid == 0) {
      int64_t w = warp_tot[lane];
      int64_t wi = w;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        int64_t u = __shfl_up_sync(0xffffffffu, wi, o);
        if (lane >= o) wi += u;
      }
      warp_tot[lane] = wi - w;  // exclusive prefix of the warp totals
    }
    __syncthreads();
    int64_t carry = carry_s;
    int64_t excl = carry + warp_tot[wid] + (incl - s);
    // tile total = prefix of the last thread + its sum
    __syncthreads();
    if (t == 1023) carry_s = excl + s;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      if (i0 + k < n) out[i0 + k] = int32_t(excl);
      excl += v[k];
    }
    __syncthreads();
  }
  if (t == 0) {
    int64_t tot = carry_s;
    out[n] = int32_t(tot);
    if (total_dev) *total_dev = tot;
    if (overflow_dev && tot > int64_t(0x7fffffff)) *overflow_dev = 1;
  }
}

// Three-kernel scan for long arrays (needs ceil(n / 4096) + 1 int64 of scratch): tile sums -> scan of the tile sums (one
// CTA) -> every tile rescans itself from its base.  In-place safe: a tile is read completely before it is written.
__global__ void __launch_bounds__(1024) scan_tile_sum_kernel(const int32_t* __restrict__ in, int64_t n, int64_t* __restrict__ tile_sum) {
  __shared__ int64_t warp_tot[32];
  const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
  const int64_t i0 = int64_t(blockIdx.x) * 4096 + int64_t(t) * 4;
  int64_t s = 0;
#pragma unroll
  for (int k = 0; k < 4; ++k) s += (i0 + k < n) ? in[i0 + k] : 0;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (lane == 0) warp_tot[wid] = s;
  __syncthreads();
  if (wid == 0) {
    int64_t w = warp_tot[lane];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) w += __shfl_xor_sync(0xffffffffu, w, o);
    if (lane == 0) tile_sum[blockIdx.x] = w;
  }
}

__global__ void __launch_bounds__(1024) scan_tile_base_kernel(int64_t* __restrict__ tile_sum, int64_t n_tiles, int32_t* __restrict__ out,
                                                              int64_t n, int64_t* total_dev, int32_t* overflow_dev) {
  if (threadIdx.x == 0) {                      // a few hundred tiles at most: a serial walk is a microsecond
    int64_t run = 0;
    for (int64_t b = 0; b < n_tiles; ++b) {
      const int64_t v = tile_sum[b];
      tile_sum[b] = run;
      run += v;
    }
    out[n] = int32_t(run);
    if (total_dev) *total_dev = run;
    if (overflow_dev && run > int64_t(0x7fffffff)) *overflow_dev = 1;
  }
}

__global__ void __launch_bounds__(1024) scan_tile_kernel(const int32_t* __restrict__ in, int32_t* __restrict__ out, int64_t n,
                                                         const int64_t* __restrict__ tile_base) {
  __shared__ int64_t warp_tot[32];
  const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
  const int64_t i0 = int64_t(blockIdx.x) * 4096 + int64_t(t) * 4;
  int32_t v[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) v[k] = (i0 + k < n) ? in[i0 + k] : 0;
  const int64_t s = int64_t(v[0]) + v[1] + v[2] + v[3];
  int64_t incl = s;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int64_t u = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += u;
  }
  if (lane == 31) warp_tot[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    const int64_t w = warp_tot[lane];
    int64_t wi = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int64_t u = __shfl_up_sync(0xffffffffu, wi, o);
      if (lane >= o) wi += u;
    }
    warp_tot[lane] = wi - w;
  }
  __syncthreads();
  int64_t excl = tile_base[blockIdx.x] + warp_tot[wid] + (incl - s);
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    if (i0 + k < n) out[i0 + k] = int32_t(excl);
    excl += v[k];
  }
}

qhap_status exclusive_scan_i32(const int32_t* in, int32_t* out, int64_t n, int64_t* total_dev, int32_t* overflow_dev,
                               cudaStream_t stream, int64_t* scratch) {
  const int64_t n_tiles = ceil_div(n, 4096);
  if (scratch == nullptr || n_tiles < 8 || n_tiles > 4096) {
    scan_i32_kernel<<<1, 1024, 0, stream>>>(in, out, n, total_dev, overflow_dev);
    QHAP_LAUNCH_CHECK();
    return QHAP_OK;
  }
  scan_tile_sum_kernel<<<int(n_tiles), 1024, 0, stream>>>(in, n, scratch);
  QHAP_LAUNCH_CHECK();
  scan_tile_base_kernel<<<1, 32, 0, stream>>>(scratch, n_tiles, out, n, total_dev, overflow_dev);
  QHAP_LAUNCH_CHECK();
  scan_tile_kernel<<<int(n_tiles), 1024, 0, stream>>>(in, out, n, scratch);
  QHAP_LAUNCH_CHECK();
  return QHAP_OK;
}

}  // namespace qhap

extern "C" const char* qhap_last_error(void) { return qhap::g_err; }
extern "C" uint64_t qhap_launch_count(void) { return qhap::g_launches.load(std::memory_order_relaxed); }
extern "C" const char* qhap_version(void) { return "qhap-b200 0.2 sm_100a"; }
