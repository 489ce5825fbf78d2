// Shared host/device helpers of libqhap (CUDA path only; nothing here is used by oracle/).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include <string>

#include "qhap.h"

namespace qhap {

// ---------------------------------------------------------------------------------------------- errors
void set_error(const char* fmt, ...);

#define QHAP_CUDA_TRY(expr)                                                                    \
  do {                                                                                         \
    cudaError_t e__ = (expr);                                                                  \
    if (e__ != cudaSuccess) {                                                                  \
      ::qhap::set_error("%s:%d: %s -> %s", __FILE__, __LINE__, #expr, cudaGetErrorString(e__)); \
      return QHAP_ERR_CUDA;                                                                    \
    }                                                                                          \
  } while (0)

#define QHAP_TRY(expr)                 \
  do {                                 \
    qhap_status s__ = (expr);          \
    if (s__ != QHAP_OK) return s__;    \
  } while (0)

#define QHAP_REQUIRE(cond, ...)        \
  do {                                 \
    if (!(cond)) {                     \
      ::qhap::set_error(__VA_ARGS__);  \
      return QHAP_ERR_INVALID_ARG;     \
    }                                  \
  } while (0)

// Every kernel launch of the library is followed by QHAP_LAUNCH_CHECK(): it counts the launch (qhap_launch_count) and
// turns a launch error into QHAP_ERR_CUDA.
void count_launches(uint64_t n);
#define QHAP_LAUNCH_CHECK()                 \
  do {                                      \
    ::qhap::count_launches(1);              \
    QHAP_CUDA_TRY(cudaGetLastError());      \
  } while (0)

// sm_100 present on the CURRENT device?  (cached per device ordinal)
qhap_status require_device();
// SM count of the current device (queried once per device; 148 on B200)
int sm_count();

// ------------------------------------------------------------------------------------------- workspace
// Bump allocator over the caller's workspace.  In "measure" mode (base == nullptr) it only adds sizes up.  Every layout
// is written ONCE, as a function that walks a Workspace: the size query runs it in measure mode, the call runs the same
// function on the real pointer, so the two cannot disagree.  `cap` bounds a real carve: a take() that would pass it sets
// `overflow` (checked by the caller -> QHAP_ERR_WORKSPACE) and returns nullptr instead of a pointer past the end.
struct Workspace {
  char* base;
  size_t cap;
  size_t off = 0;
  bool overflow = false;
  explicit Workspace(void* p, size_t cap_bytes = ~size_t(0)) : base(static_cast<char*>(p)), cap(cap_bytes) {}
  template <class T>
  T* take(size_t count) {
    size_t bytes = (count * sizeof(T) + 255) & ~size_t(255);
    T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
    if (base && (bytes > cap || off > cap - bytes)) { overflow = true; p = nullptr; }
    off += bytes;
    return p;
  }
  size_t used() const { return off; }
};

// Standard epilogue of the workspace protocol (see qhap.h).  Returns true if the caller must return `*st` now.
inline bool workspace_protocol(const Workspace& need, void* workspace, size_t* ws_bytes, qhap_status* st) {
  if (ws_bytes == nullptr) {
    set_error("ws_bytes must not be NULL");
    *st = QHAP_ERR_INVALID_ARG;
    return true;
  }
  if (workspace == nullptr) {
    *ws_bytes = need.used();
    *st = QHAP_OK;
    return true;
  }
  if (*ws_bytes < need.used()) {
    set_error("workspace too small: %zu < %zu", *ws_bytes, need.used());
    *ws_bytes = need.used();
    *st = QHAP_ERR_WORKSPACE;
    return true;
  }
  if ((reinterpret_cast<uintptr_t>(workspace) & 255) != 0) {
    set_error("workspace must be 256-byte aligned");
    *st = QHAP_ERR_INVALID_ARG;
    return true;
  }
  return false;
}

// ------------------------------------------------------------------------------------------ primitives
// Exclusive scan of `n` int32 counts into out[0..n] (out[n] = total), in place allowed (out == in is fine when
// in has n+1 slots).  Single launch; total returned through *total_dev (int64, device) when not NULL.
// Sets *overflow_dev (int32, device) to 1 if the total does not fit int32.
// `scratch` (optional, device, ceil(n / 4096) + 1 int64): enables the multi-CTA scan for long arrays.
qhap_status exclusive_scan_i32(const int32_t* in, int32_t* out, int64_t n, int64_t* total_dev, int32_t* overflow_dev,
                               cudaStream_t stream, int64_t* scratch = nullptr);

static inline int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }

// ---------------------------------------------------------------------------------------- device helpers
#ifdef __CUDACC__
__device__ __forceinline__ int lane_id() { return threadIdx.x & 31; }

template <class T>
__device__ __forceinline__ T warp_sum(T v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Canonical edge weight of entry e in the graph's integer units (qhap.h QHAP_WEIGHT_*).
__device__ __forceinline__ int64_t edge_weight(int mode, const int32_t* __restrict__ d, const int32_t* __restrict__ c,
                                               const int64_t* __restrict__ w_fx, int64_t e) {
  if (mode == QHAP_WEIGHT_D) return int64_t(d[e]);
  if (mode == QHAP_WEIGHT_D_MINUS_C) return int64_t(d[e]) - int64_t(c[e]);
  return w_fx[e];
}
#endif

}  // namespace qhap
