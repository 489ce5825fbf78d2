// (1) Read-graph build.  PAPER.md:L235-L246 [Eq. 2-3]: vertices = fragments, w_ab = # shared SNPs with opposing
// alleles; we also count the concordant shared SNPs C_ab (BASELINE.json config 0 weight = D - C; R1).
// Edge set = pairs sharing >= 1 covered (non-missing) SNP.  Integer work only -> bit-exact.
//
// With fragments sorted by their first SNP index, the partners of fragment a lie in an index window:
//   b <= hi_a = last b with first_b <= last_a,   b >= lo_a = first b with max(last_0..last_b) >= first_a.
// One warp owns fragment a; its lanes take 32 candidates b at a time and count D, C over the shared SNPs (direct
// offset walk when both fragments are contiguous index ranges, sorted two-pointer merge otherwise, e.g. Pore-C
// fragments).  M_aj M_bj = -1 <=> the two alleles differ, so the gauge h1 drops out (R2).
// Two passes (count -> scan -> fill) give an exact-size symmetric CSR with ascending columns and no atomics.
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "kernels.cuh"

namespace qhap {

namespace {

struct FragMeta {
  int32_t* first;   // [n] first SNP index
  int32_t* last;    // [n] last SNP index
  int32_t* pmax;    // [n] prefix maximum of last
  int32_t* flags;   // [0] unsorted / empty fragment seen, [1] nnz overflow, [2] dense range error
  int64_t* total;   // directed nnz
};

__global__ void __launch_bounds__(256) frag_meta_kernel(int32_t n, const int64_t* __restrict__ frag_ptr,
                                                        const int32_t* __restrict__ snp_idx, FragMeta m) {
  const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int64_t p0 = frag_ptr[i], p1 = frag_ptr[i + 1];
  if (p1 <= p0) { m.flags[0] = 1; m.first[i] = 0; m.last[i] = -1; return; }
  const int32_t f = snp_idx[p0], l = snp_idx[p1 - 1];
  m.first[i] = f;
  // bit 31 of `last` is free (indices are < 2^31): keep the plain value, contiguity is recomputed where needed
  m.last[i] = l;
  if (i > 0) {
    const int64_t q0 = frag_ptr[i - 1];
    if (frag_ptr[i] > q0 && snp_idx[q0] > f) m.flags[0] = 1;   // not sorted by first SNP index
  }
}

// Single CTA prefix maximum (n is the number of fragments: small).
__global__ void __launch_bounds__(1024) prefix_max_kernel(int32_t n, const int32_t* __restrict__ in, int32_t* __restrict__ out) {
  __shared__ int32_t wmax[32];
  __shared__ int32_t carry_s;
  const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
  if (t == 0) carry_s = INT32_MIN;
  __syncthreads();
  for (int32_t base = 0; base < n; base += 1024) {
    const int32_t i = base + t;
    int32_t v = (i < n) ? in[i] : INT32_MIN;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int32_t u = __shfl_up_sync(0xffffffffu, v, o);
      if (lane >= o) v = max(v, u);
    }
    if (lane == 31) wmax[wid] = v;
    __syncthreads();
    if (wid == 0) {
      int32_t w = wmax[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        int32_t u = __shfl_up_sync(0xffffffffu, w, o);
        if (lane >= o) w = max(w, u);
      }
      wmax[lane] = w;   // inclusive maximum over warps 0..lane
    }
    __syncthreads();
    int32_t r = max(carry_s, v);
    if (wid > 0) r = max(r, wmax[wid - 1]);
    if (i < n) out[i] = r;
    __syncthreads();
    if (t == 1023) carry_s = r;
    __syncthreads();
  }
}

// D and C of the pair (a, b).  Returns D in .x, C in .y.
__device__ __forceinline__ int2 pair_counts(const int64_t* __restrict__ frag_ptr, const int32_t* __restrict__ snp_idx,
                                            const uint8_t* __restrict__ allele, int32_t a, int32_t fa, int32_t la,
                                            int32_t b, int32_t fb, int32_t lb) {
  int D = 0, C = 0;
  const int32_t s = max(fa, fb), t = min(la, lb);
  if (s > t) return make_int2(0, 0);
  const int64_t a0 = frag_ptr[a], a1 = frag_ptr[a + 1], b0 = frag_ptr[b], b1 = frag_ptr[b + 1];
  const bool contig = (int64_t(la) - fa + 1 == a1 - a0) && (int64_t(lb) - fb + 1 == b1 - b0);
  if (contig) {
    const uint8_t* pa = allele + a0 + (s - fa);
    const uint8_t* pb = allele + b0 + (s - fb);
    const int len = t - s + 1;
    for (int k = 0; k < len; ++k) {
      const uint8_t x = pa[k], y = pb[k];
      if (x <= 1 && y <= 1) { D += (x != y); C += (x == y); }
    }
  } else {
    int64_t ia = a0, ib = b0;
    while (ia < a1 && ib < b1) {
      const int32_t ja = snp_idx[ia], jb = snp_idx[ib];
      if (ja < jb) ++ia;
      else if (jb < ja) ++ib;
      else {
        const uint8_t x = allele[ia], y = allele[ib];
        if (x <= 1 && y <= 1) { D += (x != y); C += (x == y); }
        ++ia; ++ib;
      }
    }
  }
  return make_int2(D, C);
}

template <bool FILL>
__global__ void __launch_bounds__(256) read_pairs_kernel(int32_t n, const int64_t* __restrict__ frag_ptr,
                                                         const int32_t* __restrict__ snp_idx,
                                                         const uint8_t* __restrict__ allele, FragMeta m,
                                                         int32_t* __restrict__ row_ptr /*COUNT: counts out; FILL: offsets in*/,
                                                         int32_t* __restrict__ col, int32_t* __restrict__ dd,
                                                         int32_t* __restrict__ cc, int64_t capacity) {
  const int32_t a = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (a >= n) return;
  // FILL runs right behind the count and the scan, without a host round trip in between: it looks at their verdict itself
  // (bad input, 2^31 entries, more entries than the caller's arrays hold) and leaves the arrays alone if there is one
  if (FILL && (m.flags[0] != 0 || m.flags[1] != 0 || *m.total > capacity)) return;
  const int lane = threadIdx.x & 31;
  const int32_t fa = m.first[a], la = m.last[a];
  // lo = first b with pmax[b] >= fa; hi = last b with first[b] <= la  (both arrays are non-decreasing)
  int32_t lo, hi;
  {
    int32_t l = 0, h = a;                    // pmax[a] >= la >= fa, so the answer is <= a
    while (l < h) { int32_t mid = (l + h) >> 1; if (m.pmax[mid] >= fa) h = mid; else l = mid + 1; }
    lo = l;
    l = a; h = n - 1;                        // first[a] <= la
    while (l < h) { int32_t mid = (l + h + 1) >> 1; if (m.first[mid] <= la) l = mid; else h = mid - 1; }
    hi = l;
  }
  int32_t out_pos = FILL ? row_ptr[a] : 0;
  for (int32_t base = lo; base <= hi; base += 32) {
    const int32_t b = base + lane;
    int2 dc = make_int2(0, 0);
    if (b <= hi && b != a) dc = pair_counts(frag_ptr, snp_idx, allele, a, fa, la, b, m.first[b], m.last[b]);
    const bool edge = (dc.x + dc.y) > 0;
    const uint32_t mask = __ballot_sync(0xffffffffu, edge);
    if (FILL && edge) {
      const int32_t p = out_pos + __popc(mask & ((1u << lane) - 1u));
      col[p] = b; dd[p] = dc.x; cc[p] = dc.y;
    }
    out_pos += __popc(mask);
  }
  if (!FILL && lane == 0) row_ptr[a] = out_pos;
}

// Dense J = -w: one CTA per row builds the row in shared memory in chunks and streams it out with 16-byte stores.
template <class HT>
__device__ __forceinline__ HT to_half_type(float v);
template <>
__device__ __forceinline__ __half to_half_type<__half>(float v) { return __float2half_rn(v); }
template <>
__device__ __forceinline__ __nv_bfloat16 to_half_type<__nv_bfloat16>(float v) { return __float2bfloat16_rn(v); }

constexpr int kDenseChunk = 8192;   // columns per shared-memory chunk (16 KB)

template <class HT>
__global__ void __launch_bounds__(256) dense_j_kernel(int32_t n, int32_t ld, const int32_t* __restrict__ row_ptr,
                                                      const int32_t* __restrict__ col, const int32_t* __restrict__ dd,
                                                      const int32_t* __restrict__ cc, int mode, int32_t limit,
                                                      HT* __restrict__ J, int32_t* __restrict__ flags,
                                                      const int64_t* __restrict__ total, int64_t capacity) {
  __shared__ __align__(16) HT row[kDenseChunk];
  if (flags[0] != 0 || flags[1] != 0 || *total > capacity) return;      // see read_pairs_kernel<true>
  const int32_t a = blockIdx.x;
  const int32_t e0 = a < n ? row_ptr[a] : 0, e1 = a < n ? row_ptr[a + 1] : 0;
  for (int32_t c0 = 0; c0 < ld; c0 += kDenseChunk) {
    const int32_t width = min(kDenseChunk, ld - c0);
    for (int i = threadIdx.x; i < kDenseChunk / 8; i += blockDim.x) reinterpret_cast<uint4*>(row)[i] = make_uint4(0, 0, 0, 0);
    __syncthreads();
    for (int32_t e = e0 + threadIdx.x; e < e1; e += blockDim.x) {
      const int32_t b = col[e];
      if (b >= c0 && b < c0 + width) {
        const int32_t w = (mode == QHAP_WEIGHT_D) ? dd[e] : dd[e] - cc[e];
        if (w > limit || w < -limit) flags[2] = 1;       // not exactly representable
        row[b - c0] = to_half_type<HT>(float(-w));      // Eq. 4: J = -A
      }
    }
    __syncthreads();
    uint4* dst = reinterpret_cast<uint4*>(J + size_t(a) * ld + c0);   // ld % 8 == 0 -> 16-byte aligned
    for (int i = threadIdx.x; i < width / 8; i += blockDim.x) dst[i] = reinterpret_cast<const uint4*>(row)[i];
    __syncthreads();
  }
}

}  // namespace
}  // namespace qhap

using namespace qhap;

extern "C" qhap_status qhap_build_read_graph(const qhap_frags* fr, int32_t weight_mode, qhap_csr* out, void* dense_J,
                                             int32_t dense_ld, int32_t dense_dtype, void* workspace, size_t* ws_bytes,
                                             void* stream_v) {
  QHAP_REQUIRE(fr && out, "frags and out must not be NULL");
  QHAP_REQUIRE(fr->n_frag >= 0 && fr->n_snp >= 0, "negative sizes");
  QHAP_REQUIRE(weight_mode == QHAP_WEIGHT_D || weight_mode == QHAP_WEIGHT_D_MINUS_C, "weight_mode must be 0 (D) or 1 (D-C)");
  const int32_t n = fr->n_frag;
  Workspace ws(workspace);
  FragMeta m;
  m.first = ws.take<int32_t>(n);
  m.last = ws.take<int32_t>(n);
  m.pmax = ws.take<int32_t>(n);
  m.flags = ws.take<int32_t>(4);
  m.total = ws.take<int64_t>(1);
  qhap_status st;
  if (workspace_protocol(ws, workspace, ws_bytes, &st)) return st;
  QHAP_TRY(require_device());
  QHAP_REQUIRE(out->row_ptr, "out->row_ptr must point to n_frag+1 ints");
  QHAP_REQUIRE(n == 0 || (fr->frag_ptr && fr->snp_idx && fr->allele), "fragment arrays must not be NULL");
  if (dense_J) {
    QHAP_REQUIRE(dense_dtype == QHAP_DENSE_FP16 || dense_dtype == QHAP_DENSE_BF16, "dense_dtype must be fp16 or bf16");
    QHAP_REQUIRE(dense_ld >= n && dense_ld % 8 == 0, "dense_ld must be >= n_frag and a multiple of 8");
  }
  cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
  const int64_t capacity = out->col ? out->nnz : 0;
  out->n = n;
  QHAP_CUDA_TRY(cudaMemsetAsync(m.flags, 0, 4 * sizeof(int32_t), stream));
  if (n > 0) {
    frag_meta_kernel<<<int(ceil_div(n, 256)), 256, 0, stream>>>(n, fr->frag_ptr, fr->snp_idx, m);
    QHAP_LAUNCH_CHECK();
    prefix_max_kernel<<<1, 1024, 0, stream>>>(n, m.last, m.pmax);
    QHAP_LAUNCH_CHECK();
    read_pairs_kernel<false><<<int(ceil_div(int64_t(n) * 32, 256)), 256, 0, stream>>>(n, fr->frag_ptr, fr->snp_idx, fr->allele,
                                                                                  m, out->row_ptr, nullptr, nullptr, nullptr, 0);
    QHAP_LAUNCH_CHECK();
  }
  QHAP_TRY(exclusive_scan_i32(out->row_ptr, out->row_ptr, n, m.total, m.flags + 1, stream));
  // Count-only call, or count + fill in ONE round trip: the fill kernels check the count's verdict on the device, the host
  // reads it once at the end.
  const bool fill = out->col != nullptr;
  if (fill) {
    QHAP_REQUIRE(out->d && out->c, "out->d and out->c must not be NULL when out->col is given");
    if (n > 0) {
      read_pairs_kernel<true><<<int(ceil_div(int64_t(n) * 32, 256)), 256, 0, stream>>>(n, fr->frag_ptr, fr->snp_idx, fr->allele, m,
                                                                                   out->row_ptr, out->col, out->d, out->c, capacity);
      QHAP_LAUNCH_CHECK();
    }
    if (dense_J && dense_ld > 0) {
      if (dense_dtype == QHAP_DENSE_FP16)
        dense_j_kernel<__half><<<dense_ld, 256, 0, stream>>>(n, dense_ld, out->row_ptr, out->col, out->d, out->c, weight_mode,
                                                            2048, static_cast<__half*>(dense_J), m.flags, m.total, capacity);
      else
        dense_j_kernel<__nv_bfloat16><<<dense_ld, 256, 0, stream>>>(n, dense_ld, out->row_ptr, out->col, out->d, out->c,
                                                                   weight_mode, 256, static_cast<__nv_bfloat16*>(dense_J), m.flags,
                                                                   m.total, capacity);
      QHAP_LAUNCH_CHECK();
    }
  }
  int64_t total = 0;
  int32_t flags[4] = {0, 0, 0, 0};
  QHAP_CUDA_TRY(cudaMemcpyAsync(&total, m.total, sizeof(total), cudaMemcpyDeviceToHost, stream));
  QHAP_CUDA_TRY(cudaMemcpyAsync(flags, m.flags, sizeof(flags), cudaMemcpyDeviceToHost, stream));
  QHAP_CUDA_TRY(cudaStreamSynchronize(stream));
  if (flags[0]) { set_error("fragments must be non-empty and sorted by their first SNP index"); return QHAP_ERR_INVALID_ARG; }
  if (flags[1]) { set_error("read graph has >= 2^31 directed entries"); return QHAP_ERR_RANGE; }
  out->nnz = total;
  if (!fill) return QHAP_OK;   // count-only call
  if (capacity < total) { set_error("edge capacity too small: %lld < %lld", (long long)capacity, (long long)total); return QHAP_ERR_WORKSPACE; }
  if (flags[2]) { set_error("a weight is not exactly representable in the dense dtype (|w| > %d)", dense_dtype == QHAP_DENSE_FP16 ? 2048 : 256); return QHAP_ERR_RANGE; }
  return QHAP_OK;
}
