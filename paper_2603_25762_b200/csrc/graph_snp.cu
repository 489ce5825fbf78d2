// (2) SNP-graph build.  PAPER.md:L287-L319 [Eq. 9-14], linkage depth L85, Pore-C scaling L350.
//   q = 1 - 10^(-Q/10) (9);  P_cis = qu qv + (1-qu)(1-qv) (11);  P_trans = qu(1-qv) + (1-qu)qv (12);
//   l = sgn(W_iu W_iv) log10(P_cis/P_trans) (13);  w_uv = - sum_i alpha_i l / (|S_i| - 1) (14).
// Canonical sum (R6): each term is computed in fp64 with individually rounded operations, scaled by 2^32,
// rounded to int64 (nearest even) and INTEGER-added, so any accumulation order gives the same bits.
//
// Row-gather design: the fragment matrix is compacted (missing entries dropped) and transposed (per-SNP lists of
// covering fragment entries).  One CTA owns SNP row u: for every covering fragment it walks the partners of u inside
// the linkage reach (both directions -- the relation |p - t| <= reach is symmetric), accumulates the int64 terms per
// partner v in a shared-memory hash table (atomicCAS on the key, 64-bit atomicAdd on the value), then bitonic-sorts the
// table by v and streams the row out.  Pass 1 only counts distinct partners; an exclusive scan gives row_ptr; pass 2
// fills.  No global sort, no global atomics on weights, HBM traffic ~ the compulsory input + output.
#include <math.h>

#include <vector>

#include "kernels.cuh"

namespace qhap {

namespace {

constexpr int32_t kEmpty = 0x7fffffff;

struct Compact {
  int32_t* k;        // [n_frag+1] non-missing count per fragment -> exclusive scan (cptr)
  int32_t* csnp;     // [cnnz] SNP index
  uint8_t* cm;       // [cnnz] 1 if allele == h1[snp] (M = +1) else 0 (M = -1)
  uint8_t* cq;       // [cnnz] Phred clamped to [1, 93]
  int32_t* cfrag;    // [cnnz] owning fragment
  int32_t* colptr;   // [n_snp+1] coverage per SNP -> exclusive scan
  int32_t* cursor;   // [n_snp] fill cursors
  int32_t* csc;      // [cnnz] compact entry indices grouped by SNP
  uint8_t* cls;      // [n_snp] size class of the row
  int32_t* flags;    // [0] cnnz overflow, [1] nnz overflow, [2] a row is too large, [3] hash table overflow
  int64_t* total;    // [2] cnnz, nnz
  double* table;     // [94*94] log10(P_cis / P_trans)
};

__global__ void __launch_bounds__(256) count_nonmissing_kernel(int32_t n_frag, const int64_t* __restrict__ frag_ptr,
                                                               const uint8_t* __restrict__ allele, int32_t* __restrict__ k) {
  const int32_t i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (i >= n_frag) return;
  const int lane = threadIdx.x & 31;
  int cnt = 0;
  for (int64_t e = frag_ptr[i] + lane; e < frag_ptr[i + 1]; e += 32) cnt += (allele[e] <= 1);
  cnt = warp_sum(cnt);
  if (lane == 0) k[i] = cnt;
}

__global__ void __launch_bounds__(256) compact_kernel(int32_t n_frag, const int64_t* __restrict__ frag_ptr,
                                                      const int32_t* __restrict__ snp_idx, const uint8_t* __restrict__ allele,
                                                      const uint8_t* __restrict__ qual, const uint8_t* __restrict__ h1,
                                                      Compact c) {
  const int32_t i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (i >= n_frag) return;
  const int lane = threadIdx.x & 31;
  int32_t pos = c.k[i];   // cptr after the scan
  for (int64_t base = frag_ptr[i]; base < frag_ptr[i + 1]; base += 32) {
    const int64_t e = base + lane;
    const bool ok = e < frag_ptr[i + 1] && allele[e] <= 1;
    const uint32_t mask = __ballot_sync(0xffffffffu, ok);
    if (ok) {
      const int32_t p = pos + __popc(mask & ((1u << lane) - 1u));
      const int32_t u = snp_idx[e];
      c.csnp[p] = u;
      c.cm[p] = (allele[e] == (h1 ? h1[u] : uint8_t(0))) ? 1 : 0;                 // Eq. 1
      c.cq[p] = uint8_t(min(93, max(1, int(qual[e]))));                             // R5
      c.cfrag[p] = i;
      atomicAdd(&c.colptr[u], 1);
    }
    pos += __popc(mask);
  }
}

__global__ void __launch_bounds__(256) csc_fill_kernel(int32_t cnnz, Compact c) {
  const int32_t p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= cnnz) return;
  const int32_t u = c.csnp[p];
  c.csc[c.colptr[u] + atomicAdd(&c.cursor[u], 1)] = p;
}

struct Reach {
  int32_t base, p, k, tlo, thi;
  double alpha_i;
};

__device__ __forceinline__ Reach reach_of(const Compact& c, const uint8_t* __restrict__ frag_flags, int32_t tenths,
                                          double alpha, int32_t ce) {
  Reach r;
  const int32_t i = c.cfrag[ce];
  r.base = c.k[i];
  r.k = c.k[i + 1] - r.base;
  r.p = ce - r.base;
  const bool porec = frag_flags && (frag_flags[i] & 1);
  const int32_t reach = porec ? (r.k - 1) : int32_t((int64_t(tenths) * (r.k - 1)) / 10);   // floor, L85; R8
  r.alpha_i = porec ? alpha : 1.0;                                                          // L350
  r.tlo = max(0, r.p - reach);
  r.thi = min(r.k - 1, r.p + reach);
  return r;
}

// Size class of each row from cheap bounds: distinct partners <= min(#contributions, index window).
__global__ void __launch_bounds__(256) classify_kernel(int32_t n_snp, const uint8_t* __restrict__ frag_flags, int32_t tenths,
                                                       double alpha, Compact c) {
  const int32_t u = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (u >= n_snp) return;
  const int lane = threadIdx.x & 31;
  int64_t contrib = 0;
  int32_t vmin = kEmpty, vmax = -1;
  for (int32_t s = c.colptr[u] + lane; s < c.colptr[u + 1]; s += 32) {
    const Reach r = reach_of(c, frag_flags, tenths, alpha, c.csc[s]);
    if (r.k < 2 || r.thi <= r.tlo) continue;
    contrib += r.thi - r.tlo;
    vmin = min(vmin, c.csnp[r.base + r.tlo]);
    vmax = max(vmax, c.csnp[r.base + r.thi]);
  }
  contrib = warp_sum(contrib);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    vmin = min(vmin, __shfl_xor_sync(0xffffffffu, vmin, o));
    vmax = max(vmax, __shfl_xor_sync(0xffffffffu, vmax, o));
  }
  if (lane == 0) {
    int64_t bound = contrib == 0 ? 0 : min(contrib, int64_t(vmax) - vmin);
    uint8_t cl = bound == 0 ? 0 : bound <= 85 ? 1 : bound <= 680 ? 2 : bound <= 5400 ? 3 : 4;
    c.cls[u] = cl;
    if (cl == 4) c.flags[2] = 1;
  }
}

template <int TS>
__device__ __forceinline__ void bitonic_sort(int32_t* keys, unsigned long long* vals) {
  for (int size = 2; size <= TS; size <<= 1)
    for (int stride = size >> 1; stride > 0; stride >>= 1) {
      __syncthreads();
      for (int t = threadIdx.x; t < TS / 2; t += blockDim.x) {
        const int lo = 2 * t - (t & (stride - 1));
        const int hi = lo + stride;
        const bool up = (lo & size) == 0;
        const int32_t a = keys[lo], b = keys[hi];
        if ((a > b) == up) {
          keys[lo] = b; keys[hi] = a;
          const unsigned long long va = vals[lo]; vals[lo] = vals[hi]; vals[hi] = va;
        }
      }
    }
  __syncthreads();
}

template <int TS, int THREADS, bool FILL>
__global__ void __launch_bounds__(THREADS) snp_rows_kernel(int32_t n_snp, int cls, const uint8_t* __restrict__ frag_flags,
                                                           int32_t tenths, double alpha, Compact c,
                                                           int32_t* __restrict__ row_ptr, int32_t* __restrict__ col,
                                                           int64_t* __restrict__ w_fx, float* __restrict__ w) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  unsigned long long* vals = reinterpret_cast<unsigned long long*>(smem_raw);
  int32_t* keys = reinterpret_cast<int32_t*>(smem_raw + size_t(TS) * 8);
  __shared__ int32_t n_keys;
  const int32_t u = blockIdx.x;
  if (c.cls[u] != cls) return;
  for (int t = threadIdx.x; t < TS; t += THREADS) { keys[t] = kEmpty; vals[t] = 0ull; }
  if (threadIdx.x == 0) n_keys = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  constexpr int NW = THREADS / 32;
  for (int32_t s = c.colptr[u] + warp; s < c.colptr[u + 1]; s += NW) {
    const int32_t ce = c.csc[s];
    const Reach r = reach_of(c, frag_flags, tenths, alpha, ce);
    if (r.k < 2) continue;
    const int mu = c.cm[ce], qu = c.cq[ce];
    const double km1 = double(r.k - 1);
    for (int32_t t = r.tlo + lane; t <= r.thi; t += 32) {
      if (t == r.p) continue;
      const int32_t ce2 = r.base + t;
      const int32_t v = c.csnp[ce2];
      if (FILL) {
        const int mv = c.cm[ce2], qv = c.cq[ce2];
        const double sg = (mu == mv) ? 1.0 : -1.0;                                         // sgn(W_iu W_iv), Eq. 13
        const double T = (u < v) ? c.table[qu * 94 + qv] : c.table[qv * 94 + qu];          // lower SNP index first
        const double t1 = __dmul_rn(__dmul_rn(r.alpha_i, sg), T);
        const double term = __ddiv_rn(-t1, km1);                                           // Eq. 14
        const long long fx = __double2ll_rn(__dmul_rn(term, 4294967296.0));                // R6
        uint32_t h = (uint32_t(v) * 2654435761u) & (TS - 1);
        for (int probe = 0; probe < TS; ++probe) {
          const int32_t prev = atomicCAS(&keys[h], kEmpty, v);
          if (prev == kEmpty || prev == v) { atomicAdd(&vals[h], (unsigned long long)fx); break; }
          h = (h + 1) & (TS - 1);
          if (probe == TS - 1) c.flags[3] = 1;
        }
      } else {
        uint32_t h = (uint32_t(v) * 2654435761u) & (TS - 1);
        for (int probe = 0; probe < TS; ++probe) {
          const int32_t prev = atomicCAS(&keys[h], kEmpty, v);
          if (prev == kEmpty) { atomicAdd(&n_keys, 1); break; }
          if (prev == v) break;
          h = (h + 1) & (TS - 1);
          if (probe == TS - 1) c.flags[3] = 1;
        }
      }
    }
  }
  __syncthreads();
  if (!FILL) {
    if (threadIdx.x == 0) row_ptr[u] = n_keys;
    return;
  }
  bitonic_sort<TS>(keys, vals);
  const int32_t base = row_ptr[u], cnt = row_ptr[u + 1] - base;
  for (int t = threadIdx.x; t < cnt; t += THREADS) {
    const long long s = (long long)vals[t];
    col[base + t] = keys[t];
    w_fx[base + t] = s;
    w[base + t] = float(double(s) * (1.0 / 4294967296.0));
  }
}

// ------------------------------------------------------------------------------------------ block split
__global__ void __launch_bounds__(256) split_kernel(bool fill, int32_t n_out, int32_t nb, const int64_t* __restrict__ win,
                                                    const int32_t* __restrict__ off, const int32_t* __restrict__ row_ptr,
                                                    const int32_t* __restrict__ col, const int64_t* __restrict__ w_fx,
                                                    const float* __restrict__ w, int32_t* __restrict__ out_row_ptr,
                                                    int32_t* __restrict__ out_col, int64_t* __restrict__ out_w_fx,
                                                    float* __restrict__ out_w) {
  const int32_t ro = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (ro >= n_out) return;
  const int lane = threadIdx.x & 31;
  int lo = 0, hi = nb;
  while (hi - lo > 1) { int mid = (lo + hi) >> 1; if (off[mid] <= ro) lo = mid; else hi = mid; }
  const int b = lo;
  const int64_t ws = win[2 * b], we = win[2 * b + 1];
  const int64_t g = ws + (ro - off[b]);
  int32_t pos = fill ? out_row_ptr[ro] : 0;
  for (int32_t base = row_ptr[g]; base < row_ptr[g + 1]; base += 32) {
    const int32_t e = base + lane;
    int32_t cv = -1;
    if (e < row_ptr[g + 1]) cv = col[e];
    const bool ok = cv >= ws && cv < we;
    const uint32_t mask = __ballot_sync(0xffffffffu, ok);
    if (fill && ok) {
      const int32_t p = pos + __popc(mask & ((1u << lane) - 1u));
      out_col[p] = int32_t(off[b] + (cv - ws));
      if (out_w_fx) out_w_fx[p] = w_fx[e];
      if (out_w) out_w[p] = w[e];
    }
    pos += __popc(mask);
  }
  if (!fill && lane == 0) out_row_ptr[ro] = pos;
}

void host_llr_table(double* T) {
  // Eq. 9, 11, 12 with the C library; entries with Q = 0 are never indexed (qualities are clamped to [1, 93]).
  for (int qu = 0; qu < 94; ++qu)
    for (int qv = 0; qv < 94; ++qv) {
      const double a = 1.0 - pow(10.0, -double(qu) / 10.0);
      const double b = 1.0 - pow(10.0, -double(qv) / 10.0);
      const double pc = a * b + (1.0 - a) * (1.0 - b);
      const double pt = a * (1.0 - b) + (1.0 - a) * b;
      T[qu * 94 + qv] = (qu == 0 || qv == 0) ? 0.0 : log10(pc / pt);
    }
}

template <bool FILL>
qhap_status launch_rows(int32_t n_snp, const uint8_t* flags, int32_t tenths, double alpha, const Compact& c, int32_t* row_ptr,
                        int32_t* col, int64_t* w_fx, float* w, cudaStream_t stream) {
  QHAP_CUDA_TRY(cudaFuncSetAttribute(snp_rows_kernel<8192, 512, FILL>, cudaFuncAttributeMaxDynamicSharedMemorySize, 8192 * 12));   // per device
  snp_rows_kernel<128, 64, FILL><<<n_snp, 64, 128 * 12, stream>>>(n_snp, 1, flags, tenths, alpha, c, row_ptr, col, w_fx, w);
  QHAP_LAUNCH_CHECK();
  snp_rows_kernel<1024, 256, FILL><<<n_snp, 256, 1024 * 12, stream>>>(n_snp, 2, flags, tenths, alpha, c, row_ptr, col, w_fx, w);
  QHAP_LAUNCH_CHECK();
  snp_rows_kernel<8192, 512, FILL><<<n_snp, 512, 8192 * 12, stream>>>(n_snp, 3, flags, tenths, alpha, c, row_ptr, col, w_fx, w);
  QHAP_LAUNCH_CHECK();
  return QHAP_OK;
}

}  // namespace
}  // namespace qhap

using namespace qhap;

extern "C" qhap_status qhap_build_snp_graph(const qhap_frags* fr, int32_t linkage_tenths, double alpha,
                                            const double* llr_table, qhap_csr* out, void* workspace, size_t* ws_bytes,
                                            void* stream_v) {
  QHAP_REQUIRE(fr && out, "frags and out must not be NULL");
  QHAP_REQUIRE(fr->n_frag >= 0 && fr->n_snp >= 0, "negative sizes");
  QHAP_REQUIRE(linkage_tenths >= 1 && linkage_tenths <= 10, "linkage_tenths must be 1..10");
  const int32_t nf = fr->n_frag, ns = fr->n_snp;
  const int64_t fnnz = fr->nnz;
  QHAP_REQUIRE(fnnz >= 0 && fnnz < (int64_t(1) << 31), "fragment matrix must have < 2^31 entries");
  Workspace ws(workspace);
  Compact c;
  c.k = ws.take<int32_t>(size_t(nf) + 1);
  c.csnp = ws.take<int32_t>(size_t(fnnz));
  c.cm = ws.take<uint8_t>(size_t(fnnz));
  c.cq = ws.take<uint8_t>(size_t(fnnz));
  c.cfrag = ws.take<int32_t>(size_t(fnnz));
  c.colptr = ws.take<int32_t>(size_t(ns) + 1);
  c.cursor = ws.take<int32_t>(size_t(ns));
  c.csc = ws.take<int32_t>(size_t(fnnz));
  c.cls = ws.take<uint8_t>(size_t(ns));
  c.flags = ws.take<int32_t>(4);
  c.total = ws.take<int64_t>(2);
  c.table = ws.take<double>(94 * 94);
  int64_t* scan_scratch = ws.take<int64_t>(size_t(std::max(nf, ns)) / 4096 + 2);
  qhap_status st;
  if (workspace_protocol(ws, workspace, ws_bytes, &st)) return st;
  QHAP_TRY(require_device());
  QHAP_REQUIRE(out->row_ptr, "out->row_ptr must point to n_snp+1 ints");
  QHAP_REQUIRE(nf == 0 || (fr->frag_ptr && fr->snp_idx && fr->allele && fr->qual), "frag_ptr, snp_idx, allele and qual must not be NULL");
  cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
  const int64_t capacity = out->col ? out->nnz : 0;
  out->n = ns;

  std::vector<double> T(94 * 94);
  if (llr_table) std::copy(llr_table, llr_table + 94 * 94, T.begin());
  else host_llr_table(T.data());
  QHAP_CUDA_TRY(cudaMemcpyAsync(c.table, T.data(), sizeof(double) * 94 * 94, cudaMemcpyHostToDevice, stream));
  QHAP_CUDA_TRY(cudaMemsetAsync(c.flags, 0, 4 * sizeof(int32_t), stream));
  QHAP_CUDA_TRY(cudaMemsetAsync(c.colptr, 0, sizeof(int32_t) * (size_t(ns) + 1), stream));
  QHAP_CUDA_TRY(cudaMemsetAsync(c.cursor, 0, sizeof(int32_t) * size_t(ns), stream));
  QHAP_CUDA_TRY(cudaMemsetAsync(c.cls, 0, size_t(ns), stream));
  if (nf > 0) {
    count_nonmissing_kernel<<<int(ceil_div(int64_t(nf) * 32, 256)), 256, 0, stream>>>(nf, fr->frag_ptr, fr->allele, c.k);
    QHAP_LAUNCH_CHECK();
  }
  QHAP_TRY(exclusive_scan_i32(c.k, c.k, nf, c.total, c.flags, stream, scan_scratch));
  if (nf > 0) {
    compact_kernel<<<int(ceil_div(int64_t(nf) * 32, 256)), 256, 0, stream>>>(nf, fr->frag_ptr, fr->snp_idx, fr->allele, fr->qual,
                                                                         fr->h1, c);
    QHAP_LAUNCH_CHECK();
  }
  QHAP_TRY(exclusive_scan_i32(c.colptr, c.colptr, ns, nullptr, nullptr, stream, scan_scratch));
  int64_t cnnz = 0;
  QHAP_CUDA_TRY(cudaMemcpyAsync(&cnnz, c.total, sizeof(int64_t), cudaMemcpyDeviceToHost, stream));
  QHAP_CUDA_TRY(cudaStreamSynchronize(stream));
  if (cnnz > 0) {
    csc_fill_kernel<<<int(ceil_div(cnnz, 256)), 256, 0, stream>>>(int32_t(cnnz), c);
    QHAP_LAUNCH_CHECK();
  }
  if (ns > 0) {
    classify_kernel<<<int(ceil_div(int64_t(ns) * 32, 256)), 256, 0, stream>>>(ns, fr->frag_flags, linkage_tenths, alpha, c);
    QHAP_LAUNCH_CHECK();
    QHAP_CUDA_TRY(cudaMemsetAsync(out->row_ptr, 0, sizeof(int32_t) * (size_t(ns) + 1), stream));
    QHAP_TRY(launch_rows<false>(ns, fr->frag_flags, linkage_tenths, alpha, c, out->row_ptr, nullptr, nullptr, nullptr, stream));
  }
  QHAP_TRY(exclusive_scan_i32(out->row_ptr, out->row_ptr, ns, c.total + 1, c.flags + 1, stream, scan_scratch));
  int64_t total = 0;
  int32_t flags[4] = {0, 0, 0, 0};
  QHAP_CUDA_TRY(cudaMemcpyAsync(&total, c.total + 1, sizeof(total), cudaMemcpyDeviceToHost, stream));
  QHAP_CUDA_TRY(cudaMemcpyAsync(flags, c.flags, sizeof(flags), cudaMemcpyDeviceToHost, stream));
  QHAP_CUDA_TRY(cudaStreamSynchronize(stream));
  if (flags[1]) { set_error("SNP graph has >= 2^31 directed entries"); return QHAP_ERR_RANGE; }
  if (flags[2] || flags[3]) { set_error("a SNP has more than 5400 candidate partners (unsupported row size)"); return QHAP_ERR_RANGE; }
  out->nnz = total;
  if (out->col == nullptr) return QHAP_OK;
  if (capacity < total) { set_error("edge capacity too small: %lld < %lld", (long long)capacity, (long long)total); return QHAP_ERR_WORKSPACE; }
  QHAP_REQUIRE(out->w_fx && out->w, "out->w_fx and out->w must not be NULL when out->col is given");
  if (ns > 0) QHAP_TRY(launch_rows<true>(ns, fr->frag_flags, linkage_tenths, alpha, c, out->row_ptr, out->col, out->w_fx, out->w, stream));
  return QHAP_OK;
}

extern "C" qhap_status qhap_block_split(const qhap_csr* graph, int32_t n_blocks, const int64_t* win, qhap_csr* out,
                                        void* workspace, size_t* ws_bytes, void* stream_v) {
  QHAP_REQUIRE(graph && out && n_blocks >= 1 && win, "graph, out, win must not be NULL");
  std::vector<int32_t> off(size_t(n_blocks) + 1, 0);
  for (int b = 0; b < n_blocks; ++b) {
    QHAP_REQUIRE(win[2 * b] >= 0 && win[2 * b] <= win[2 * b + 1] && win[2 * b + 1] <= graph->n, "window outside [0, n]");
    const int64_t o = int64_t(off[b]) + (win[2 * b + 1] - win[2 * b]);
    QHAP_REQUIRE(o < (int64_t(1) << 31), "too many rows");
    off[b + 1] = int32_t(o);
  }
  const int32_t n_out = off[n_blocks];
  Workspace ws(workspace);
  int64_t* win_d = ws.take<int64_t>(2 * size_t(n_blocks));
  int32_t* off_d = ws.take<int32_t>(size_t(n_blocks) + 1);
  int64_t* total_d = ws.take<int64_t>(1);
  int32_t* flags_d = ws.take<int32_t>(1);
  qhap_status st;
  if (workspace_protocol(ws, workspace, ws_bytes, &st)) return st;
  QHAP_TRY(require_device());
  QHAP_REQUIRE(out->row_ptr && graph->row_ptr, "row_ptr arrays must not be NULL");
  cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
  const int64_t capacity = out->col ? out->nnz : 0;
  out->n = n_out;
  QHAP_CUDA_TRY(cudaMemcpyAsync(win_d, win, sizeof(int64_t) * 2 * size_t(n_blocks), cudaMemcpyHostToDevice, stream));
  QHAP_CUDA_TRY(cudaMemcpyAsync(off_d, off.data(), sizeof(int32_t) * (size_t(n_blocks) + 1), cudaMemcpyHostToDevice, stream));
  QHAP_CUDA_TRY(cudaMemsetAsync(flags_d, 0, sizeof(int32_t), stream));
  const int blocks = int(ceil_div(int64_t(n_out) * 32, 256));
  if (n_out > 0) {
    split_kernel<<<blocks, 256, 0, stream>>>(false, n_out, n_blocks, win_d, off_d, graph->row_ptr, graph->col, graph->w_fx,
                                             graph->w, out->row_ptr, nullptr, nullptr, nullptr);
    QHAP_LAUNCH_CHECK();
  }
  QHAP_TRY(exclusive_scan_i32(out->row_ptr, out->row_ptr, n_out, total_d, flags_d, stream));
  int64_t total = 0;
  QHAP_CUDA_TRY(cudaMemcpyAsync(&total, total_d, sizeof(total), cudaMemcpyDeviceToHost, stream));
  QHAP_CUDA_TRY(cudaStreamSynchronize(stream));   // also keeps `off` alive until the copies above are done
  out->nnz = total;
  if (out->col == nullptr) return QHAP_OK;
  if (capacity < total) { set_error("edge capacity too small: %lld < %lld", (long long)capacity, (long long)total); return QHAP_ERR_WORKSPACE; }
  if (n_out > 0) {
    split_kernel<<<blocks, 256, 0, stream>>>(true, n_out, n_blocks, win_d, off_d, graph->row_ptr, graph->col, graph->w_fx,
                                             graph->w, out->row_ptr, out->col, out->w_fx, out->w);
    QHAP_LAUNCH_CHECK();
  }
  return QHAP_OK;
}
