// (2) SNP-graph build.  PAPER.md:L287-L319 [Eq. 9-14], linkage depth L85, Pore-C scaling L350.
//   q = 1 - 10^(-Q/10) (9);  P_cis = qu qv + (1-qu)(1-qv) (11);  P_trans = qu(1-qv) + (1-qu)qv (12);
//   l = sgn(W_iu W_iv) log10(P_cis/P_trans) (13);  w_uv = - sum_i alpha_i l / (|S_i| - 1) (14).
// Canonical sum (R6): each term is computed in fp64 with individually rounded operations, scaled by 2^32,
// rounded to int64 (nearest even) and INTEGER-added, so any accumulation order gives the same bits.
//
// Row-gather design: the fragment matrix is compacted (missing entries dropped) and transposed (per-SNP lists of
// covering fragment entries).  One CTA owns SNP row u at a time: for every covering fragment it walks the partners of u
// inside the linkage reach (both directions -- the relation |p - t| <= reach is symmetric) and accumulates the int64
// terms per partner v in shared memory.  Two table kinds, chosen per row by classify_kernel from cheap bounds:
//   * direct: the partners of u lie in the SNP-index window [vmin, vmax] (fragments are index-sorted); when the window
//     fits the table, slot = v - vmin -- no hashing, no compare-and-swap, and the row leaves already sorted through a
//     ballot compaction.  Every row of a short-range (non Pore-C) graph is of this kind.
//   * hash: few partners spread over a wide window (Pore-C contacts): open addressing (atomicCAS on the key, 64-bit
//     atomicAdd on the value), then a bitonic sort of the table by v.
// Rows are binned by (kind, table size) into six lists; each list is processed by a grid of resident CTAs that stride
// over it.  Pass 1 only counts distinct partners; an exclusive scan gives row_ptr; pass 2 fills.  No global sort, no
// global atomics on weights, HBM traffic ~ the compulsory input + output.
#include <math.h>

#include <algorithm>
#include <cstring>

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
  int4* meta;        // [cnnz] grouped by SNP: for covering entry (fragment i, position p): {first partner entry
                     //        base_i + tlo, p - tlo, partner range length thi - tlo + 1 (0 if k_i < 2), k_i - 1}
  int32_t* maux;     // [cnnz] same order: M bit | Phred << 8 | Pore-C flag << 16 of the covering entry
  uint8_t* cls;      // [n_snp] class of the row in pass 1 (0: no partners)
  int32_t* wbase;    // [n_snp] first SNP index of the row's partner window (slot 0 of a direct table)
  int4* list;        // [6][n_snp] rows of each class: {u, colptr[u], colptr[u + 1], wbase[u]}
  int32_t* cnt;      // [8] rows per class (index = class, 1..6)
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

struct Reach {
  int32_t base, p, k, tlo, thi;
  bool porec;
};

// linkage reach of compact entry ce inside its fragment (positions tlo .. thi of the fragment's compact entries)
__device__ __forceinline__ Reach reach_of(const Compact& c, const uint8_t* __restrict__ frag_flags, int32_t tenths, int32_t ce) {
  Reach r;
  const int32_t i = c.cfrag[ce];
  r.base = c.k[i];
  r.k = c.k[i + 1] - r.base;
  r.p = ce - r.base;
  r.porec = frag_flags && (frag_flags[i] & 1);
  const int32_t reach = r.porec ? (r.k - 1) : int32_t((int64_t(tenths) * (r.k - 1)) / 10);   // floor, L85; R8
  r.tlo = max(0, r.p - reach);
  r.thi = min(r.k - 1, r.p + reach);
  return r;
}

// transpose: every compact entry files its partner range under its SNP (order inside a SNP's list is arbitrary)
__global__ void __launch_bounds__(256) csc_fill_kernel(int32_t cnnz, const uint8_t* __restrict__ frag_flags, int32_t tenths,
                                                       Compact c) {
  const int32_t p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= cnnz) return;
  const int32_t u = c.csnp[p];
  const Reach r = reach_of(c, frag_flags, tenths, p);
  const int32_t s = c.colptr[u] + atomicAdd(&c.cursor[u], 1);
  c.meta[s] = make_int4(r.base + r.tlo, r.p - r.tlo, r.k >= 2 ? r.thi - r.tlo + 1 : 0, r.k - 1);
  c.maux[s] = int32_t(c.cm[p]) | (int32_t(c.cq[p]) << 8) | (r.porec ? (1 << 16) : 0);
}

// Class of each row from cheap bounds: distinct partners <= min(#contributions, index window - 1).
//   1 / 3 / 5: direct table of 128 / 1024 / 8192 slots (window fits);  2 / 4 / 6: hash table of the same sizes at a load
//   factor <= 2/3;  the cheapest table that is valid wins.  The row is appended to its class's list (one atomicAdd per
//   class and CTA; the order inside a list does not matter, every row owns its own output range).
constexpr int kNumClasses = 6;

// Appends row u to the list of class cl (0: none); all 256 threads of the CTA call it.  One global atomicAdd per class
// and CTA; the order inside a list does not matter (every row owns its own output range).
__device__ __forceinline__ void append_to_class(const Compact& c, int32_t n_snp, int cl, int32_t u, int32_t vmin) {
  __shared__ int s_cnt[kNumClasses + 1], s_off[kNumClasses + 1];
  if (threadIdx.x <= kNumClasses) s_cnt[threadIdx.x] = 0;
  __syncthreads();
  const int my = cl ? atomicAdd(&s_cnt[cl], 1) : 0;
  __syncthreads();
  if (threadIdx.x >= 1 && threadIdx.x <= kNumClasses && s_cnt[threadIdx.x])
    s_off[threadIdx.x] = atomicAdd(&c.cnt[threadIdx.x], s_cnt[threadIdx.x]);
  __syncthreads();
  if (cl) c.list[size_t(cl - 1) * n_snp + s_off[cl] + my] = make_int4(u, c.colptr[u], c.colptr[u + 1], vmin);
}

__global__ void __launch_bounds__(256) classify_kernel(int32_t n_snp, Compact c) {
  const int32_t u = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  int cl = 0;
  int32_t vmin = kEmpty, vmax = -1;
  if (u < n_snp) {
    int64_t contrib = 0;
    for (int32_t s = c.colptr[u] + lane; s < c.colptr[u + 1]; s += 32) {
      const int4 m = c.meta[s];
      if (m.z < 2) continue;
      contrib += m.z - 1;
      vmin = min(vmin, c.csnp[m.x]);
      vmax = max(vmax, c.csnp[m.x + m.z - 1]);
    }
    contrib = warp_sum(contrib);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      vmin = min(vmin, __shfl_xor_sync(0xffffffffu, vmin, o));
      vmax = max(vmax, __shfl_xor_sync(0xffffffffu, vmax, o));
    }
    if (contrib > 0) {
      const int64_t window = int64_t(vmax) - vmin + 1;
      const int64_t bound = min(contrib, window - 1);
      cl = window <= 128 ? 1 : bound <= 85 ? 2 : window <= 1024 ? 3 : bound <= 680 ? 4 : window <= 8192 ? 5 : bound <= 5400 ? 6 : 7;
      if (lane == 0) {
        c.wbase[u] = vmin;
        if (cl == 7) c.flags[2] = 1;
      }
      if (cl == 7) cl = 0;
    }
  }
  if (lane == 0 && u < n_snp) c.cls[u] = uint8_t(cl);
  append_to_class(c, n_snp, lane == 0 ? cl : 0, u, vmin);
}

// Pass 2 knows the exact number of distinct partners: a hash row takes the smallest table that holds it at a load
// factor <= 2/3 (a row with 70 partners over a wide window was sized by its ~1,000 contributions in pass 1).
__global__ void __launch_bounds__(256) reclassify_kernel(int32_t n_snp, const int32_t* __restrict__ row_ptr, Compact c) {
  const int32_t u = blockIdx.x * blockDim.x + threadIdx.x;
  int cl = 0;
  if (u < n_snp) {
    cl = c.cls[u];
    const int32_t cnt = row_ptr[u + 1] - row_ptr[u];
    if (cl == 2 || cl == 4 || cl == 6 || (cl == 5 && cnt <= 680)) cl = cnt <= 85 ? 2 : cnt <= 680 ? 4 : 6;
  }
  append_to_class(c, n_snp, cl, u, cl ? c.wbase[u] : 0);
}

// ascending sort of the first n (a power of two) table entries by key, all threads of the CTA
__device__ __forceinline__ void bitonic_sort(int32_t* keys, unsigned long long* vals, int n) {
  for (int size = 2; size <= n; size <<= 1)
    for (int stride = size >> 1; stride > 0; stride >>= 1) {
      __syncthreads();
      for (int t = threadIdx.x; t < n / 2; t += blockDim.x) {
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

// Rows of one class: CTAs stride over the class's list.  DIRECT: keys[] holds presence flags indexed by v - wbase[u];
// otherwise keys[] is the open-addressing key array.  vals[] are the int64 sums (two's complement through unsigned adds).
template <int TS, int THREADS, bool DIRECT, bool FILL>
__global__ void __launch_bounds__(THREADS) snp_rows_kernel(int32_t n_snp, int cls, double alpha, Compact c,
                                                           int32_t* __restrict__ row_ptr, int32_t* __restrict__ col,
                                                           int64_t* __restrict__ w_fx, float* __restrict__ w) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  unsigned long long* vals = reinterpret_cast<unsigned long long*>(smem_raw);
  int32_t* keys = reinterpret_cast<int32_t*>(smem_raw + size_t(TS) * 8);
  __shared__ int32_t n_keys;
  constexpr int NW = THREADS / 32;
  __shared__ int32_t w_tot[NW];
  __shared__ int32_t s_base[THREADS], s_self[THREADS], s_aux[THREADS], s_km1[THREADS], s_pref[THREADS + 1];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int32_t n_rows = c.cnt[cls];
  const int4* rows = c.list + size_t(cls - 1) * n_snp;
  int4 row = blockIdx.x < n_rows ? rows[blockIdx.x] : make_int4(0, 0, 0, 0);
  for (int32_t idx = blockIdx.x; idx < n_rows; idx += gridDim.x) {
    const int32_t u = row.x, f_begin = row.y, f_end = row.z;
    const int32_t vb = DIRECT ? row.w : 0;
    if (idx + int(gridDim.x) < n_rows) row = rows[idx + gridDim.x];          // next row's header, off the critical path
    for (int t = threadIdx.x; t < TS; t += THREADS) {
      keys[t] = DIRECT ? 0 : kEmpty;
      if (FILL) vals[t] = 0ull;
    }
    if (threadIdx.x == 0) n_keys = 0;
    __syncthreads();
    // The covering fragments are staged THREADS at a time (one 16-byte record per thread, written by the transpose),
    // their partner ranges are laid end to end by a prefix sum, and the threads stride over the flattened
    // (fragment, partner) list, four independent loads in flight each.
    for (int32_t f0 = f_begin; f0 < f_end; f0 += THREADS) {
      int32_t n_part = 0;
      if (f0 + int(threadIdx.x) < f_end) {
        const int4 m = c.meta[f0 + threadIdx.x];
        n_part = m.z;                                       // includes u's own position, skipped below
        s_base[threadIdx.x] = m.x;
        s_self[threadIdx.x] = m.y;
        s_km1[threadIdx.x] = m.w;
        if (FILL) s_aux[threadIdx.x] = c.maux[f0 + threadIdx.x];
      }
      // exclusive prefix sum of n_part over the CTA -> s_pref[0 .. THREADS]
      int32_t incl = n_part;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int32_t y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += y;
      }
      if (lane == 31) w_tot[warp] = incl;
      __syncthreads();
      int32_t woff = 0;
      for (int q = 0; q < warp; ++q) woff += w_tot[q];
      s_pref[threadIdx.x] = woff + incl - n_part;
      if (threadIdx.x == THREADS - 1) s_pref[THREADS] = woff + incl;
      __syncthreads();
      const int32_t total = s_pref[THREADS];
      int f = 0;                                            // fragment of the current j: advances monotonically
      for (int32_t j0 = threadIdx.x; j0 < total; j0 += 4 * THREADS) {
        int32_t ce2[4], fi[4], vv[4], mq[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const int32_t j = j0 + q * THREADS;
          ce2[q] = -1; fi[q] = 0; vv[q] = 0; mq[q] = 0;
          if (j < total) {
            while (s_pref[f + 1] <= j) ++f;                 // s_pref[THREADS] = total > j ends the scan
            const int lo = f;
            const int32_t t = j - s_pref[lo];
            if (t != s_self[lo]) {
              fi[q] = lo;
              ce2[q] = s_base[lo] + t;
              vv[q] = c.csnp[ce2[q]];
              if (FILL) mq[q] = int32_t(c.cm[ce2[q]]) | (int32_t(c.cq[ce2[q]]) << 8);
            }
          }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          if (ce2[q] < 0) continue;
          const int32_t v = vv[q];
          long long fx = 0;
          if (FILL) {
            const int32_t aux = s_aux[fi[q]];
            const int mu = aux & 0xff, qu = (aux >> 8) & 0xff, mv = mq[q] & 0xff, qv = (mq[q] >> 8) & 0xff;
            const double alpha_i = (aux & (1 << 16)) ? alpha : 1.0;                            // L350, R8
            const double km1 = double(s_km1[fi[q]]);
            const double sg = (mu == mv) ? 1.0 : -1.0;                                         // sgn(W_iu W_iv), Eq. 13
            const double T = (u < v) ? c.table[qu * 94 + qv] : c.table[qv * 94 + qu];          // lower SNP index first
            const double t1 = __dmul_rn(__dmul_rn(alpha_i, sg), T);
            const double term = __ddiv_rn(-t1, km1);                                           // Eq. 14
            fx = __double2ll_rn(__dmul_rn(term, 4294967296.0));                                // R6
          }
          if (DIRECT) {
            const uint32_t slot = uint32_t(v - vb);
            if (slot >= uint32_t(TS)) { c.flags[3] = 1; continue; }                            // not index-sorted input
            keys[slot] = 1;
            if (FILL) atomicAdd(&vals[slot], (unsigned long long)fx);
          } else {
            uint32_t h = (uint32_t(v) * 2654435761u) & (TS - 1);
            for (int probe = 0; probe < TS; ++probe) {
              const int32_t prev = atomicCAS(&keys[h], kEmpty, v);
              if (prev == kEmpty || prev == v) {
                if (FILL) atomicAdd(&vals[h], (unsigned long long)fx);
                else if (prev == kEmpty) atomicAdd(&n_keys, 1);
                break;
              }
              h = (h + 1) & (TS - 1);
              if (probe == TS - 1) c.flags[3] = 1;
            }
          }
        }
      }
      __syncthreads();                          // the staging arrays are reused by the next chunk
    }
    __syncthreads();
    if (DIRECT) {
      // ordered compaction: warp `warp` owns slots [warp SEG, (warp + 1) SEG)
      constexpr int SEG = TS / NW;
      int32_t cnt = 0;
      for (int g = 0; g < SEG; g += 32) cnt += __popc(__ballot_sync(0xffffffffu, keys[warp * SEG + g + lane] != 0));
      if (lane == 0) w_tot[warp] = cnt;
      __syncthreads();
      if (!FILL) {
        if (threadIdx.x == 0) {
          int32_t tot = 0;
          for (int q = 0; q < NW; ++q) tot += w_tot[q];
          row_ptr[u] = tot;
        }
      } else {
        int32_t pos = row_ptr[u];
        for (int q = 0; q < warp; ++q) pos += w_tot[q];
        for (int g = 0; g < SEG; g += 32) {
          const int slot = warp * SEG + g + lane;
          const bool on = keys[slot] != 0;
          const uint32_t m = __ballot_sync(0xffffffffu, on);
          if (on) {
            const int32_t o = pos + __popc(m & ((1u << lane) - 1u));
            const long long sv = (long long)vals[slot];
            col[o] = vb + slot;
            w_fx[o] = sv;
            w[o] = float(double(sv) * (1.0 / 4294967296.0));
          }
          pos += __popc(m);
        }
      }
    } else if (!FILL) {
      if (threadIdx.x == 0) row_ptr[u] = n_keys;
    } else {
      // occupied entries to the front (any order), padded with empty keys to a power of two, sorted, streamed out
      constexpr int E = TS / THREADS;
      int32_t kk[E];
      unsigned long long kv[E];
#pragma unroll
      for (int e = 0; e < E; ++e) {
        kk[e] = keys[e * THREADS + threadIdx.x];
        kv[e] = vals[e * THREADS + threadIdx.x];
      }
      __syncthreads();
#pragma unroll
      for (int e = 0; e < E; ++e)
        if (kk[e] != kEmpty) {
          const int32_t o = atomicAdd(&n_keys, 1);
          keys[o] = kk[e];
          vals[o] = kv[e];
        }
      __syncthreads();
      const int32_t base = row_ptr[u], cnt = row_ptr[u + 1] - base;
      if (n_keys != cnt && threadIdx.x == 0) c.flags[3] = 1;   // cannot happen: pass 1 counted the same table
      int n2 = 2;
      while (n2 < cnt) n2 <<= 1;
      n2 = min(n2, TS);
      for (int t = cnt + threadIdx.x; t < n2; t += THREADS) keys[t] = kEmpty;
      bitonic_sort(keys, vals, n2);
      for (int t = threadIdx.x; t < cnt; t += THREADS) {
        const long long sv = (long long)vals[t];
        col[base + t] = keys[t];
        w_fx[base + t] = sv;
        w[base + t] = float(double(sv) * (1.0 / 4294967296.0));
      }
    }
    __syncthreads();                            // the tables are reused by the next row
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

template <int TS, int THREADS, bool DIRECT, bool FILL>
qhap_status launch_class(int cls, int ctas_per_sm, int32_t n_snp, double alpha, const Compact& c, int32_t* row_ptr, int32_t* col, int64_t* w_fx, float* w, cudaStream_t stream) {
  auto kern = snp_rows_kernel<TS, THREADS, DIRECT, FILL>;
  if (TS * 12 > 48 * 1024) QHAP_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, TS * 12));   // per device
  const int grid = int(std::min<int64_t>(n_snp, int64_t(sm_count()) * ctas_per_sm));
  kern<<<grid, THREADS, TS * 12, stream>>>(n_snp, cls, alpha, c, row_ptr, col, w_fx, w);
  QHAP_LAUNCH_CHECK();
  return QHAP_OK;
}

// one resident wave per class; a class without rows costs an empty launch
template <bool FILL>
qhap_status launch_rows(int32_t n_snp, double alpha, const Compact& c, int32_t* row_ptr,
                        int32_t* col, int64_t* w_fx, float* w, cudaStream_t stream) {
  QHAP_TRY((launch_class<128, 64, true, FILL>(1, 32, n_snp, alpha, c, row_ptr, col, w_fx, w, stream)));
  QHAP_TRY((launch_class<128, 64, false, FILL>(2, 32, n_snp, alpha, c, row_ptr, col, w_fx, w, stream)));
  QHAP_TRY((launch_class<1024, 256, true, FILL>(3, 8, n_snp, alpha, c, row_ptr, col, w_fx, w, stream)));
  QHAP_TRY((launch_class<1024, 256, false, FILL>(4, 8, n_snp, alpha, c, row_ptr, col, w_fx, w, stream)));
  QHAP_TRY((launch_class<8192, 512, true, FILL>(5, 2, n_snp, alpha, c, row_ptr, col, w_fx, w, stream)));
  QHAP_TRY((launch_class<8192, 512, false, FILL>(6, 2, n_snp, alpha, c, row_ptr, col, w_fx, w, stream)));
  return QHAP_OK;
}

}  // namespace
}  // namespace qhap

using namespace qhap;

namespace {

// What the count pass leaves at the head of the workspace for qhap_build_snp_graph_fill to check.
struct SnpTag {
  int64_t magic, n_frag, n_snp, fnnz, tenths, alpha_bits, nnz;
  const void* row_ptr;
};
constexpr int64_t kSnpMagic = 0x51484150534e5031ll;   // "QHAPSNP1"

struct SnpWorkspace {
  SnpTag* tag;
  Compact c;
  int64_t* scan_scratch;
};

SnpWorkspace carve_snp(Workspace& ws, int32_t nf, int32_t ns, int64_t fnnz) {
  SnpWorkspace w;
  Compact& c = w.c;
  w.tag = ws.take<SnpTag>(1);
  c.k = ws.take<int32_t>(size_t(nf) + 1);
  c.csnp = ws.take<int32_t>(size_t(fnnz));
  c.cm = ws.take<uint8_t>(size_t(fnnz));
  c.cq = ws.take<uint8_t>(size_t(fnnz));
  c.cfrag = ws.take<int32_t>(size_t(fnnz));
  c.colptr = ws.take<int32_t>(size_t(ns) + 1);
  c.cursor = ws.take<int32_t>(size_t(ns));
  c.meta = ws.take<int4>(size_t(fnnz));
  c.maux = ws.take<int32_t>(size_t(fnnz));
  c.cls = ws.take<uint8_t>(size_t(ns));
  c.wbase = ws.take<int32_t>(size_t(ns));
  c.list = ws.take<int4>(size_t(kNumClasses) * size_t(ns));
  c.cnt = ws.take<int32_t>(8);
  c.flags = ws.take<int32_t>(4);
  c.total = ws.take<int64_t>(2);
  c.table = ws.take<double>(94 * 94);
  w.scan_scratch = ws.take<int64_t>(size_t(std::max(nf, ns)) / 4096 + 2);
  return w;
}

qhap_status check_snp_args(const qhap_frags* fr, const qhap_csr* out, int32_t linkage_tenths) {
  QHAP_REQUIRE(fr && out, "frags and out must not be NULL");
  QHAP_REQUIRE(fr->n_frag >= 0 && fr->n_snp >= 0, "negative sizes");
  QHAP_REQUIRE(linkage_tenths >= 1 && linkage_tenths <= 10, "linkage_tenths must be 1..10");
  QHAP_REQUIRE(fr->nnz >= 0 && fr->nnz < (int64_t(1) << 31), "fragment matrix must have < 2^31 entries");
  return QHAP_OK;
}

// Pass 1: compaction, transpose, classification, distinct-partner counts, row_ptr; *total = directed entries.
qhap_status snp_count_pass(const qhap_frags* fr, int32_t linkage_tenths, double alpha, const double* llr_table,
                           const SnpWorkspace& w, int32_t* row_ptr, int64_t* total, cudaStream_t stream) {
  const Compact& c = w.c;
  const int32_t nf = fr->n_frag, ns = fr->n_snp;
  std::vector<double> T(94 * 94);
  if (llr_table) std::copy(llr_table, llr_table + 94 * 94, T.begin());
  else host_llr_table(T.data());
  QHAP_CUDA_TRY(cudaMemcpyAsync(c.table, T.data(), sizeof(double) * 94 * 94, cudaMemcpyHostToDevice, stream));
  QHAP_CUDA_TRY(cudaMemsetAsync(w.tag, 0, sizeof(SnpTag), stream));
  QHAP_CUDA_TRY(cudaMemsetAsync(c.flags, 0, 4 * sizeof(int32_t), stream));
  QHAP_CUDA_TRY(cudaMemsetAsync(c.colptr, 0, sizeof(int32_t) * (size_t(ns) + 1), stream));
  QHAP_CUDA_TRY(cudaMemsetAsync(c.cursor, 0, sizeof(int32_t) * size_t(ns), stream));
  QHAP_CUDA_TRY(cudaMemsetAsync(c.cnt, 0, 8 * sizeof(int32_t), stream));
  if (nf > 0) {
    count_nonmissing_kernel<<<int(ceil_div(int64_t(nf) * 32, 256)), 256, 0, stream>>>(nf, fr->frag_ptr, fr->allele, c.k);
    QHAP_LAUNCH_CHECK();
  }
  QHAP_TRY(exclusive_scan_i32(c.k, c.k, nf, c.total, c.flags, stream, w.scan_scratch));
  if (nf > 0) {
    compact_kernel<<<int(ceil_div(int64_t(nf) * 32, 256)), 256, 0, stream>>>(nf, fr->frag_ptr, fr->snp_idx, fr->allele, fr->qual,
                                                                         fr->h1, c);
    QHAP_LAUNCH_CHECK();
  }
  QHAP_TRY(exclusive_scan_i32(c.colptr, c.colptr, ns, nullptr, nullptr, stream, w.scan_scratch));
  int64_t cnnz = 0;
  QHAP_CUDA_TRY(cudaMemcpyAsync(&cnnz, c.total, sizeof(int64_t), cudaMemcpyDeviceToHost, stream));
  QHAP_CUDA_TRY(cudaStreamSynchronize(stream));   // also keeps T alive until its copy is done
  if (cnnz > 0) {
    csc_fill_kernel<<<int(ceil_div(cnnz, 256)), 256, 0, stream>>>(int32_t(cnnz), fr->frag_flags, linkage_tenths, c);
    QHAP_LAUNCH_CHECK();
  }
  if (ns > 0) {
    classify_kernel<<<int(ceil_div(int64_t(ns) * 32, 256)), 256, 0, stream>>>(ns, c);
    QHAP_LAUNCH_CHECK();
    QHAP_CUDA_TRY(cudaMemsetAsync(row_ptr, 0, sizeof(int32_t) * (size_t(ns) + 1), stream));
    QHAP_TRY(launch_rows<false>(ns, alpha, c, row_ptr, nullptr, nullptr, nullptr, stream));
  }
  QHAP_TRY(exclusive_scan_i32(row_ptr, row_ptr, ns, c.total + 1, c.flags + 1, stream, w.scan_scratch));
  int32_t flags[4] = {0, 0, 0, 0};
  QHAP_CUDA_TRY(cudaMemcpyAsync(total, c.total + 1, sizeof(int64_t), cudaMemcpyDeviceToHost, stream));
  QHAP_CUDA_TRY(cudaMemcpyAsync(flags, c.flags, sizeof(flags), cudaMemcpyDeviceToHost, stream));
  QHAP_CUDA_TRY(cudaStreamSynchronize(stream));
  if (flags[1]) { set_error("SNP graph has >= 2^31 directed entries"); return QHAP_ERR_RANGE; }
  if (flags[2] || flags[3]) { set_error("a SNP has more than 5400 candidate partners (unsupported row size)"); return QHAP_ERR_RANGE; }
  return QHAP_OK;
}

// Pass 2: the rows are re-binned by their exact sizes and filled.
qhap_status snp_fill_pass(int32_t ns, double alpha, const SnpWorkspace& w, const qhap_csr* out, cudaStream_t stream) {
  if (ns == 0) return QHAP_OK;
  const Compact& c = w.c;
  QHAP_CUDA_TRY(cudaMemsetAsync(c.cnt, 0, 8 * sizeof(int32_t), stream));
  reclassify_kernel<<<int(ceil_div(ns, 256)), 256, 0, stream>>>(ns, out->row_ptr, c);
  QHAP_LAUNCH_CHECK();
  QHAP_TRY(launch_rows<true>(ns, alpha, c, out->row_ptr, out->col, out->w_fx, out->w, stream));
  int32_t flag = 0;
  QHAP_CUDA_TRY(cudaMemcpyAsync(&flag, c.flags + 3, sizeof(flag), cudaMemcpyDeviceToHost, stream));
  QHAP_CUDA_TRY(cudaStreamSynchronize(stream));
  if (flag) { set_error("SNP graph fill: table overflow (fragment SNP indices not strictly ascending?)"); return QHAP_ERR_INVALID_ARG; }
  return QHAP_OK;
}

}  // namespace

extern "C" qhap_status qhap_build_snp_graph(const qhap_frags* fr, int32_t linkage_tenths, double alpha,
                                            const double* llr_table, qhap_csr* out, void* workspace, size_t* ws_bytes,
                                            void* stream_v) {
  QHAP_TRY(check_snp_args(fr, out, linkage_tenths));
  const int32_t nf = fr->n_frag, ns = fr->n_snp;
  Workspace ws(workspace);
  const SnpWorkspace w = carve_snp(ws, nf, ns, fr->nnz);
  qhap_status st;
  if (workspace_protocol(ws, workspace, ws_bytes, &st)) return st;
  QHAP_TRY(require_device());
  QHAP_REQUIRE(out->row_ptr, "out->row_ptr must point to n_snp+1 ints");
  QHAP_REQUIRE(nf == 0 || (fr->frag_ptr && fr->snp_idx && fr->allele && fr->qual), "frag_ptr, snp_idx, allele and qual must not be NULL");
  cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
  const int64_t capacity = out->col ? out->nnz : 0;
  out->n = ns;
  int64_t total = 0;
  QHAP_TRY(snp_count_pass(fr, linkage_tenths, alpha, llr_table, w, out->row_ptr, &total, stream));
  out->nnz = total;
  // the workspace now holds everything pass 2 needs: tag it for qhap_build_snp_graph_fill
  SnpTag tag;
  std::memset(&tag, 0, sizeof(tag));
  tag.magic = kSnpMagic; tag.n_frag = nf; tag.n_snp = ns; tag.fnnz = fr->nnz; tag.tenths = linkage_tenths;
  std::memcpy(&tag.alpha_bits, &alpha, sizeof(double));
  tag.nnz = total; tag.row_ptr = out->row_ptr;
  QHAP_CUDA_TRY(cudaMemcpyAsync(w.tag, &tag, sizeof(tag), cudaMemcpyHostToDevice, stream));
  QHAP_CUDA_TRY(cudaStreamSynchronize(stream));   // `tag` is a stack object
  if (out->col == nullptr) return QHAP_OK;
  if (capacity < total) { set_error("edge capacity too small: %lld < %lld", (long long)capacity, (long long)total); return QHAP_ERR_WORKSPACE; }
  QHAP_REQUIRE(out->w_fx && out->w, "out->w_fx and out->w must not be NULL when out->col is given");
  return snp_fill_pass(ns, alpha, w, out, stream);
}

extern "C" qhap_status qhap_build_snp_graph_fill(const qhap_frags* fr, int32_t linkage_tenths, double alpha, qhap_csr* out,
                                                 void* workspace, size_t* ws_bytes, void* stream_v) {
  QHAP_TRY(check_snp_args(fr, out, linkage_tenths));
  const int32_t nf = fr->n_frag, ns = fr->n_snp;
  Workspace ws(workspace);
  const SnpWorkspace w = carve_snp(ws, nf, ns, fr->nnz);
  qhap_status st;
  if (workspace_protocol(ws, workspace, ws_bytes, &st)) return st;
  QHAP_TRY(require_device());
  QHAP_REQUIRE(out->row_ptr && out->col && out->w_fx && out->w, "out->row_ptr, col, w_fx and w must not be NULL");
  cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
  SnpTag tag;
  QHAP_CUDA_TRY(cudaMemcpyAsync(&tag, w.tag, sizeof(tag), cudaMemcpyDeviceToHost, stream));
  QHAP_CUDA_TRY(cudaStreamSynchronize(stream));
  int64_t alpha_bits;
  std::memcpy(&alpha_bits, &alpha, sizeof(double));
  QHAP_REQUIRE(tag.magic == kSnpMagic && tag.n_frag == nf && tag.n_snp == ns && tag.fnnz == fr->nnz &&
                   tag.tenths == linkage_tenths && tag.alpha_bits == alpha_bits && tag.row_ptr == out->row_ptr,
               "workspace does not hold the count pass of qhap_build_snp_graph for these arguments");
  if (out->nnz < tag.nnz) { set_error("edge capacity too small: %lld < %lld", (long long)out->nnz, (long long)tag.nnz); return QHAP_ERR_WORKSPACE; }
  out->n = ns;
  out->nnz = tag.nnz;
  return snp_fill_pass(ns, alpha, w, out, stream);
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
  int64_t* scan_scratch = ws.take<int64_t>(size_t(ceil_div(int64_t(n_out), 4096)) + 1);
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
  QHAP_TRY(exclusive_scan_i32(out->row_ptr, out->row_ptr, n_out, total_d, flags_d, stream, scan_scratch));
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
