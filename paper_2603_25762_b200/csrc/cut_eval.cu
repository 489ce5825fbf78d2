// (5) Cut / Ising-energy evaluation and best-replica selection.  PAPER.md:L254-L267 [Eq. 4-6].
//   cut_r = sum_{a<b, s_a != s_b} w_ab,  E_r = W_tot - 2 cut_r,  r* = lowest r with maximal cut.
// Integer arithmetic only (int32 counts or int64 2^-32 fixed point) -> bit-exact and order independent.
// The signs are first packed to one bit per (spin, replica) (pack_signs_kernel: 4 n R bytes of x read once, n R / 8 bytes
// written); the accumulation then runs on the packed words: lanes across replicas, a warp owns a tile of consecutive rows and
// a chunk of 32*VEC replicas, keeps VEC int64 partial cuts per lane in registers and flushes them with one atomicAdd per
// (lane, slot) when its tile (or the instance) ends.  Per edge a warp reads 4-16 bytes of packed signs instead of the
// neighbour's 128-512 bytes of fp32 x.
#include <atomic>

#include "kernels.cuh"

namespace qhap {

namespace {

constexpr int kRowsPerWarp = 8;   // a CTA of 8 warps owns 64 consecutive rows and one chunk of replicas
constexpr int kBitplaneMinR = 256; // above this many replicas the integer weight modes use the bit-plane kernel (below, its
                                   // 32-replica lanes are mostly empty and the per-replica kernel is cheaper)

// Packed signs: one bit per (spin, replica), word w of row a holds replicas 32 w .. 32 w + 31, bit set = spin -1.
// The accumulation kernel reads these words (R / 8 bytes per row) instead of gathering the neighbour's fp32 x row
// (4 R bytes) for every edge.
struct PackedBits {};

template <class SpinT, int VEC>
struct SpinLoad;

// load(base, row, R, r) returns a mask with bit k set when replica r + k of `row` is -1.
template <>
struct SpinLoad<PackedBits, 4> {
  static __device__ __forceinline__ uint32_t load(const PackedBits* base, int32_t row, int32_t R, int r) {
    const uint32_t W = uint32_t(R + 31) >> 5;
    const uint32_t w = __ldg(reinterpret_cast<const uint32_t*>(base) + size_t(row) * W + (uint32_t(r) >> 5));
    return (w >> (uint32_t(r) & 31u)) & 0xFu;                  // r is a multiple of 4: the four bits do not straddle a word
  }
};
template <>
struct SpinLoad<PackedBits, 1> {
  static __device__ __forceinline__ uint32_t load(const PackedBits* base, int32_t row, int32_t R, int r) {
    const uint32_t W = uint32_t(R + 31) >> 5;
    const uint32_t w = __ldg(reinterpret_cast<const uint32_t*>(base) + size_t(row) * W + (uint32_t(r) >> 5));
    return (w >> (uint32_t(r) & 31u)) & 1u;
  }
};

// sign sources of the packing kernel: int8 spins or fp32 positions (s = +1 if x >= 0 else -1, R10e)
__device__ __forceinline__ bool is_minus(int8_t v) { return v < 0; }
__device__ __forceinline__ bool is_minus(float v) { return !(v >= 0.f); }

// One warp per row: 32 replicas per ballot -> one word.
template <class SrcT>
__global__ void __launch_bounds__(256) pack_signs_kernel(int32_t n, int32_t R, const SrcT* __restrict__ src, uint32_t* __restrict__ bits) {
  const int lane = threadIdx.x & 31;
  const int32_t W = (R + 31) >> 5;
  const int64_t n_items = int64_t(n) * W;
  for (int64_t it = (int64_t(blockIdx.x) * blockDim.x + threadIdx.x) >> 5; it < n_items; it += (int64_t(gridDim.x) * blockDim.x) >> 5) {
    const int32_t a = int32_t(it / W), w = int32_t(it % W);
    const int r = w * 32 + lane;
    const bool m = r < R && is_minus(src[size_t(a) * R + r]);
    const uint32_t word = __ballot_sync(0xffffffffu, m);
    if (lane == 0) bits[it] = word;
  }
}

template <class SpinT, int VEC>
__global__ void __launch_bounds__(256) cut_accumulate_kernel(int32_t n, const int32_t* __restrict__ row_ptr,
                                                             const int32_t* __restrict__ col,
                                                             const int32_t* __restrict__ d, const int32_t* __restrict__ c,
                                                             const int64_t* __restrict__ w_fx, int mode,
                                                             const SpinT* __restrict__ spins, int32_t R, int32_t n_inst,
                                                             const int32_t* __restrict__ inst_ptr,
                                                             unsigned long long* __restrict__ cut,
                                                             unsigned long long* __restrict__ wtot) {
  // Work item of a CTA = (tile of 8 x kRowsPerWarp consecutive rows, chunk of 32 x VEC replicas); its 8 warps split the
  // rows.  The partial cuts of the 8 warps are summed in shared memory and leave with ONE atomicAdd per replica and CTA
  // (integer adds: any order gives the same bits); a tile that straddles an instance boundary flushes per warp instead.
  __shared__ long long s_acc[8][32 * VEC];
  const int lane = threadIdx.x & 31, wic = threadIdx.x >> 5;
  const int chunks = (R + 32 * VEC - 1) / (32 * VEC);
  constexpr int kTileRows = 8 * kRowsPerWarp;
  const int64_t n_tiles = (int64_t(n) + kTileRows - 1) / kTileRows;
  for (int64_t work = blockIdx.x; work < n_tiles * chunks; work += gridDim.x) {
    const int chunk = int(work % chunks);
    const int32_t t0 = int32_t(work / chunks) * kTileRows;
    const int32_t a0 = min(n, t0 + wic * kRowsPerWarp);
    const int32_t a1 = min(n, a0 + kRowsPerWarp);
    const int r = chunk * 32 * VEC + lane * VEC;
    const bool active = r < R;  // R % VEC == 0 is guaranteed by the dispatcher
    // instance of the first row (binary search; inst_ptr is tiny)
    int inst = 0;
    bool one_inst = true;         // the whole CTA tile lies in one instance (block-uniform)
    if (n_inst > 1) {
      int lo = 0, hi = n_inst;
      const int32_t key = min(a0, n - 1);
      while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (inst_ptr[mid] <= key) lo = mid; else hi = mid;
      }
      inst = lo;
      lo = 0; hi = n_inst;
      while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (inst_ptr[mid] <= t0) lo = mid; else hi = mid;
      }
      one_inst = min(n, t0 + kTileRows) <= inst_ptr[lo + 1];
    }
    int64_t acc[VEC];
#pragma unroll
    for (int k = 0; k < VEC; ++k) acc[k] = 0;
    int64_t wsum = 0;
    auto flush = [&](int b) {
      if (active) {
#pragma unroll
        for (int k = 0; k < VEC; ++k)
          if (acc[k] != 0) atomicAdd(&cut[size_t(b) * R + r + k], (unsigned long long)acc[k]);
      }
#pragma unroll
      for (int k = 0; k < VEC; ++k) acc[k] = 0;
      if (chunk == 0) {
        int64_t t = warp_sum(wsum);
        if (lane == 0 && t != 0) atomicAdd(&wtot[b], (unsigned long long)t);
      }
      wsum = 0;
    };
    for (int32_t a = a0; a < a1; ++a) {
      if (n_inst > 1 && a >= inst_ptr[inst + 1]) {
        flush(inst);
        while (a >= inst_ptr[inst + 1]) ++inst;
      }
      const int32_t e0 = row_ptr[a], e1 = row_ptr[a + 1];
      const uint32_t sa = active ? SpinLoad<SpinT, VEC>::load(spins, a, R, r) : 0u;
      for (int32_t eb = e0; eb < e1; eb += 32) {
        // lanes fetch 32 entries, then broadcast them one by one
        const int32_t e = eb + lane;
        int32_t my_col = -1;
        int64_t my_w = 0;
        if (e < e1) {
          my_col = col[e];
          if (my_col > a) my_w = edge_weight(mode, d, c, w_fx, e);   // each undirected edge once
        }
        if (chunk == 0 && my_col > a) wsum += my_w;
        const int cnt = min(32, e1 - eb);
        for (int j = 0; j < cnt; ++j) {            // every lane takes part in the shuffles; lower-triangle entries are skipped
          const int32_t b = __shfl_sync(0xffffffffu, my_col, j);
          const int64_t w = __shfl_sync(0xffffffffu, my_w, j);
          if (b <= a || !active) continue;
          const uint32_t diff = sa ^ SpinLoad<SpinT, VEC>::load(spins, b, R, r);
#pragma unroll
          for (int k = 0; k < VEC; ++k) acc[k] += ((diff >> k) & 1u) ? w : 0;
        }
      }
    }
    if (!one_inst) {
      flush(inst);
    } else {
#pragma unroll
      for (int k = 0; k < VEC; ++k) s_acc[wic][lane * VEC + k] = acc[k];
      if (chunk == 0) {
        int64_t t = warp_sum(wsum);
        if (lane == 0 && t != 0) atomicAdd(&wtot[inst], (unsigned long long)t);
      }
      __syncthreads();
      if (wic == 0 && active) {
#pragma unroll
        for (int k = 0; k < VEC; ++k) {
          long long t = 0;
#pragma unroll
          for (int w8 = 0; w8 < 8; ++w8) t += s_acc[w8][lane * VEC + k];
          if (t != 0) atomicAdd(&cut[size_t(inst) * R + r + k], (unsigned long long)t);
        }
      }
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------ bit-plane accumulation
// Integer weight modes (read graphs), one instance, many replicas.  Lanes run across the packed WORDS (lane = 32 replicas), an
// edge costs one XOR per lane, and the per-replica sums are kept BIT-SLICED: plane p of an accumulator is a word whose bit k
// is bit p of replica k's sum.  Adding the warp-uniform magnitude |w| to the replicas selected by diff = bits[a] ^ bits[b] is
// a ripple-carry adder of bitwise instructions -- about 2 LOP3 per plane for 32 replicas at once, instead of ~6 instructions
// per replica.  Two levels:
//   level 1: two unsigned accumulators of kP1 planes (edges with w > 0 / w < 0; unsigned, so that carries die out a plane or
//            two above the weight's top bit and the adder stops there), flushed every kL1Edges edges (16 (2^15 - 1) < 2^19);
//   level 2: one signed two's-complement accumulator of 32 planes (+= level-1 positive, -= level-1 negative), flushed at the
//            end of the warp's rows or after kItemEdges edges (|sum| < 2^15 2^15).
// A level-2 flush transposes the planes through shared memory, rebuilds one int32 per replica and adds it to cut[] with one
// coalesced 64-bit atomic per 32 replicas.  Weights with |w| >= 2^15 (not expected from read depths) take a per-replica atomic
// path.  All integer: any order of the additions gives the same bits as the oracle's sum.
constexpr int kP1 = 19, kL1Edges = 16, kItemEdges = 1 << 15;
constexpr int kBpWarps = 4;       // warps per CTA, each with its own items and its own 4 KB transposition tile

// acc += mag (warp-uniform, < 2^15) on the replicas whose bit is set in diff
__device__ __forceinline__ void bp_add(uint32_t (&acc)[kP1], uint32_t mag, uint32_t diff) {
  uint32_t carry = 0;
#pragma unroll
  for (int q = 0; q < (kP1 + 3) / 4; ++q) {
    const uint32_t rest = mag >> (4 * q);           // weight bits at and above this group of four planes
    if (rest == 0) {
      if (!__any_sync(0xffffffffu, carry != 0)) return;
#pragma unroll
      for (int p = 4 * q; p < 4 * q + 4 && p < kP1; ++p) {
        const uint32_t t = acc[p];
        acc[p] = t ^ carry;
        carry &= t;
      }
    } else {
#pragma unroll
      for (int p = 4 * q; p < 4 * q + 4 && p < kP1; ++p) {
        const uint32_t add = ((mag >> p) & 1u) ? diff : 0u;
        const uint32_t t = acc[p];
        acc[p] = t ^ add ^ carry;
        carry = (t & add) | (t & carry) | (add & carry);
      }
    }
  }
}

__global__ void __launch_bounds__(32 * kBpWarps) cut_bitplane_kernel(int32_t n, const int32_t* __restrict__ row_ptr, const int32_t* __restrict__ col,
                                                                    const int32_t* __restrict__ d, const int32_t* __restrict__ c, int mode,
                                                                    const uint32_t* __restrict__ bits, int32_t R, int32_t rows_per_item,
                                                                    unsigned long long* __restrict__ cut, unsigned long long* __restrict__ wtot) {
  __shared__ uint32_t s_t[kBpWarps][32][33];
  const int lane = threadIdx.x & 31, wic = threadIdx.x >> 5;
  const int32_t W = (R + 31) >> 5;
  const int chunks = (W + 31) >> 5;
  const int64_t n_items = int64_t((n + rows_per_item - 1) / rows_per_item) * chunks;
  uint32_t (*tile)[33] = s_t[wic];
  for (int64_t item = int64_t(blockIdx.x) * kBpWarps + wic; item < n_items; item += int64_t(gridDim.x) * kBpWarps) {
    const int chunk = int(item % chunks);
    const int32_t a0 = int32_t(item / chunks) * rows_per_item, a1 = min(n, a0 + rows_per_item);
    const int32_t wj = chunk * 32 + lane;
    const bool active = wj < W;
    uint32_t l1p[kP1], l1n[kP1], l2[32];
#pragma unroll
    for (int p = 0; p < kP1; ++p) { l1p[p] = 0; l1n[p] = 0; }
#pragma unroll
    for (int p = 0; p < 32; ++p) l2[p] = 0;
    int n1 = 0, n2 = 0;
    int64_t wsum = 0;
    auto flush1 = [&]() {                       // l2 += l1p (zero-extended); l2 -= l1n; both cleared
      uint32_t carry = 0, borrow = 0;
#pragma unroll
      for (int p = 0; p < 32; ++p) {
        const uint32_t add = p < kP1 ? l1p[p] : 0u, sub = p < kP1 ? l1n[p] : 0u;
        uint32_t t = l2[p];
        const uint32_t s1 = t ^ add ^ carry;
        carry = (t & add) | (t & carry) | (add & carry);
        t = s1;
        l2[p] = t ^ sub ^ borrow;
        borrow = (~t & sub) | (~t & borrow) | (sub & borrow);
      }
#pragma unroll
      for (int p = 0; p < kP1; ++p) { l1p[p] = 0; l1n[p] = 0; }
      n2 += n1;
      n1 = 0;
    };
    auto flush2 = [&]() {
      if (n1) flush1();
#pragma unroll
      for (int p = 0; p < 32; ++p) tile[p][lane] = l2[p];
      __syncwarp();
      const int words = min(32, W - chunk * 32);
      for (int j = 0; j < words; ++j) {         // word j of the chunk: lane k rebuilds replica 32 (32 chunk + j) + k
        uint32_t v = 0;
#pragma unroll
        for (int p = 0; p < 32; ++p) v = __funnelshift_r(v, tile[p][j] >> lane, 1);
        const int32_t r = (chunk * 32 + j) * 32 + lane;
        if (r < R && v != 0) atomicAdd(&cut[r], (unsigned long long)(long long)(int32_t)v);
      }
      __syncwarp();
#pragma unroll
      for (int p = 0; p < 32; ++p) l2[p] = 0;
      n2 = 0;
    };
    for (int32_t a = a0; a < a1; ++a) {
      const int32_t e0 = row_ptr[a], e1 = row_ptr[a + 1];
      const uint32_t sa = active ? __ldg(bits + size_t(a) * W + wj) : 0u;
      for (int32_t eb = e0; eb < e1; eb += 32) {
        const int32_t e = eb + lane;
        int32_t my_col = -1, my_w = 0;
        if (e < e1) {
          my_col = col[e];
          if (my_col > a) {                      // each undirected edge once
            const int64_t w = edge_weight(mode, d, c, nullptr, e);
            if (chunk == 0) wsum += w;
            const bool big = w >= (1 << 15) || w <= -(1 << 15);
            my_w = big ? 0 : int32_t(w);
            if (big) {                           // per-replica path, this lane walks the words of the chunk itself
              for (int j = 0; j < min(32, W - chunk * 32); ++j) {
                const int32_t wq = chunk * 32 + j;
                uint32_t df = __ldg(bits + size_t(a) * W + wq) ^ __ldg(bits + size_t(my_col) * W + wq);
                while (df) {
                  const int k = __ffs(df) - 1;
                  df &= df - 1;
                  if (wq * 32 + k < R) atomicAdd(&cut[wq * 32 + k], (unsigned long long)w);
                }
              }
            }
          }
        }
        uint32_t m = __ballot_sync(0xffffffffu, my_w != 0);
        // the neighbour's word of the NEXT listed edge is requested before the current one is added.  Every lane takes part
        // in every shuffle (the inactive ones too): the shuffles stay outside the `active` branches.
        uint32_t nxt = 0;
        int jn = m ? __ffs(m) - 1 : 0;
        const int32_t b0 = __shfl_sync(0xffffffffu, my_col, jn);
        if (m && active) nxt = __ldg(bits + size_t(b0) * W + wj);
        while (m) {
          const int j = jn;
          const uint32_t sb = nxt;
          m &= m - 1;
          jn = m ? __ffs(m) - 1 : 0;
          const int32_t bn = __shfl_sync(0xffffffffu, my_col, jn);
          if (m && active) nxt = __ldg(bits + size_t(bn) * W + wj);
          const int32_t w = __shfl_sync(0xffffffffu, my_w, j);
          const uint32_t diff = active ? (sa ^ sb) : 0u;
          if (w > 0) bp_add(l1p, uint32_t(w), diff); else bp_add(l1n, uint32_t(-w), diff);
          if (++n1 == kL1Edges) {
            flush1();
            if (n2 >= kItemEdges) flush2();
          }
        }
      }
    }
    flush2();
    if (chunk == 0) {
      const int64_t t = warp_sum(wsum);
      if (lane == 0 && t != 0) atomicAdd(&wtot[0], (unsigned long long)t);
    }
  }
}

// One CTA per instance: energy = W_tot - 2 cut, best replica = lowest index with maximal cut.
__global__ void __launch_bounds__(256) cut_finalize_kernel(int32_t R, const long long* __restrict__ cut,
                                                           const long long* __restrict__ wtot,
                                                           long long* __restrict__ energy,
                                                           long long* __restrict__ best_cut,
                                                           int32_t* __restrict__ best_replica) {
  const int b = blockIdx.x;
  __shared__ long long s_cut[256];
  __shared__ int s_idx[256];
  long long bc = 0;
  int bi = 0x7fffffff;
  for (int r = threadIdx.x; r < R; r += blockDim.x) {
    long long v = cut[size_t(b) * R + r];
    if (energy) energy[size_t(b) * R + r] = wtot[b] - 2 * v;
    if (bi == 0x7fffffff || v > bc) { bc = v; bi = r; }   // ascending r per thread: ties keep the lower index
  }
  s_cut[threadIdx.x] = bc;
  s_idx[threadIdx.x] = bi;
  __syncthreads();
  for (int o = blockDim.x / 2; o > 0; o >>= 1) {
    if (threadIdx.x < o) {
      long long v2 = s_cut[threadIdx.x + o];
      int i2 = s_idx[threadIdx.x + o];
      int i1 = s_idx[threadIdx.x];
      if (i2 != 0x7fffffff && (i1 == 0x7fffffff || v2 > s_cut[threadIdx.x] || (v2 == s_cut[threadIdx.x] && i2 < i1))) {
        s_cut[threadIdx.x] = v2;
        s_idx[threadIdx.x] = i2;
      }
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    if (best_cut) best_cut[b] = s_cut[0];
    if (best_replica) best_replica[b] = s_idx[0];
  }
}

__global__ void __launch_bounds__(256) gather_best_spins_kernel(int32_t n, int32_t R, const float* __restrict__ x,
                                                                int32_t n_inst, const int32_t* __restrict__ inst_ptr,
                                                                const int32_t* __restrict__ best_replica,
                                                                int8_t* __restrict__ best_spins) {
  const int32_t a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= n) return;
  int inst = 0;
  if (n_inst > 1) {
    int lo = 0, hi = n_inst;
    while (hi - lo > 1) {
      int mid = (lo + hi) >> 1;
      if (inst_ptr[mid] <= a) lo = mid; else hi = mid;
    }
    inst = lo;
  }
  best_spins[a] = (x[size_t(a) * R + best_replica[inst]] >= 0.f) ? int8_t(1) : int8_t(-1);
}

template <class SrcT>
qhap_status launch_cut(const CsrView& g, int mode, const SrcT* src, int32_t R, int32_t n_inst,
                       const int32_t* inst_ptr_dev, int64_t* cut, int64_t* wtot, uint32_t* bits, cudaStream_t stream) {
  QHAP_CUDA_TRY(cudaMemsetAsync(cut, 0, sizeof(int64_t) * size_t(n_inst) * R, stream));
  QHAP_CUDA_TRY(cudaMemsetAsync(wtot, 0, sizeof(int64_t) * size_t(n_inst), stream));
  if (g.n == 0 || R == 0) return QHAP_OK;
  const int64_t items = int64_t(g.n) * ((R + 31) / 32);
  pack_signs_kernel<SrcT><<<int(std::min<int64_t>(ceil_div(items, 8), int64_t(sm_count()) * 16)), 256, 0, stream>>>(g.n, R, src, bits);
  QHAP_LAUNCH_CHECK();
  auto* cu = reinterpret_cast<unsigned long long*>(cut);
  auto* wt = reinterpret_cast<unsigned long long*>(wtot);
  if (mode != QHAP_WEIGHT_FX && n_inst == 1 && R > kBitplaneMinR) {
    // rows per warp item: enough items for ~16 warps per SM, at least 2 and at most 16 rows (a level-2 flush per item)
    const int64_t chunks_w = ceil_div(ceil_div(R, 32), 32);
    const int32_t rows = int32_t(std::min<int64_t>(16, std::max<int64_t>(2, int64_t(g.n) * chunks_w / (int64_t(sm_count()) * 16))));
    const int64_t items = ceil_div(g.n, rows) * chunks_w;
    cut_bitplane_kernel<<<int(ceil_div(items, kBpWarps)), 32 * kBpWarps, 0, stream>>>(g.n, g.row_ptr, g.col, g.d, g.c, mode, bits, R, rows, cu, wt);
    QHAP_LAUNCH_CHECK();
    return QHAP_OK;
  }
  const bool vec4 = R % 4 == 0;
  const int chunks = vec4 ? (R + 127) / 128 : (R + 31) / 32;
  const int64_t work = ceil_div(g.n, 8 * kRowsPerWarp) * chunks;
  const int blocks = int(std::max<int64_t>(1, std::min<int64_t>(work, int64_t(sm_count()) * 8)));
  const PackedBits* pb = reinterpret_cast<const PackedBits*>(bits);
  if (vec4)
    cut_accumulate_kernel<PackedBits, 4><<<blocks, 256, 0, stream>>>(g.n, g.row_ptr, g.col, g.d, g.c, g.w_fx, mode, pb, R,
                                                                     n_inst, inst_ptr_dev, cu, wt);
  else
    cut_accumulate_kernel<PackedBits, 1><<<blocks, 256, 0, stream>>>(g.n, g.row_ptr, g.col, g.d, g.c, g.w_fx, mode, pb, R,
                                                                     n_inst, inst_ptr_dev, cu, wt);
  QHAP_LAUNCH_CHECK();
  return QHAP_OK;
}

}  // namespace

size_t cut_bits_words(int32_t n, int32_t R) { return size_t(n) * size_t((R + 31) / 32); }

qhap_status cut_from_spins(const CsrView& g, int mode, const int8_t* spins, int32_t R, int32_t n_inst,
                           const int32_t* inst_ptr_dev, int64_t* cut, int64_t* wtot, uint32_t* bits, cudaStream_t stream) {
  return launch_cut<int8_t>(g, mode, spins, R, n_inst, inst_ptr_dev, cut, wtot, bits, stream);
}

qhap_status cut_from_x(const CsrView& g, int mode, const float* x, int32_t R, int32_t n_inst,
                       const int32_t* inst_ptr_dev, int64_t* cut, int64_t* wtot, uint32_t* bits, cudaStream_t stream) {
  return launch_cut<float>(g, mode, x, R, n_inst, inst_ptr_dev, cut, wtot, bits, stream);
}

qhap_status cut_finalize(int32_t n_inst, int32_t R, const int64_t* cut, const int64_t* wtot, int64_t* energy,
                         int64_t* best_cut, int32_t* best_replica, cudaStream_t stream) {
  if (n_inst == 0) return QHAP_OK;
  cut_finalize_kernel<<<n_inst, 256, 0, stream>>>(R, reinterpret_cast<const long long*>(cut),
                                                  reinterpret_cast<const long long*>(wtot),
                                                  reinterpret_cast<long long*>(energy),
                                                  reinterpret_cast<long long*>(best_cut), best_replica);
  QHAP_LAUNCH_CHECK();
  return QHAP_OK;
}

qhap_status gather_best_spins(int32_t n, int32_t R, const float* x, int32_t n_inst, const int32_t* inst_ptr_dev,
                              const int32_t* best_replica, int8_t* best_spins, cudaStream_t stream) {
  if (n == 0) return QHAP_OK;
  gather_best_spins_kernel<<<int(ceil_div(n, 256)), 256, 0, stream>>>(n, R, x, n_inst, inst_ptr_dev, best_replica,
                                                                    best_spins);
  QHAP_LAUNCH_CHECK();
  return QHAP_OK;
}

}  // namespace qhap

// ------------------------------------------------------------------ qhap_cut_eval_static: the cut evaluation with NO workspace
// For callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc): the scratch of the
// cut evaluation -- W_tot and the packed sign bits -- lives in a file-scope device array of QHAP_CUT_STATIC_BYTES.  Every GPU
// that loads the library holds the array until the process exits.  In host code the array's NAME is a host-side stand-in, not
// a device address: the address comes from cudaGetSymbolAddress, once per device, with that device current.
// All calls on a device share the array: calls that overlap on the GPU (different streams) race.  It keeps the last call's
// contents; W_tot is cleared by launch_cut and every packed word a call reads is written by its own pack_signs_kernel.
namespace qhap {
namespace {
static __device__ __align__(256) unsigned char g_cut_static_scratch[QHAP_CUT_STATIC_BYTES];

constexpr int kStaticMaxDevices = 64;
constexpr size_t kStaticBitsOffset = 512;                 // [0, 8): W_tot; [256, 264): instance pointer (unused: one instance)
std::atomic<unsigned char*> g_cut_static_ptr[kStaticMaxDevices];

qhap_status cut_static_scratch(unsigned char** out) {
  int dev = -1;
  QHAP_CUDA_TRY(cudaGetDevice(&dev));
  QHAP_REQUIRE(dev >= 0 && dev < kStaticMaxDevices, "qhap_cut_eval_static: device ordinal %d not supported (max %d)", dev, kStaticMaxDevices - 1);
  unsigned char* p = g_cut_static_ptr[dev].load(std::memory_order_acquire);
  if (p == nullptr) {                                     // racing first calls resolve the same address twice: harmless
    void* sym = nullptr;
    QHAP_CUDA_TRY(cudaGetSymbolAddress(&sym, g_cut_static_scratch));
    QHAP_REQUIRE(sym != nullptr, "qhap_cut_eval_static: cudaGetSymbolAddress returned NULL");
    p = static_cast<unsigned char*>(sym);
    g_cut_static_ptr[dev].store(p, std::memory_order_release);
  }
  *out = p;
  return QHAP_OK;
}
}  // namespace
}  // namespace qhap

extern "C" qhap_status qhap_cut_eval_static(const qhap_csr* graph, int32_t weight_mode, const int8_t* spins, int32_t replicas,
                                            int64_t* cut, int64_t* energy, void* stream_v) {
  using namespace qhap;
  QHAP_REQUIRE(graph, "graph must not be NULL");
  QHAP_REQUIRE(graph->n >= 0 && graph->nnz >= 0 && replicas >= 1, "bad sizes");
  QHAP_REQUIRE(weight_mode >= 0 && weight_mode <= 2, "bad weight_mode");
  const size_t need = kStaticBitsOffset + sizeof(uint32_t) * cut_bits_words(graph->n, replicas);
  if (need > size_t(QHAP_CUT_STATIC_BYTES)) {
    set_error("qhap_cut_eval_static: n = %d spins x %d replicas need %zu bytes of scratch, the static array holds %zu "
              "(QHAP_CUT_STATIC_BYTES); use qhap_cut_eval with a caller workspace", graph->n, replicas, need, size_t(QHAP_CUT_STATIC_BYTES));
    return QHAP_ERR_WORKSPACE;
  }
  QHAP_TRY(require_device());
  QHAP_REQUIRE(spins && cut, "spins and cut must not be NULL");
  QHAP_REQUIRE(graph->n == 0 || (graph->row_ptr && (graph->nnz == 0 || graph->col)), "graph arrays must not be NULL");
  if (weight_mode == QHAP_WEIGHT_FX) QHAP_REQUIRE(graph->nnz == 0 || graph->w_fx, "w_fx required for weight_mode 2");
  else QHAP_REQUIRE(graph->nnz == 0 || (graph->d && (weight_mode == 0 || graph->c)), "d (and c) required for weight_mode 0/1");
  unsigned char* base = nullptr;
  QHAP_TRY(cut_static_scratch(&base));
  int64_t* wtot = reinterpret_cast<int64_t*>(base);
  const int32_t* inst_ptr = reinterpret_cast<const int32_t*>(base + 256);
  uint32_t* bits = reinterpret_cast<uint32_t*>(base + kStaticBitsOffset);
  cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
  const CsrView g = view_of(*graph);
  QHAP_TRY(launch_cut<int8_t>(g, weight_mode, spins, replicas, 1, inst_ptr, cut, wtot, bits, stream));
  QHAP_TRY(cut_finalize(1, replicas, cut, wtot, energy, nullptr, nullptr, stream));
  return QHAP_OK;
}
