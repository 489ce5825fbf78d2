// (3) Dense bSB step on the 5th-generation tensor cores: F = J X for all replicas as a tcgen05 GEMM with TMEM
// accumulators fed by TMA, with the y/x update, the a(t) ramp and the inelastic wall fused into the epilogue.
// PAPER.md:L252-L265 [Eq. 4-6] (the solver), L235-L246 (J = -w of the read graph); recurrence: DESIGN.md R10a-f.
//
// GEMM orientation: D[r][i] = sum_k xs[r][k] J[i][k], i.e.
//   A (M side) = replicas: the fp16 split copies x_hi, x_lo of the state, stored [R][n_k] (spin index contiguous = K-major);
//   B (N side) = output spins: rows of J (fp16, integers exact to 2048), row-major [ld][ld] (K-major);
//   D in TMEM: lane = replica, column = spin  ->  the epilogue's fp32 state accesses x[i][r], y[i][r] are coalesced
//   across the 32 lanes of a warp without any shared-memory transpose.
// x is carried in fp32; the tensor cores see 2^15 x = x_hi + x_lo (two fp16 terms, relative error <= 2^-23),
// both terms accumulate into the same fp32 TMEM tile against the same J tile in shared memory.
// Jacobi update across CTAs: the fp16 copies are double-buffered (read buffer b, write buffer 1-b); fp32 x, y are
// private to the tile that owns them and are updated in place.  One launch per step (grid-wide step boundary).
//
// Warp roles (608 threads): warp 0 = TMA producer, warp 1 = TMEM allocator + MMA issuer (one elected lane), warp 18 =
// TMA stores of the fp16 copies, warps 2..17 = epilogue (TMEM lane quarter = warp % 4, four warps per quarter interleave 8-column chunks; the state of
// the next chunk is prefetched into registers; at BN = 64 the fp16 copies leave through shared memory and TMA stores).
// Pipelines: n_stages shared-memory stages (full/empty mbarriers) and 2 TMEM accumulator stages (tmem_full/tmem_empty).
// Later additions, each described where it lives (DESIGN.md 4.4d-g): fused launches (all steps of a call in one cooperative
// launch, tile-level step boundary through done[]), state16 (x carried between steps as the fp16 pair; kernels X16), split
// accumulators, paired tiles (two 64-spin boxes per N = 128 accumulator; kernels PAIR), y by plain loads with its own epilogue
// loop (kernels YLDG), the fp32 x written next to the pair for the remainder gather of the hybrid block path (kernels XW).
#include <cuda.h>
#include <cuda_fp16.h>

#include <cstring>
#include <vector>

#include "kernels.cuh"
#include "sm100_ptx.cuh"

namespace qhap {

namespace {

constexpr int kBM = 128;                 // replicas per tile (UMMA M)
constexpr int kBK = 64;                  // spins per k-block: 64 fp16 = one 128-byte swizzle row
constexpr int kMaxBN = 256;              // output spins per tile (UMMA N), runtime 32..256 in steps of 16
constexpr int kMaxStages = 8;             // shared-memory pipeline depth: as many stages as fit (3 at BN = 256, 5 at BN = 64)
constexpr int kStageX = kBM * kBK * 2;               // 16 KB each for x_hi, x_lo
constexpr int kSmemBudget = 224 * 1024;              // operand stages (+ fp16 staging + state ring); + 1 KB slack + 1 KB barriers <= 227 KB
constexpr int kEpiWarps = 16;
constexpr int kChunk = 8;                // accumulator columns (spins) per tcgen05.ld in the epilogue
constexpr int kStoreWarp = 2 + kEpiWarps;  // one lane: TMA stores of the fp16 copies (+ the fused steps' progress signal)
constexpr int kThreads = 32 * (kStoreWarp + 1);
constexpr int kRingSlot = kChunk * 32 * 4;           // one work item of x (or y): 8 spins x 32 replicas fp32 = 1 KB
constexpr int kRingBytes = kEpiWarps * 2 * 2 * kRingSlot;   // per warp: 2 slots x (x, y)
constexpr int kRingBytes16 = kEpiWarps * 2 * kRingSlot;     // state16: per warp 2 slots x (y)
constexpr int kTmemCols = 512;                       // 2 accumulator stages x 256 columns
constexpr size_t kSmemBytes = size_t(kSmemBudget) + 1024 /*alignment slack*/ + 1024 /*barriers*/;

struct DenseArgs {
  int32_t n, R, n_k;          // spins, replicas, row pitch (elements) of the fp16 copies
  int32_t BN;                 // tile width in output spins
  int32_t n_stages;           // shared-memory stages of (BN x 64 J tile, 128 x 64 x_hi, 128 x 64 x_lo)
  int32_t ring;               // 1: the fp32 state of the work items arrives through per-warp TMA boxes (BN == 64, R % 4 == 0)
  int32_t stage_out;          // 1: the fp16 copies leave through swizzled shared-memory tiles and TMA stores (BN == 64)
  int32_t n_tiles_m, n_tiles_n, n_kblocks;
  uint32_t inv_tm;            // floor(2^32 / n_tiles_m) + 1: tile / n_tiles_m == umulhi(tile, inv_tm) for tile n_tiles_m < 2^32 (0: n_tiles_m == 1)
  const int32_t* kb_cnt;      // [n_tiles_n] number of listed k-blocks per N tile, or nullptr = all k-blocks
  const int32_t* kb_idx;      // [n_tiles_n][n_kblocks]
  const float* c1;            // [1] dt c0 (dense J), or per-row factors [n] when c1_per_row != 0 (block-compressed J)
  int32_t c1_per_row;
  int32_t j_terms;            // 1: J exact in fp16; 2: J = J_hi + J_lo (fp32 weights), a third MMA per k-slice
  const int32_t* blk_ptr;     // block-compressed J: tile (tn, j-th listed k-block) is block blk_ptr[tn] + j of the
                              // [blocks x 64][64] block arrays (nullptr: J is the dense matrix)
  float c2, c3;
  float* x;                   // [n][R] fp32, in place
  float* y;
  __half* xh_out;             // [R][n_k] next step's split copies
  __half* xl_out;
  // Fused steps: one launch runs n_steps bSB steps.  Virtual tile vt = s tile_stride + tile (step s of this launch); the
  // operand loads of tile (tn, tm) at step s wait until every tile (kb, tm), kb in tn's k-block list, has finished step
  // s - 1 (`done` counts the steps each tile has completed in this launch).  Needs BN == kBK (k-block == tile row),
  // k-block lists, TMA-stored copies and at least two tiles per CTA and step (state prefetch distance).
  int32_t n_steps;            // steps run by this launch (1 unless fused)
  int32_t fused;
  int32_t tile_stride;        // n_tiles rounded up to a multiple of the grid
  int32_t k0, steps_total;    // ramp (R10b): step index of s = 0, T
  double dt, a0;
  uint32_t* done;             // [n_tiles_n * n_tiles_m], zero at launch
  uint32_t fence_every;       // state ring: generic -> async proxy fence after every fence_every-th tile of a CTA
  // L2 eviction priorities: when x and the four fp16 copies fit the L2 next to the streaming y, they are
  // kept (evict_last) and y passes through (evict_first); otherwise both are the normal policy
  uint64_t pol_keep, pol_stream;
  uint32_t store_warp;        // 1: warp 18 issues the TMA stores of the fp16 copies (mbarrier hand-off; needed by fused launches
                              // and by a single staging buffer); 0: epilogue thread 0 issues them behind a named barrier
  uint32_t epi_sync;          // 1: the epilogue warps meet at a named barrier after every tile
  uint32_t stg_bufs;          // staging buffers of (x_hi', x_lo') tiles: 2, or 1 to free 32 KB for another operand stage
  // state16 (X16 kernels): between the steps of a call x lives ONLY as the fp16 pair the tensor cores read (2^15 x = x_hi + x_lo,
  // [R][n_k] arrays); the tile's own pair arrives in the staging buffer by TMA, is updated IN PLACE and leaves by TMA store.
  // The fp32 x array is not touched by the step kernel (split before the first step, merged after the last).
  int32_t x16;
  int32_t dsb;                // dSB: the copies hold 2^15 sgn(x) (x_lo = 0), so F = J sgn(x)
  // split accumulators: the tcgen05 fp32 accumulation truncates toward zero at every MMA, a bias of a few ulp of F.  The
  // small terms (x_lo J and x_hi J_lo, 2^-11 of the leading one) go to a second accumulator 128 TMEM columns further, where
  // their truncation is 2^-11 smaller; the epilogue adds the two.  Halves the MMAs that truncate at full magnitude.
  // Needs BN <= 128 (two accumulator stages x 2 x 128 columns = the 512 TMEM columns).
  int32_t sacc;
  // state16: y of the next work item comes by plain coalesced loads into registers instead of the per-warp TMA ring (frees
  // the ring's 32 KB for a fourth operand stage; every thread re-reads only y values it wrote itself one step earlier)
  int32_t yldg;
  // Paired tiles (state16, tile_skip lists, dense J): the unit of CTA work is a SLOT = one 64-spin box, or a PAIR of boxes
  // (2q, 2q + 1) of the same replica tile that share one N = 128 accumulator: every staged x k-block then feeds 128 output
  // spins instead of 64 (the operand feed -- bytes in flight per SM against the L2 latency -- is what bounds the 64-wide
  // step).  Slots of a step: first the pairs (q-major, replica tile fastest), then the remaining boxes as singles; the state
  // side (staging buffers, TMA stores, done[]) stays per box.  pair_lines = pairs per replica tile (0: every slot is a box).
  // state16 next to a remainder CSR (hybrid block path): the remainder gather reads fp32 x rows of the whole graph between two
  // tile steps, so the epilogue also writes x' = (x_hi' + x_lo') 2^-15 to the fp32 array (write only: 20 B per spin-update)
  int32_t xw32;
  // fused state16: the staging buffer is reloaded (the pair of the box two ahead) as soon as the store has READ it, before the
  // store's completion is waited for and signalled.  Safe only if that box is not the one just stored, i.e. every CTA has at
  // least three boxes per step (its pair was then stored, and waited for, at least one box earlier).
  int32_t early_reload;
  int32_t pair_lines, n_slots;
  const int32_t* pk_cnt;      // [pair_lines] union of the two boxes' k-block lists
  const int32_t* pk_idx;      // [pair_lines][n_kblocks]
  // block path: the union lists are stored back to back (pair q: entries pk_ptr[q] .. pk_ptr[q + 1]) with, per entry, the tile of
  // the left and of the right box in the block arrays (a box that does not list the k-block points at an all-zero tile)
  const int32_t* pk_ptr;      // [pair_lines + 1] or nullptr (dense path: pk_cnt / pk_idx)
  const int32_t* pk_kb;
  const int32_t* pk_l;
  const int32_t* pk_r;
};

struct Slot { int tn0, tm, width, q; };

// c2 = fp32(dt (a0 - a_k)), a_k = a0 k / (T - 1): the same individually rounded fp64 operations as the host loop
__device__ __forceinline__ float ramp_c2(const DenseArgs& a, int s) {
  const double a_k = a.steps_total > 1 ? __ddiv_rn(__dmul_rn(a.a0, double(a.k0 + s)), double(a.steps_total - 1)) : 0.0;
  return __double2float_rn(__dmul_rn(a.dt, __dsub_rn(a.a0, a_k)));
}

// tile -> (N tile, M tile), M fastest; the division by the run-time n_tiles_m is a multiply-high (an integer division costs
// ~20 instructions, and the epilogue needs the pair for every 8-spin work item)
__device__ __forceinline__ void tile_split(const DenseArgs& a, int tile, int& tn, int& tm) {
  tn = a.inv_tm ? int(__umulhi(uint32_t(tile), a.inv_tm)) : tile;
  tm = tile - tn * a.n_tiles_m;
}

// slot -> (first box, replica tile, width); slots [0, pair_lines n_tiles_m) are pairs, the rest single boxes
template <bool PAIR>
__device__ __forceinline__ Slot slot_of(const DenseArgs& a, int slot) {
  Slot s;
  tile_split(a, slot, s.q, s.tm);
  if (PAIR && s.q < a.pair_lines) { s.tn0 = 2 * s.q; s.width = 2; }
  else { s.tn0 = PAIR ? s.q + a.pair_lines : s.q; s.width = 1; }
  return s;
}
// k-block list of a slot (nullptr: all k-blocks)
template <bool PAIR>
__device__ __forceinline__ const int32_t* slot_list(const DenseArgs& a, const Slot& sl, int& nkb) {
  if (a.kb_cnt == nullptr) { nkb = a.n_kblocks; return nullptr; }
  if (PAIR && sl.width == 2) {
    if (a.pk_ptr) { const int32_t b = a.pk_ptr[sl.q]; nkb = a.pk_ptr[sl.q + 1] - b; return a.pk_kb + b; }
    nkb = a.pk_cnt[sl.q];
    return a.pk_idx + size_t(sl.q) * a.n_kblocks;
  }
  nkb = a.kb_cnt[sl.tn0];
  return a.kb_idx + size_t(sl.tn0) * a.n_kblocks;
}

// fp32 -> two fp16 terms of xs = 2^15 x (|x| <= 1 -> |xs| <= 32768, inside fp16's range): hi = rn(xs), lo = rn(xs - hi)
// (the difference is exact in fp32).  The scale keeps lo a NORMAL fp16 number for every |x| >= 2^-17, so that
// |xs - hi - lo| <= 2^-23 |xs|: a relative resolution one bit short of fp32's at every magnitude (unscaled, lo would be
// a subnormal below |x| = 0.25 and the resolution an absolute 2^-25).  The accumulator then holds 2^15 F; the epilogue
// folds the exact factor 2^-15 into c1, so fma(c1 2^-15, 2^15 F, .) == fma(c1, F, .) bit for bit.
constexpr float kXScale = 32768.0f;
__device__ __forceinline__ void split_half(float v, __half& hi, __half& lo) {
  const float vs = v * kXScale;
  hi = __float2half_rn(vs);
  lo = __float2half_rn(vs - __half2float(hi));
}

// state16: the pair IS the state, so it must be a fixed point of the split: (h, l) == split((h + l) 2^-15).  rn(xs - h) can
// round up to exactly half an ulp of h, and h + l then re-splits to the neighbouring (h', l') with the same sum; splitting
// the (exact) sum once more gives the canonical pair, for which x fp32 -> pair -> x fp32 -> pair reproduces itself, so a
// resumed call continues bit for bit.
__device__ __forceinline__ void split_half_canonical(float v, __half& hi, __half& lo) {
  __half h, l;
  split_half(v, h, l);
  const float s2 = __half2float(h) + __half2float(l);      // exact: at most 23 significant bits
  hi = __float2half_rn(s2);
  lo = __float2half_rn(s2 - __half2float(hi));              // exact
}
__device__ __forceinline__ void split_sign(float v, __half& hi, __half& lo) {     // dSB operand: 2^15 sgn(x), sgn(0) = +1
  hi = __float2half_rn(v >= 0.f ? kXScale : -kXScale);
  lo = __float2half_rn(0.f);
}

struct EpiConsts {
  float c1, c2, c3;
  int lane_r;            // replica of this thread inside the tile
};

// One bSB update (R10a-f) of a (spin, replica) plus the fp16 split of the new x.
__device__ __forceinline__ void epi_point(const EpiConsts& ec, float c1, float F, float x, float y, float& xn, float& yn) {
  yn = fmaf(c1, F, fmaf(-ec.c2, x, y));
  xn = fmaf(ec.c3, yn, x);
  if (fabsf(xn) > 1.0f) {                    // inelastic wall, strict inequality (R10d)
    xn = copysignf(1.0f, xn);
    yn = 0.0f;
  }
}
template <int MODE>   // 0: fp32-x kernels, 1: dSB sign copies, 2: state16 canonical pair
__device__ __forceinline__ void epi_pack(int j, float xn, uint32_t (&hp)[kChunk / 2], uint32_t (&lp)[kChunk / 2]) {
  __half h, l;
  if constexpr (MODE == 2) split_half_canonical(xn, h, l);
  else if constexpr (MODE == 1) split_sign(xn, h, l);
  else split_half(xn, h, l);
  const uint32_t hb = __half_as_ushort(h), lb = __half_as_ushort(l);
  if (j & 1) { hp[j >> 1] |= hb << 16; lp[j >> 1] |= lb << 16; }
  else       { hp[j >> 1] = hb;        lp[j >> 1] = lb; }
}

// fp32 state of one work item (kChunk spins x this thread's replica) -> registers; masked entries read as 0.
// Element offsets are 32-bit (the host checks n R < 2^32): one integer add and one wide multiply-add per address.
__device__ __forceinline__ void epi_load(const DenseArgs& a, const EpiConsts& ec, int tn, int tm, int ch, float (&xv)[kChunk],
                                         float (&yv)[kChunk]) {
  const int r = tm * kBM + ec.lane_r, i0 = tn * a.BN + ch * kChunk;
  const bool r_ok = r < a.R;
  uint32_t off = uint32_t(i0) * uint32_t(a.R) + uint32_t(r);
  if (r_ok && i0 + kChunk <= a.n) {          // interior item: no per-element predicates
#pragma unroll
    for (int j = 0; j < kChunk; ++j, off += uint32_t(a.R)) {
      xv[j] = a.x[off];
      yv[j] = a.y[off];
    }
  } else {
#pragma unroll
    for (int j = 0; j < kChunk; ++j, off += uint32_t(a.R)) {
      const bool ok = r_ok && (i0 + j) < a.n;
      xv[j] = ok ? a.x[off] : 0.f;
      yv[j] = ok ? a.y[off] : 0.f;
    }
  }
}

// Fused update of one work item: y' = y + dt(-(a0 - a_k) x + c0 F), x' = x + dt a0 y', inelastic wall; stores x', y'
// (fp32, coalesced across the warp's 32 replicas) and the fp16 split of x' (16 contiguous bytes per thread and array: into the staging tiles, or directly).
template <bool hints>
__device__ __forceinline__ void epi_update_store(const DenseArgs& a, const EpiConsts& ec, int tn, int tm, int ch,
                                                 const uint32_t (&v)[kChunk], const float (&xv)[kChunk],
                                                 const float (&yv)[kChunk], uint32_t stg) {
  const int r = tm * kBM + ec.lane_r, i0 = tn * a.BN + ch * kChunk;
  const bool r_ok = r < a.R;
  uint32_t off = uint32_t(i0) * uint32_t(a.R) + uint32_t(r);
  uint32_t hp[kChunk / 2], lp[kChunk / 2];    // fp16 pairs (spin i0 + 2q, i0 + 2q + 1) of x_hi', x_lo'
  float xs[kChunk];
  if (r_ok && i0 + kChunk <= a.n) {
#pragma unroll
    for (int j = 0; j < kChunk; ++j, off += uint32_t(a.R)) {
      float xn, yn;
      const float c1 = a.c1_per_row ? __ldg(a.c1 + i0 + j) : ec.c1;
      epi_point(ec, c1, __uint_as_float(v[j]), xv[j], yv[j], xn, yn);
      if constexpr (hints) {
        ptx::st_global_f32_hint(a.x + off, xn, a.pol_keep);
        ptx::st_global_f32_hint(a.y + off, yn, a.pol_stream);
      } else {
        a.x[off] = xn;
        a.y[off] = yn;
      }
      xs[j] = xn;
    }
  } else {
#pragma unroll
    for (int j = 0; j < kChunk; ++j, off += uint32_t(a.R)) {
      const bool ok = r_ok && (i0 + j) < a.n;
      float xn, yn;
      const float c1 = (a.c1_per_row && (i0 + j) < a.n) ? __ldg(a.c1 + i0 + j) : ec.c1;
      epi_point(ec, c1, __uint_as_float(v[j]), xv[j], yv[j], xn, yn);
      if (ok) {
        ptx::st_global_f32_hint(a.x + off, xn, a.pol_keep);
        ptx::st_global_f32_hint(a.y + off, yn, a.pol_stream);
      }
      xs[j] = ok ? xn : 0.f;              // masked entries: zeros in the copies (dSB: sgn(0) = +1, never read -- J is 0 there)
    }
  }
  if (a.dsb) {                              // one warp-uniform branch per work item, outside the unrolled loops
#pragma unroll
    for (int j = 0; j < kChunk; ++j) epi_pack<1>(j, xs[j], hp, lp);
  } else {
#pragma unroll
    for (int j = 0; j < kChunk; ++j) epi_pack<0>(j, xs[j], hp, lp);
  }
  if (stg != 0) {
    // staging tile [128 replicas][64 spins] fp16 per array, rows of 128 B, 16-byte pieces XOR-swizzled by (row & 7):
    // the layout a TMA box {64, 128} with the 128-byte swizzle expects; x_lo's tile follows x_hi's (16 KB each)
    const int row = ec.lane_r;
    const uint32_t base = stg + uint32_t(row) * 128u;
#pragma unroll
    for (int q = 0; q < kChunk / 8; ++q) {
      const uint32_t piece = uint32_t(((ch * kChunk) >> 3) + q) ^ uint32_t(row & 7);
      ptx::st_shared_v4(base + piece * 16u, hp[4 * q], hp[4 * q + 1], hp[4 * q + 2], hp[4 * q + 3]);
      ptx::st_shared_v4(base + kStageX + piece * 16u, lp[4 * q], lp[4 * q + 1], lp[4 * q + 2], lp[4 * q + 3]);
    }
  } else if (r_ok && i0 < a.n) {               // n_k >= round_up(n, 64) keeps the kChunk-spin run in bounds
    uint4* ph = reinterpret_cast<uint4*>(a.xh_out + size_t(r) * a.n_k + i0);
    uint4* pl = reinterpret_cast<uint4*>(a.xl_out + size_t(r) * a.n_k + i0);
#pragma unroll
    for (int q = 0; q < kChunk / 8; ++q) {
      ph[q] = make_uint4(hp[4 * q], hp[4 * q + 1], hp[4 * q + 2], hp[4 * q + 3]);
      pl[q] = make_uint4(lp[4 * q], lp[4 * q + 1], lp[4 * q + 2], lp[4 * q + 3]);
    }
  }
}

// state16: one work item (kChunk spins x this thread's replica).  x comes from the tile's own (x_hi, x_lo) in the staging
// buffer `stg` (TMA-loaded, 128-byte swizzle: 16-byte piece p of row r sits at piece p ^ (r & 7)), x = (x_hi + x_lo) 2^-15
// exactly; the new canonical pair goes back to the SAME 16 bytes (this thread is their only reader and writer), y' to global.
// Rows / replicas outside the problem arrive as zeros (TMA fill), stay zero (F = 0 there) and are clipped by the TMA store.
// The arithmetic runs on xs = 2^15 x directly (every factor 2^15 is exact): y' = fma(c1 2^-15, 2^15 F, fma(-(c2 2^-15), xs, y)),
// xs' = fma(c3 2^15, y', xs), wall at |xs'| > 2^15 -- bit for bit the fp32 update of x.  Pairs of spins are split and
// canonicalised with packed fp16 instructions: (h, l) = (rn(xs'), rn(xs' - h)); H = h + l in fp16 (= rn16 of the exact sum),
// L = (h - H) + l (both exact): (H, L) has the same sum and is a fixed point of the split (see split_half_canonical).
template <bool hints, bool PER_ROW, bool XW = false>
__device__ __forceinline__ void epi_update_x16(const DenseArgs& a, const EpiConsts& ec, int tn, int tm, int ch, const uint32_t (&v)[kChunk],
                                               const float (&yv)[kChunk], uint32_t stg) {
  const int r = tm * kBM + ec.lane_r, i0 = tn * a.BN + ch * kChunk;
  const int row = ec.lane_r;
  static_assert(kChunk == 8, "one work item = one 16-byte piece of the swizzled staging row");
  const uint32_t addr = stg + uint32_t(row) * 128u + ((uint32_t(ch) ^ uint32_t(row & 7)) << 4);
  uint32_t hq[4], lq[4];
  ptx::ld_shared_v4(addr, hq[0], hq[1], hq[2], hq[3]);
  ptx::ld_shared_v4(addr + kStageX, lq[0], lq[1], lq[2], lq[3]);
  const bool interior = r < a.R && i0 + kChunk <= a.n;
  float c1v[kChunk];
  if constexpr (PER_ROW) {
    if (i0 + kChunk <= a.n) {                  // 32-byte aligned run of the per-row factors (warp-uniform address)
      const float4 ca = __ldg(reinterpret_cast<const float4*>(a.c1 + i0)), cb = __ldg(reinterpret_cast<const float4*>(a.c1 + i0 + 4));
      c1v[0] = ca.x; c1v[1] = ca.y; c1v[2] = ca.z; c1v[3] = ca.w; c1v[4] = cb.x; c1v[5] = cb.y; c1v[6] = cb.z; c1v[7] = cb.w;
    } else {
#pragma unroll
      for (int j = 0; j < kChunk; ++j) c1v[j] = (i0 + j) < a.n ? __ldg(a.c1 + i0 + j) : 0.f;
    }
  }
  float yn[kChunk];
  float xf[XW ? kChunk : 1];
  uint32_t hp[kChunk / 2], lp[kChunk / 2];
#pragma unroll
  for (int q = 0; q < kChunk / 2; ++q) {
    const float2 hf = __half22float2(*reinterpret_cast<const __half2*>(&hq[q]));
    const float2 lf = __half22float2(*reinterpret_cast<const __half2*>(&lq[q]));
    float xn[2];
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      const int j = 2 * q + e;
      const float xs = e ? hf.y + lf.y : hf.x + lf.x;                       // exact
      const float c1 = PER_ROW ? c1v[j] : ec.c1;
      float y1 = fmaf(c1, __uint_as_float(v[j]), fmaf(-ec.c2, xs, yv[j]));
      float x1 = fmaf(ec.c3, y1, xs);
      if (fabsf(x1) > kXScale) {               // inelastic wall, strict inequality (R10d), in units of 2^-15
        x1 = copysignf(kXScale, x1);
        y1 = 0.0f;
      }
      xn[e] = x1; yn[j] = y1;
    }
    const __half2 h = __floats2half2_rn(xn[0], xn[1]);
    const float2 hb = __half22float2(h);
    const __half2 l = __floats2half2_rn(xn[0] - hb.x, xn[1] - hb.y);
    const __half2 H = __hadd2(h, l);
    const __half2 L = __hadd2(__hsub2(h, H), l);
    hp[q] = *reinterpret_cast<const uint32_t*>(&H);
    lp[q] = *reinterpret_cast<const uint32_t*>(&L);
    if constexpr (XW) {                          // the fp32 value of the pair, as merge_x_kernel forms it
      const float2 Hf = __half22float2(H), Lf = __half22float2(L);
      xf[2 * q] = (Hf.x + Lf.x) * (1.0f / kXScale);
      xf[2 * q + 1] = (Hf.y + Lf.y) * (1.0f / kXScale);
    }
  }
  uint32_t off = uint32_t(i0) * uint32_t(a.R) + uint32_t(r);
  if (interior) {
    float* yb = a.y + off;
#pragma unroll
    for (int j = 0; j < kChunk; ++j) {
      if constexpr (hints) ptx::st_global_f32_hint(yb + uint32_t(j) * uint32_t(a.R), yn[j], a.pol_stream);
      else yb[uint32_t(j) * uint32_t(a.R)] = yn[j];
      if constexpr (XW) a.x[off + uint32_t(j) * uint32_t(a.R)] = xf[j];
    }
  } else if (r < a.R) {
#pragma unroll
    for (int j = 0; j < kChunk; ++j, off += uint32_t(a.R))
      if (i0 + j < a.n) {
        a.y[off] = yn[j];
        if constexpr (XW) a.x[off] = xf[j];
      }
  }
  ptx::st_shared_v4(addr, hp[0], hp[1], hp[2], hp[3]);
  ptx::st_shared_v4(addr + kStageX, lp[0], lp[1], lp[2], lp[3]);
}

// RING: the fp32 state arrives through the per-warp TMA ring; HINTS: L2 eviction priorities on every state access.
// Compile-time variants keep each instantiation's hot loops small (the single run-time kernel had grown from 63 to 88 KB
// of SASS and cost cfg3 3 %).
// YLDG (state16 only): y by plain loads instead of the ring.  XW (YLDG kernels without pairs): the epilogue also writes the fp32
// x (DenseArgs::xw32; its own instantiation: as a run-time branch it cost cfg3 3.6 % through the size of the item loop).
template <bool RING, bool HINTS, bool X16, bool PAIR, bool YLDG, bool XW>
__global__ void __launch_bounds__(kThreads, 1)
dense_step_kernel(const __grid_constant__ CUtensorMap tm_j, const __grid_constant__ CUtensorMap tm_jl,
                  const __grid_constant__ CUtensorMap tm_xh,
                  const __grid_constant__ CUtensorMap tm_xl, const __grid_constant__ CUtensorMap tm_oh,
                  const __grid_constant__ CUtensorMap tm_ol, const __grid_constant__ CUtensorMap tm_sx,
                  const __grid_constant__ CUtensorMap tm_sy, const DenseArgs a) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;       // 128B swizzle needs 1024-byte alignment
  const int kStages = a.n_stages;
  const uint32_t kTileJ = uint32_t(a.BN) * kBK * 2;                    // one J tile; a second one (J_lo) follows if j_terms == 2
  // paired tiles: room for the J tiles of both boxes (rows 0..63 | 64..127 of one N = 128 operand)
  const uint32_t kStageJ = kTileJ * uint32_t(a.j_terms) * (PAIR ? 2u : 1u), kStageBytes = kStageJ + 2 * kStageX;
  const uint32_t bar_base = smem_base + kSmemBudget;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (kMaxStages + s); };
  auto tfull_bar = [&](int s) { return bar_base + 8u * (2 * kMaxStages + s); };
  auto tempty_bar = [&](int s) { return bar_base + 8u * (2 * kMaxStages + 2 + s); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * kMaxStages + 4);
  auto ring_bar = [&](int s) { return bar_base + 8u * (2 * kMaxStages + 6 + s); };
  auto stg_full = [&](uint32_t b) { return bar_base + 8u * (2 * kMaxStages + 6 + 2 * kEpiWarps + b); };       // staging tile b written
  auto stg_empty = [&](uint32_t b) { return bar_base + 8u * (2 * kMaxStages + 8 + 2 * kEpiWarps + b); };      // ... read by its TMA store
  auto stg_in = [&](uint32_t b) { return bar_base + 8u * (2 * kMaxStages + 10 + 2 * kEpiWarps + b); };        // state16: the tile's own pair has arrived
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == 0 && ptx::elect_one()) {
    ptx::prefetch_tensormap(&tm_j);
    ptx::prefetch_tensormap(&tm_xh);
    ptx::prefetch_tensormap(&tm_xl);
    ptx::prefetch_tensormap(&tm_oh);
    ptx::prefetch_tensormap(&tm_ol);
    for (int s = 0; s < kStages; ++s) {
      ptx::mbar_init(full_bar(s), 1);
      ptx::mbar_init(empty_bar(s), 1);
    }
    for (int s = 0; s < 2; ++s) {
      ptx::mbar_init(tfull_bar(s), 1);
      ptx::mbar_init(tempty_bar(s), kEpiWarps);
    }
    for (int s = 0; s < 2 * kEpiWarps; ++s) ptx::mbar_init(ring_bar(s), 1);
    for (uint32_t b = 0; b < 2; ++b) {
      ptx::mbar_init(stg_full(b), kEpiWarps);
      ptx::mbar_init(stg_empty(b), 1);
      ptx::mbar_init(stg_in(b), 1);
    }
    ptx::fence_barrier_init();
  }
  if (warp == 1) ptx::tmem_alloc(tmem_slot, kTmemCols);
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  // Programmatic dependent launch: the next step's CTAs may be scheduled as soon as SMs free up (their prologue above
  // -- barrier init, TMEM allocation, descriptor prefetch -- overlaps this step's tail); everything below reads state
  // written by the previous step, so it first waits for that grid to have completed and flushed.
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  const int n_tiles = a.n_slots;                                          // slots of a step (boxes, or pairs of boxes)
  const int stride = a.tile_stride, vt_end = a.n_steps * a.tile_stride;   // virtual slots: step-major, holes in [n_slots, stride)

  if (warp == 0) {
    // ===================================================================================== TMA producer
    // Lane 0 issues the loads.  Fused steps: before a tile of step s > 0 the WHOLE warp polls the progress counters of
    // the tiles it reads (one k-block per lane, so the L2 round trips overlap), then lane 0 crosses to the async proxy.
    if (lane == 0 || a.fused) {
      int stage = 0;
      uint32_t phase = 0;
      for (int vt = blockIdx.x; vt < vt_end; vt += gridDim.x) {
        const int s = vt / stride, slot = vt - s * stride;
        if (slot >= n_tiles) continue;
        const Slot sl = slot_of<PAIR>(a, slot);                                // replica tile fastest: neighbouring CTAs share the J tile in L2
        const int tn = sl.tn0, tm = sl.tm;
        int nkb;
        const int32_t* list = slot_list<PAIR>(a, sl, nkb);
        if (s > 0) {
          for (int j = lane; j < nkb; j += 32)                           // box (kb, tm) has finished step s - 1
            ptx::wait_at_least_acquire(a.done + list[j] * a.n_tiles_m + tm, uint32_t(s));
          __syncwarp();
          ptx::fence_proxy_async_global();
        }
        if (lane != 0) continue;
        const CUtensorMap* mh = (s & 1) ? &tm_oh : &tm_xh;               // odd steps of a fused launch read what even steps wrote
        const CUtensorMap* ml = (s & 1) ? &tm_ol : &tm_xl;
        const uint32_t stage_tx = kTileJ * uint32_t(a.j_terms) * uint32_t(sl.width) + 2u * kStageX;
        // the list entries of k-block j + 1 are requested before k-block j is issued, so that their round trip is not on the
        // path of every stage
        const bool bpair = PAIR && sl.width == 2 && a.blk_ptr != nullptr;
        const int32_t e0 = bpair ? a.pk_ptr[sl.q] : 0;
        int kb_n = list ? list[0] : 0, tl_n = bpair ? a.pk_l[e0] : 0, tr_n = bpair ? a.pk_r[e0] : 0;
        for (int j = 0; j < nkb; ++j) {
          const int kb = kb_n, tl = tl_n, tr = tr_n;
          if (j + 1 < nkb) {
            kb_n = list ? list[j + 1] : j + 1;
            if (bpair) { tl_n = a.pk_l[e0 + j + 1]; tr_n = a.pk_r[e0 + j + 1]; }
          }
          ptx::mbar_wait(empty_bar(stage), phase ^ 1);
          const uint32_t sj = smem_base + stage * kStageBytes;
          ptx::mbar_arrive_expect_tx(full_bar(stage), stage_tx);
          if (a.blk_ptr) {
            if (bpair) {                                              // one J term; tiles of the left and the right box
              ptx::tma_load_2d(sj, &tm_j, full_bar(stage), 0, tl * kBK);
              ptx::tma_load_2d(sj + kTileJ, &tm_j, full_bar(stage), 0, tr * kBK);
            } else {
              const int brow = (a.blk_ptr[tn] + j) * kBK;
              ptx::tma_load_2d(sj, &tm_j, full_bar(stage), 0, brow);
              if (a.j_terms == 2) ptx::tma_load_2d(sj + kTileJ, &tm_jl, full_bar(stage), 0, brow);
            }
          } else {
            ptx::tma_load_2d(sj, &tm_j, full_bar(stage), kb * kBK, tn * a.BN);
            if (PAIR && sl.width == 2) ptx::tma_load_2d(sj + kTileJ, &tm_j, full_bar(stage), kb * kBK, (tn + 1) * a.BN);   // rows 64..127
          }
          if constexpr (HINTS) {
            ptx::tma_load_2d_hint(sj + kStageJ, mh, full_bar(stage), kb * kBK, tm * kBM, a.pol_keep);
            ptx::tma_load_2d_hint(sj + kStageJ + kStageX, ml, full_bar(stage), kb * kBK, tm * kBM, a.pol_keep);
          } else {
            ptx::tma_load_2d(sj + kStageJ, mh, full_bar(stage), kb * kBK, tm * kBM);
            ptx::tma_load_2d(sj + kStageJ + kStageX, ml, full_bar(stage), kb * kBK, tm * kBM);
          }
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ======================================================================================= MMA issuer
    const uint32_t idesc1 = ptx::umma_idesc_f16_f32(kBM, uint32_t(a.BN)), idesc2 = ptx::umma_idesc_f16_f32(kBM, 2u * uint32_t(a.BN));
    int stage = 0;
    uint32_t phase = 0;
    int acc = 0;
    uint32_t acc_phase = 0;
    for (int vt = blockIdx.x; vt < vt_end; vt += gridDim.x) {
      const int slot = vt % stride;
      if (slot >= n_tiles) continue;
      const Slot sl = slot_of<PAIR>(a, slot);
      int nkb;
      (void)slot_list<PAIR>(a, sl, nkb);
      const uint32_t idesc = (PAIR && sl.width == 2) ? idesc2 : idesc1;
      ptx::mbar_wait(tempty_bar(acc), acc_phase ^ 1);                    // epilogue has drained this accumulator stage
      ptx::tc_fence_after();
      const uint32_t d_tmem = tmem_base + uint32_t(acc) * kMaxBN;
      for (int j = 0; j < nkb; ++j) {
        ptx::mbar_wait(full_bar(stage), phase);
        ptx::tc_fence_after();
        if (ptx::elect_one()) {
          const uint32_t sj = smem_base + stage * kStageBytes;
          const uint64_t dj = ptx::umma_desc_k_sw128(sj);
          const uint64_t djl = ptx::umma_desc_k_sw128(sj + kTileJ);
          const uint64_t dh = ptx::umma_desc_k_sw128(sj + kStageJ);
          const uint64_t dl = ptx::umma_desc_k_sw128(sj + kStageJ + kStageX);
          // UMMA_K = 16 for 16-bit inputs: +32 B per step.  Two straight-line variants: a test of j_terms inside the
          // unrolled issue sequence costs the full GEMM 12 % (measured: 165 -> 186 us per step at cfg1).
          if (a.dsb) {                    // dSB: the operand is 2^15 sgn(x), x_lo = 0 -> one MMA per J term and k-slice
#pragma unroll
            for (int kk = 0; kk < kBK / 16; ++kk) {
              ptx::umma_f16(d_tmem, dh + 2u * kk, dj + 2u * kk, idesc, (j | kk) != 0);
              if (a.j_terms == 2) ptx::umma_f16(d_tmem, dh + 2u * kk, djl + 2u * kk, idesc, 1u);
            }
          } else if (a.sacc) {              // small terms (x_lo J, x_hi J_lo: 2^-11 of the leading one) into their own accumulator
            const uint32_t d2 = d_tmem + 128u;
            if (a.j_terms == 2) {
#pragma unroll
              for (int kk = 0; kk < kBK / 16; ++kk) {
                ptx::umma_f16(d_tmem, dh + 2u * kk, dj + 2u * kk, idesc, (j | kk) != 0);
                ptx::umma_f16(d2, dl + 2u * kk, dj + 2u * kk, idesc, (j | kk) != 0);
                ptx::umma_f16(d2, dh + 2u * kk, djl + 2u * kk, idesc, 1u);
              }
            } else {
#pragma unroll
              for (int kk = 0; kk < kBK / 16; ++kk) {
                ptx::umma_f16(d_tmem, dh + 2u * kk, dj + 2u * kk, idesc, (j | kk) != 0);
                ptx::umma_f16(d2, dl + 2u * kk, dj + 2u * kk, idesc, (j | kk) != 0);
              }
            }
          } else if (a.j_terms == 2) {
#pragma unroll
            for (int kk = 0; kk < kBK / 16; ++kk) {
              ptx::umma_f16(d_tmem, dh + 2u * kk, dj + 2u * kk, idesc, (j | kk) != 0);
              ptx::umma_f16(d_tmem, dl + 2u * kk, dj + 2u * kk, idesc, 1u);
              ptx::umma_f16(d_tmem, dh + 2u * kk, djl + 2u * kk, idesc, 1u);   // x_lo J_lo ~ 2^-22: dropped
            }
          } else {
#pragma unroll
            for (int kk = 0; kk < kBK / 16; ++kk) {
              ptx::umma_f16(d_tmem, dh + 2u * kk, dj + 2u * kk, idesc, (j | kk) != 0);
              ptx::umma_f16(d_tmem, dl + 2u * kk, dj + 2u * kk, idesc, 1u);
            }
          }
          ptx::umma_commit(empty_bar(stage));                            // frees the smem stage when these MMAs are done
          if (j == nkb - 1) ptx::umma_commit(tfull_bar(acc));            // accumulator complete -> epilogue
        }
        __syncwarp();
        if (++stage == kStages) { stage = 0; phase ^= 1; }
      }
      if (++acc == 2) { acc = 0; acc_phase ^= 1; }
    }
  } else if (warp == kStoreWarp) {
    // ==================================================================================== fp16 copy stores
    // One thread hands each finished pair of staging tiles to TMA, returns the buffer once the bulk reads are done and --
    // fused steps -- signals the tile's completion (done[tile] += 1) once the writes have COMPLETED.  Off the epilogue's
    // critical path: the epilogue warps only arrive on / wait for the two staging barriers.
    if (a.stage_out && a.store_warp && lane == 0) {
      const uint32_t stg_base = smem_base + uint32_t(kStages) * kStageBytes;
      uint32_t b = 0, bpar = 0;
      // state16: this thread also brings each tile's OWN (x_hi, x_lo) into the staging buffer, stg_bufs tiles ahead; the
      // epilogue updates the buffer in place and the store below writes it to the other copy.  A buffer is reloaded right
      // after its store has read it.  Fused steps: the tile's own pair of step s - 1 was stored (and waited for with
      // wait_group 0) by this same thread at least stg_bufs tiles earlier -- every CTA has >= 2 tiles per step.
      int vt_ld = blockIdx.x, bx_ld = 0;             // next box to load: slot vt_ld, box bx_ld of it
      uint32_t b_ld = 0;
      auto load_next = [&]() {
        while (vt_ld < vt_end) {
          const int s = vt_ld / stride, slot = vt_ld - s * stride;
          if (slot >= n_tiles) { vt_ld += gridDim.x; continue; }
          const Slot sl = slot_of<PAIR>(a, slot);
          const int tn = sl.tn0 + bx_ld, tm = sl.tm;
          const uint32_t stg = stg_base + b_ld * (2u * kStageX);
          ptx::mbar_arrive_expect_tx(stg_in(b_ld), 2u * kStageX);
          if constexpr (HINTS) {
            ptx::tma_load_2d_hint(stg, (s & 1) ? &tm_oh : &tm_xh, stg_in(b_ld), tn * a.BN, tm * kBM, a.pol_keep);
            ptx::tma_load_2d_hint(stg + kStageX, (s & 1) ? &tm_ol : &tm_xl, stg_in(b_ld), tn * a.BN, tm * kBM, a.pol_keep);
          } else {
            ptx::tma_load_2d(stg, (s & 1) ? &tm_oh : &tm_xh, stg_in(b_ld), tn * a.BN, tm * kBM);
            ptx::tma_load_2d(stg + kStageX, (s & 1) ? &tm_ol : &tm_xl, stg_in(b_ld), tn * a.BN, tm * kBM);
          }
          if (!PAIR || ++bx_ld == sl.width) { bx_ld = 0; vt_ld += gridDim.x; }
          if (++b_ld == a.stg_bufs) b_ld = 0;
          return;
        }
      };
      if constexpr (X16) {
        for (uint32_t q = 0; q < a.stg_bufs; ++q) load_next();
      }
      for (int vt = blockIdx.x; vt < vt_end; vt += gridDim.x) {
        const int s = vt / stride, slot = vt - s * stride;
        if (slot >= n_tiles) continue;
        const Slot sl = slot_of<PAIR>(a, slot);
        for (int bx = 0; bx < (PAIR ? sl.width : 1); ++bx) {
        const int tn = sl.tn0 + bx, tm = sl.tm;
        const uint32_t stg = stg_base + b * (2u * kStageX);
        ptx::mbar_wait(stg_full(b), bpar);
        if constexpr (HINTS) {
          ptx::tma_store_2d_hint((s & 1) ? &tm_xh : &tm_oh, stg, tn * a.BN, tm * kBM, a.pol_keep);
          ptx::tma_store_2d_hint((s & 1) ? &tm_xl : &tm_ol, stg + kStageX, tn * a.BN, tm * kBM, a.pol_keep);
        } else {
          ptx::tma_store_2d((s & 1) ? &tm_xh : &tm_oh, stg, tn * a.BN, tm * kBM);
          ptx::tma_store_2d((s & 1) ? &tm_xl : &tm_ol, stg + kStageX, tn * a.BN, tm * kBM);
        }
        ptx::tma_store_commit();
        ptx::tma_store_wait_read_all();
        if constexpr (!X16) ptx::mbar_arrive(stg_empty(b));
        if constexpr (X16) { if (a.early_reload) load_next(); }   // into the buffer just read (b_ld == b)
        if (a.fused) {
          ptx::tma_store_wait_all();
          ptx::signal_add_release(a.done + (tn * a.n_tiles_m + tm), 1u);
        }
        if constexpr (X16) { if (!a.early_reload) load_next(); }
        if (++b == a.stg_bufs) { b = 0; bpar ^= 1u; }
        }
      }
      ptx::tma_store_wait_all();                   // the bulk stores have completed before this thread exits
    }
  } else {
    // ========================================================================================= epilogue
    // Work item = (tile, 16-column chunk).  The fp32 state of item k+1 is loaded into registers before item k is
    // computed and stored (two register buffers, alternated by a 2x unrolled loop), across tile boundaries too: the
    // loads do not depend on the accumulator, so they are in flight while the warp waits for tmem_full.
    const int ew = warp - 2;
    const int quarter = warp & 3;              // TMEM lanes 32 q .. 32 q + 31 are accessible to warps with warp % 4 == q
    const int par = ew >> 2;                   // the kEpiWarps / 4 warps of a quarter take chunks par, par + P, par + 2P, ...
    constexpr int P = kEpiWarps / 4;
    EpiConsts ec;
    ec.c1 = a.c1_per_row ? 0.f : __ldg(a.c1) * (1.0f / kXScale);    // accumulator = 2^15 F (per-row factors include it)
    // state16 works on xs = 2^15 x: the exact powers of two move into the constants
    constexpr float kC2s = X16 ? 1.0f / kXScale : 1.0f, kC3s = X16 ? kXScale : 1.0f;
    ec.c2 = a.c2 * kC2s; ec.c3 = a.c3 * kC3s;
    ec.lane_r = quarter * 32 + lane;
    int acc = 0;
    uint32_t acc_phase = 0;
    // fp16 output staging: two buffers of (x_hi tile, x_lo tile) behind the operand stages, alternated per tile
    const uint32_t stg_base = smem_base + uint32_t(kStages) * kStageBytes;
    uint32_t tcount = 0;
    int cur_s = 0;                             // step (of this launch) whose ramp constant ec.c2 holds
    if (a.fused) ec.c2 = ramp_c2(a, 0) * kC2s;
    // every warp owns chunk `par` of every tile (possibly fully masked), so that it arrives on tmem_empty once per tile.
    // Items are addressed by the VIRTUAL tile (step-major); the last wave of a step may have a hole for this CTA.
    // A position carries the virtual tile (ordering, end test) and the real tile next to it, so that the item loop needs
    // no division by the runtime stride.
    // vt / rt: virtual and real slot; bx: box of the slot (0, or 1 in a pair); (tn, tm) of the BOX travel along
    struct Pos { int vt, rt, ch, tn, tm, bx, width; };
    auto next_box = [&](Pos& p) {                           // first item of this warp in the box after p's
      p.ch = par;
      if constexpr (PAIR) {
        if (p.bx + 1 < p.width) {                           // second box of a pair: same accumulator, columns BN .. 2 BN - 1
          ++p.bx; ++p.tn;
          return;
        }
      }
      p.vt += gridDim.x; p.rt += gridDim.x;
      if (p.rt >= n_tiles) {                                // past the step's slots
        if (p.rt < stride) { p.vt += gridDim.x; p.rt += gridDim.x; }   // hole in the last wave (stride % grid == 0)
        p.rt -= stride;                                     // first wave of the next step
      }
      const Slot sl = slot_of<PAIR>(a, p.rt);
      p.tn = sl.tn0; p.tm = sl.tm; p.bx = 0; p.width = sl.width;
    };
    auto advance = [&](Pos& p) {
      p.ch += P;
      if (p.ch * kChunk >= a.BN || p.tn * a.BN + p.ch * kChunk >= a.n) next_box(p);
    };
    auto first_pos = [&]() {
      const Slot sl = slot_of<PAIR>(a, int(blockIdx.x));
      return Pos{int(blockIdx.x), int(blockIdx.x), par, sl.tn0, sl.tm, 0, sl.width};
    };
    auto same_box = [](const Pos& p, const Pos& q) { return p.vt == q.vt && (!PAIR || p.bx == q.bx); };
    auto box_of = [](const Pos& p) { return PAIR ? p.bx : 0; };
    int step_end = stride;                     // first virtual tile of step cur_s + 1
    auto set_step = [&](int vt) {              // items are visited in ascending vt
      if (a.fused && vt >= step_end) { ++cur_s; step_end += stride; ec.c2 = ramp_c2(a, cur_s) * kC2s; }
    };
    uint32_t stg_i = 0, stg_par = 0;           // staging buffer of the current tile and its use parity
    // last chunk of this warp in a tile: hand the accumulator stage back and arrive on the staging tile's barrier (the
    // store warp takes it from there).  Fused steps: the fp32 state was written with generic stores and is re-read
    // through TMA one step later by the same warp (requested while the warp works on the tile BEFORE it in the CTA's
    // order), so every lane crosses to the async proxy in between: after every fence_every-th tile, with
    // fence_every <= (fewest tiles a CTA has per step) - 1, the fence that follows a tile's stores comes at most
    // fence_every - 1 tiles later, the request at least (tiles per step) - 1 tiles later.
    int cur_tn = 0, cur_tm = 0;                // box of the item being finished (for the store below)
    auto tile_done = [&](bool slot_end) {      // last chunk of this warp in a box; slot_end: ... and in the slot's accumulator
      if (slot_end) {
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(tempty_bar(acc));
        if (++acc == 2) { acc = 0; acc_phase ^= 1; }
      }
      if (a.stage_out && a.store_warp) {
        ptx::fence_proxy_async();
        if constexpr (RING && !YLDG) {                  // only the TMA ring re-reads generic stores through the async proxy
          if (a.fused && ++tcount == a.fence_every) { tcount = 0; ptx::fence_proxy_async_global(); }
        }
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(stg_full(stg_i));
        if (++stg_i == a.stg_bufs) { stg_i = 0; stg_par ^= 1u; }
        if (a.epi_sync) ptx::named_barrier_sync(1, kEpiWarps * 32);       // measured: cfg1 32.3 -> 31.4 us per step
      } else if (a.stage_out) {
        // one launch per step with two staging buffers (cfg3, cfg4: 3 % faster than the store warp there): thread 0 waits
        // until the previous tile's stores have read their buffer, all epilogue warps meet, thread 0 issues the stores
        ptx::fence_proxy_async();
        if (ew == 0 && lane == 0) ptx::tma_store_wait_read_all();
        ptx::named_barrier_sync(1, kEpiWarps * 32);
        if (ew == 0 && lane == 0) {
          const uint32_t stg = stg_base + stg_i * (2u * kStageX);
          ptx::tma_store_2d(&tm_oh, stg, cur_tn * a.BN, cur_tm * kBM);
          ptx::tma_store_2d(&tm_ol, stg + kStageX, cur_tn * a.BN, cur_tm * kBM);
          ptx::tma_store_commit();
        }
        stg_i ^= 1u;
      }
    };
    // first chunk of a tile: the accumulator must be complete
    auto tile_begin = [&]() {
      ptx::mbar_wait(tfull_bar(acc), acc_phase);
      ptx::tc_fence_after();
    };
    // ... and, before the chunk's fp16 pieces go to the staging buffer, its previous store must have read it
    auto staging_free = [&]() {
      if (a.stage_out && a.store_warp) ptx::mbar_wait(stg_empty(stg_i), stg_par ^ 1u);
    };
    auto step = [&](Pos& p, const float (&xc)[kChunk], const float (&yc)[kChunk], float (&xn)[kChunk],
                    float (&yn)[kChunk]) -> bool {
      if (p.ch == par && box_of(p) == 0) tile_begin();
      uint32_t v[kChunk];
      ptx::tmem_ld_32x32b_x8(tmem_base + (uint32_t(quarter * 32) << 16) + uint32_t(acc * kMaxBN + box_of(p) * a.BN + p.ch * kChunk), v);
      uint32_t v2[kChunk];
      if (a.sacc) ptx::tmem_ld_32x32b_x8(tmem_base + (uint32_t(quarter * 32) << 16) + uint32_t(acc * kMaxBN + 128 + box_of(p) * a.BN + p.ch * kChunk), v2);
      Pos q = p;
      advance(q);
      const bool nhave = q.vt < vt_end;
      if (nhave) epi_load(a, ec, q.tn, q.tm, q.ch, xn, yn);
      ptx::tmem_ld_wait();
      if (a.sacc) {
#pragma unroll
        for (int j = 0; j < kChunk; ++j) v[j] = __float_as_uint(__uint_as_float(v[j]) + __uint_as_float(v2[j]));
      }
      const uint32_t stg = a.stage_out ? stg_base + stg_i * (2u * kStageX) : 0u;
      if (p.ch == par) staging_free();
      set_step(p.vt);
      epi_update_store<HINTS>(a, ec, p.tn, p.tm, p.ch, v, xc, yc, stg);
      cur_tn = p.tn; cur_tm = p.tm;
      if (!same_box(p, q)) tile_done(q.vt != p.vt);
      p = q;
      return nhave;
    };
    if constexpr (X16 && YLDG) {
      {
        // state16 with y by plain loads: the loop is unrolled twice over two register buffers (current / next item's y and
        // position change roles), so that nothing is copied at the back edge; y of the NEXT box is on its way from DRAM to the
        // L2 while this box is updated (lanes 0 .. 15 touch the 16 lines this warp will read there).
        auto ldg_y = [&](const Pos& p, float (&dst)[kChunk]) {
          const int r = p.tm * kBM + ec.lane_r, i0 = p.tn * a.BN + p.ch * kChunk;
          uint32_t off = uint32_t(i0) * uint32_t(a.R) + uint32_t(r);
          if (r < a.R && i0 + kChunk <= a.n) {
            const float* yb = a.y + off;               // one wide multiply-add per address: base + j R
#pragma unroll
            for (int j = 0; j < kChunk; ++j) dst[j] = yb[uint32_t(j) * uint32_t(a.R)];
          } else {
#pragma unroll
            for (int j = 0; j < kChunk; ++j, off += uint32_t(a.R)) dst[j] = (r < a.R && i0 + j < a.n) ? a.y[off] : 0.f;
          }
        };
        auto item = [&](const Pos& p, const float (&yc)[kChunk], Pos& q, float (&yn)[kChunk]) -> bool {
          const bool first = p.ch == par;                    // this warp's first item of the box
          if (first && box_of(p) == 0) tile_begin();
          uint32_t v[kChunk], v2[kChunk];
          ptx::tmem_ld_32x32b_x8(tmem_base + (uint32_t(quarter * 32) << 16) + uint32_t(acc * kMaxBN + box_of(p) * a.BN + p.ch * kChunk), v);
          if (a.sacc) ptx::tmem_ld_32x32b_x8(tmem_base + (uint32_t(quarter * 32) << 16) + uint32_t(acc * kMaxBN + 128 + box_of(p) * a.BN + p.ch * kChunk), v2);
          q = p;
          advance(q);
          const bool nhave = q.vt < vt_end;
          if (nhave) ldg_y(q, yn);
          if (first) {
            Pos nb = p;
            next_box(nb);
            if (nb.vt < vt_end && lane < 2 * kChunk) {
              const int r = nb.tm * kBM + quarter * 32, i = nb.tn * a.BN + (par + (lane >> 3) * P) * kChunk + (lane & 7);
              if (r < a.R && i < min(a.n, (nb.tn + 1) * a.BN)) asm volatile("prefetch.global.L2 [%0];" ::"l"(a.y + size_t(i) * a.R + r));
            }
            ptx::mbar_wait(stg_in(stg_i), stg_par);          // the box's own (x_hi, x_lo) has arrived
          }
          const uint32_t stg = stg_base + stg_i * (2u * kStageX);
          ptx::tmem_ld_wait();
          if (a.sacc) {
#pragma unroll
            for (int j = 0; j < kChunk; ++j) v[j] = __float_as_uint(__uint_as_float(v[j]) + __uint_as_float(v2[j]));
          }
          if (first) set_step(p.vt);                         // the ramp constant changes between boxes only
          if constexpr (PAIR) {                              // pairs: one instance, one c1 for all rows (dense and block path)
            epi_update_x16<HINTS, false>(a, ec, p.tn, p.tm, p.ch, v, yc, stg);
          } else if constexpr (XW) {                         // hybrid block path: per-row c1, fp32 x written next to the pair
            epi_update_x16<HINTS, true, true>(a, ec, p.tn, p.tm, p.ch, v, yc, stg);
          } else {
            if (a.c1_per_row) epi_update_x16<HINTS, true>(a, ec, p.tn, p.tm, p.ch, v, yc, stg);
            else epi_update_x16<HINTS, false>(a, ec, p.tn, p.tm, p.ch, v, yc, stg);
          }
          if (!same_box(p, q)) tile_done(q.vt != p.vt);
          return nhave;
        };
        Pos pa = first_pos(), pb = pa;
        if (pa.vt < vt_end) {
          float ya[kChunk], yb[kChunk];
          ldg_y(pa, ya);
          while (true) {
            if (!item(pa, ya, pb, yb)) break;
            if (!item(pb, yb, pa, ya)) break;
          }
        }
      }
    }
    else if constexpr (RING) {
      // State through TMA: every warp owns two 2 KB slots (x and y of one work item: a box of 8 spins x 32 replicas
      // each).  The item two ahead is requested as soon as the current item's values are in registers, so the loads
      // need no registers, no address arithmetic and no LSU slots; out-of-range rows / replicas arrive as zeros.
      // (state16: y only -- x is the tile's own fp16 pair in the staging buffer)
      constexpr uint32_t kSlotBytes = X16 ? uint32_t(kRingSlot) : 2u * kRingSlot;
      const uint32_t ring_w = stg_base + a.stg_bufs * (2u * kStageX) + uint32_t(ew) * (2u * kSlotBytes);
      const uint32_t rbar0 = ring_bar(2 * ew);
      auto issue = [&](const Pos& p, int slot) {
        if (ptx::elect_one()) {
          const int ch = p.ch;
          const int tn = p.tn, tm = p.tm;
          const uint32_t dst = ring_w + uint32_t(slot) * kSlotBytes;
          ptx::mbar_arrive_expect_tx(rbar0 + 8u * slot, kSlotBytes);
          if constexpr (X16) {
            if constexpr (HINTS) ptx::tma_load_2d_hint(dst, &tm_sy, rbar0 + 8u * slot, tm * kBM + quarter * 32, tn * a.BN + ch * kChunk, a.pol_stream);
            else ptx::tma_load_2d(dst, &tm_sy, rbar0 + 8u * slot, tm * kBM + quarter * 32, tn * a.BN + ch * kChunk);
          } else if constexpr (HINTS) {
            ptx::tma_load_2d_hint(dst, &tm_sx, rbar0 + 8u * slot, tm * kBM + quarter * 32, tn * a.BN + ch * kChunk, a.pol_keep);
            ptx::tma_load_2d_hint(dst + kRingSlot, &tm_sy, rbar0 + 8u * slot, tm * kBM + quarter * 32, tn * a.BN + ch * kChunk, a.pol_stream);
          } else {
            ptx::tma_load_2d(dst, &tm_sx, rbar0 + 8u * slot, tm * kBM + quarter * 32, tn * a.BN + ch * kChunk);
            ptx::tma_load_2d(dst + kRingSlot, &tm_sy, rbar0 + 8u * slot, tm * kBM + quarter * 32, tn * a.BN + ch * kChunk);
          }
        }
        __syncwarp();
      };
      Pos p0 = first_pos(), p1 = p0, p2 = p0;
      if (p0.vt < vt_end) {
        issue(p0, 0);
        advance(p1);
        if (p1.vt < vt_end) issue(p1, 1);
        p2 = p1;
        if (p1.vt < vt_end) advance(p2);
      }
      for (uint32_t k = 0; p0.vt < vt_end; ++k) {
        const int slot = int(k & 1u);
        if (p0.ch == par && box_of(p0) == 0) tile_begin();
        uint32_t v[kChunk];
        ptx::tmem_ld_32x32b_x8(tmem_base + (uint32_t(quarter * 32) << 16) + uint32_t(acc * kMaxBN + box_of(p0) * a.BN + p0.ch * kChunk), v);
        uint32_t v2[kChunk];
        if (a.sacc) ptx::tmem_ld_32x32b_x8(tmem_base + (uint32_t(quarter * 32) << 16) + uint32_t(acc * kMaxBN + 128 + box_of(p0) * a.BN + p0.ch * kChunk), v2);
        float xv[kChunk], yv[kChunk];
        ptx::mbar_wait(rbar0 + 8u * slot, (k >> 1) & 1u);
        const uint32_t src = ring_w + uint32_t(slot) * kSlotBytes + uint32_t(lane) * 4u;
#pragma unroll
        for (int j = 0; j < kChunk; ++j) {
          if constexpr (X16) {
            asm volatile("ld.shared.f32 %0, [%1];" : "=f"(yv[j]) : "r"(src + uint32_t(j) * 128u));
          } else {
            asm volatile("ld.shared.f32 %0, [%1];" : "=f"(xv[j]) : "r"(src + uint32_t(j) * 128u));
            asm volatile("ld.shared.f32 %0, [%1];" : "=f"(yv[j]) : "r"(src + kRingSlot + uint32_t(j) * 128u));
          }
        }
        const uint32_t stg = a.stage_out ? stg_base + stg_i * (2u * kStageX) : 0u;
        if constexpr (X16) {
          if (p0.ch == par) ptx::mbar_wait(stg_in(stg_i), stg_par);      // the tile's own (x_hi, x_lo) has arrived
          ptx::tmem_ld_wait();
          if (a.sacc) {
#pragma unroll
            for (int j = 0; j < kChunk; ++j) v[j] = __float_as_uint(__uint_as_float(v[j]) + __uint_as_float(v2[j]));
          }
          set_step(p0.vt);
          if (a.c1_per_row) epi_update_x16<HINTS, true>(a, ec, p0.tn, p0.tm, p0.ch, v, yv, stg);
          else epi_update_x16<HINTS, false>(a, ec, p0.tn, p0.tm, p0.ch, v, yv, stg);
        } else {
          ptx::tmem_ld_wait();
          if (a.sacc) {
#pragma unroll
            for (int j = 0; j < kChunk; ++j) v[j] = __float_as_uint(__uint_as_float(v[j]) + __uint_as_float(v2[j]));
          }
          if (p0.ch == par) staging_free();
          set_step(p0.vt);
          epi_update_store<HINTS>(a, ec, p0.tn, p0.tm, p0.ch, v, xv, yv, stg);
        }
        cur_tn = p0.tn; cur_tm = p0.tm;
        // The slot is refilled only now: the update above has CONSUMED the values read from it, so those shared-memory
        // reads have completed.  (Requested right after the ld.shared instructions were issued, the TMA write could land
        // before the last of them had read the slot: observed as rows 5..7 of a work item carrying the next item's y.)
        __syncwarp();
        if (p1.vt < vt_end && p2.vt < vt_end) issue(p2, slot);
        if (!same_box(p0, p1)) tile_done(p1.vt != p0.vt);
        p0 = p1; p1 = p2;
        if (p2.vt < vt_end) advance(p2);
      }
      if (a.stage_out && !a.store_warp && ew == 0 && lane == 0) ptx::tma_store_wait_read_all();   // smem must outlive the bulk reads
    } else {
    Pos p = first_pos();
    if (p.vt < vt_end) {
      float xa[kChunk], ya[kChunk], xb[kChunk], yb[kChunk];
      epi_load(a, ec, p.tn, p.tm, p.ch, xa, ya);
      while (true) {
        if (!step(p, xa, ya, xb, yb)) break;
        if (!step(p, xb, yb, xa, ya)) break;
      }
      if (a.stage_out && !a.store_warp && ew == 0 && lane == 0) ptx::tma_store_wait_read_all();
    }
    }
  }

  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc(tmem_base, kTmemCols);
  }
}

// x [n][R] fp32 -> split copies [R][n_k] fp16 (transpose through shared memory, 32 x 32 tiles).
// mode 0: plain split (fp32-x kernels); 1: dSB sign copies; 2: canonical pair (state16).
__global__ void __launch_bounds__(256) split_x_kernel(int32_t n, int32_t R, int32_t n_k, int32_t mode, const float* __restrict__ x,
                                                      __half* __restrict__ xh, __half* __restrict__ xl) {
  __shared__ float t[32][33];
  const int i0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  for (int j = ty; j < 32; j += 8) {
    const int i = i0 + j, r = r0 + tx;
    t[j][tx] = (i < n && r < R) ? x[size_t(i) * R + r] : 0.f;
  }
  __syncthreads();
  for (int j = ty; j < 32; j += 8) {
    const int r = r0 + j, i = i0 + tx;
    if (r < R && i < n_k) {
      __half h, l;
      if (mode == 2) split_half_canonical(t[tx][j], h, l);
      else if (mode == 1 && i < n) split_sign(t[tx][j], h, l);
      else split_half(t[tx][j], h, l);
      xh[size_t(r) * n_k + i] = h;
      xl[size_t(r) * n_k + i] = l;
    }
  }
}

// state16, after the last step of a call: x[i][r] = (x_hi[r][i] + x_lo[r][i]) 2^-15 (exact in fp32).
__global__ void __launch_bounds__(256) merge_x_kernel(int32_t n, int32_t R, int32_t n_k, const __half* __restrict__ xh,
                                                      const __half* __restrict__ xl, float* __restrict__ x) {
  __shared__ float t[32][33];
  const int i0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  for (int j = ty; j < 32; j += 8) {
    const int r = r0 + j, i = i0 + tx;
    t[j][tx] = (r < R && i < n) ? (__half2float(xh[size_t(r) * n_k + i]) + __half2float(xl[size_t(r) * n_k + i])) * (1.0f / kXScale) : 0.f;
  }
  __syncthreads();
  for (int j = ty; j < 32; j += 8) {
    const int i = i0 + j, r = r0 + tx;
    if (i < n && r < R) x[size_t(i) * R + r] = t[tx][j];
  }
}

// tile_skip lists: flag[tn][kb] = 1 iff some row of N tile tn has a non-zero in k-block kb (one warp per row).
__global__ void __launch_bounds__(256) kb_flag_kernel(int32_t n, const int32_t* __restrict__ row_ptr, const int32_t* __restrict__ col,
                                                      int32_t BN, int32_t n_kblocks, int32_t* __restrict__ flag) {
  const int32_t a = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (a >= n) return;
  const int lane = threadIdx.x & 31;
  int32_t* f = flag + size_t(a / BN) * n_kblocks;
  for (int32_t e = row_ptr[a] + lane; e < row_ptr[a + 1]; e += 32) {
    f[col[e] / kBK] = 1;
    // tile rows == k-blocks: keep the lists symmetric even if the CSR is not (the fused steps' write-after-read
    // ordering on the fp16 copies relies on "tn lists kb  <=>  kb lists tn"; an extra zero tile is harmless)
    if (BN == kBK) flag[size_t(col[e] / kBK) * n_kblocks + a / kBK] = 1;
  }
}

// One CTA per N tile: ascending list of flagged k-blocks (at least one entry, so that every tile produces an accumulator).
__global__ void __launch_bounds__(32) kb_list_kernel(int32_t n_kblocks, int32_t BN, const int32_t* __restrict__ flag, int32_t* __restrict__ kb_cnt,
                                                     int32_t* __restrict__ kb_idx) {
  const int tn = blockIdx.x, lane = threadIdx.x;
  const int32_t* f = flag + size_t(tn) * n_kblocks;
  int32_t* out = kb_idx + size_t(tn) * n_kblocks;
  int32_t cnt = 0;
  for (int32_t base = 0; base < n_kblocks; base += 32) {
    const int32_t kb = base + lane;
    const bool on = kb < n_kblocks && f[kb] != 0;
    const uint32_t m = __ballot_sync(0xffffffffu, on);
    if (on) out[cnt + __popc(m & ((1u << lane) - 1u))] = kb;
    cnt += __popc(m);
  }
  if (lane == 0) {
    // an empty tile row lists the k-block of its own first row: for BN == kBK that is its diagonal block, which keeps the
    // lists symmetric (fused steps: "tn lists kb <=> kb lists tn") and is ordered against itself by the owning CTA
    if (cnt == 0) { out[0] = min(n_kblocks - 1, int32_t((int64_t(tn) * BN) / kBK)); cnt = 1; }
    kb_cnt[tn] = cnt;
  }
}

// Paired tiles: ascending union of the k-block flags of boxes 2q and 2q + 1 (one CTA per pair; never empty: an empty union
// lists the left box's own k-block, like kb_list_kernel).
__global__ void __launch_bounds__(32) pair_list_kernel(int32_t n_kblocks, const int32_t* __restrict__ flag, int32_t* __restrict__ pk_cnt,
                                                       int32_t* __restrict__ pk_idx) {
  const int q = blockIdx.x, lane = threadIdx.x;
  const int32_t* f0 = flag + size_t(2 * q) * n_kblocks;
  const int32_t* f1 = f0 + n_kblocks;
  int32_t* out = pk_idx + size_t(q) * n_kblocks;
  int32_t cnt = 0;
  for (int32_t base = 0; base < n_kblocks; base += 32) {
    const int32_t kb = base + lane;
    const bool on = kb < n_kblocks && (f0[kb] | f1[kb]) != 0;
    const uint32_t m = __ballot_sync(0xffffffffu, on);
    if (on) out[cnt + __popc(m & ((1u << lane) - 1u))] = kb;
    cnt += __popc(m);
  }
  if (lane == 0) {
    if (cnt == 0) { out[0] = min(n_kblocks - 1, 2 * q); cnt = 1; }
    pk_cnt[q] = cnt;
  }
}

// Block path pairs: merge of the ascending k-block lists of boxes 2q and 2q + 1.  FILL = false: union sizes; FILL = true: the
// union (pk_kb) with the tile of each box in the block arrays, `zero_tile` for a box that does not list the k-block.
template <bool FILL>
__global__ void __launch_bounds__(128) pair_merge_kernel(int32_t P, int32_t n_kblocks, const int32_t* __restrict__ kb_cnt,
                                                         const int32_t* __restrict__ kb_idx, const int32_t* __restrict__ blk_ptr,
                                                         int32_t zero_tile, int32_t* __restrict__ pk_ptr, int32_t* __restrict__ pk_kb,
                                                         int32_t* __restrict__ pk_l, int32_t* __restrict__ pk_r) {
  const int32_t q = blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= P) return;
  const int32_t *la = kb_idx + size_t(2 * q) * n_kblocks, *lb = la + n_kblocks;
  const int32_t na = kb_cnt[2 * q], nb = kb_cnt[2 * q + 1], ba = blk_ptr[2 * q], bb = blk_ptr[2 * q + 1];
  int32_t i = 0, j = 0, out = FILL ? pk_ptr[q] : 0;
  while (i < na || j < nb) {
    const int32_t ka = i < na ? la[i] : INT32_MAX, kb = j < nb ? lb[j] : INT32_MAX, k = min(ka, kb);
    if (FILL) {
      pk_kb[out] = k;
      pk_l[out] = ka == k ? ba + i : zero_tile;
      pk_r[out] = kb == k ? bb + j : zero_tile;
    }
    ++out;
    if (ka == k) ++i;
    if (kb == k) ++j;
  }
  if (!FILL) pk_ptr[q] = out;
}

// ------------------------------------------------------------------- block-compressed J (64 x 64 fp16 tiles) from a CSR
// max |J| over all entries (order-independent: integer max of the absolute value's bit pattern)
__global__ void __launch_bounds__(256) absmax_kernel(int64_t nnz, const float* __restrict__ jval, uint32_t* __restrict__ out) {
  uint32_t m = 0;
  for (int64_t e = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; e < nnz; e += int64_t(gridDim.x) * blockDim.x)
    m = max(m, __float_as_uint(fabsf(jval[e])));
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0 && m) atomicMax(out, m);
}

// scale[0] = 2^e with max|J| 2^e in [2^13, 2^14) (1 for an all-zero J or when `unit` is set: integer weights are used as
// they are); c1row[i] = c1[instance of i] 2^-15 / scale[0]  (exact power-of-two factors)
__global__ void __launch_bounds__(256) block_scale_kernel(int32_t n, int32_t n_inst, const int32_t* __restrict__ inst_ptr,
                                                          const float* __restrict__ c1, const uint32_t* __restrict__ amax,
                                                          int32_t unit, float* __restrict__ scale, float* __restrict__ c1row,
                                                          float* __restrict__ c1plain) {
  const float mx = __uint_as_float(*amax);
  const float sc = (unit || !(mx > 0.f)) ? 1.0f : ldexpf(1.0f, 13 - ilogbf(mx));
  const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) scale[0] = sc;
  if (i >= n) return;
  int inst = 0;
  if (n_inst > 1) {
    int lo = 0, hi = n_inst;
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (inst_ptr[mid] <= i) lo = mid; else hi = mid;
    }
    inst = lo;
  }
  c1row[i] = c1[inst] * (1.0f / kXScale) * (1.0f / sc);
  c1plain[i] = c1[inst];
}

// Tile occupancy: cnt[tn][kb] = number of entries of tile (tn, kb)  (one warp per row; integer atomics).
__global__ void __launch_bounds__(256) tile_count_kernel(int32_t n, const int32_t* __restrict__ row_ptr, const int32_t* __restrict__ col,
                                                         int32_t n_kblocks, int32_t* __restrict__ cnt) {
  const int32_t a = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (a >= n) return;
  const int lane = threadIdx.x & 31;
  int32_t* f = cnt + size_t(a / kBK) * n_kblocks;
  for (int32_t e = row_ptr[a] + lane; e < row_ptr[a + 1]; e += 32) atomicAdd(f + col[e] / kBK, 1);
}

// One CTA per tile row: ascending list of the k-blocks with at least `thr` entries (at least one list entry per tile row).
__global__ void __launch_bounds__(32) tile_list_kernel(int32_t n_kblocks, const int32_t* __restrict__ cnt, int32_t thr,
                                                       int32_t* __restrict__ kb_cnt, int32_t* __restrict__ kb_idx) {
  const int tn = blockIdx.x, lane = threadIdx.x;
  const int32_t* f = cnt + size_t(tn) * n_kblocks;
  int32_t* out = kb_idx + size_t(tn) * n_kblocks;
  int32_t c = 0;
  for (int32_t base = 0; base < n_kblocks; base += 32) {
    const int32_t kb = base + lane;
    const bool on = kb < n_kblocks && f[kb] >= thr;
    const uint32_t m = __ballot_sync(0xffffffffu, on);
    if (on) out[c + __popc(m & ((1u << lane) - 1u))] = kb;
    c += __popc(m);
  }
  if (lane == 0) {
    if (c == 0) { out[0] = tn < n_kblocks ? tn : 0; c = 1; }   // the diagonal tile (possibly empty) keeps the pipeline uniform
    kb_cnt[tn] = c;
  }
}

__device__ __forceinline__ bool tile_listed(const int32_t* list, int32_t cnt, int32_t kb, int& pos) {
  int lo = 0, hi = cnt;                                    // list[lo] <= kb < list[hi]
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (list[mid] <= kb) lo = mid; else hi = mid;
  }
  pos = lo;
  return list[lo] == kb;
}

// Remainder = entries whose tile is not listed (sparse long-range edges).  Pass 0 counts them per row, pass 1 writes
// them (ascending column order is kept: ballot compaction over 32 entries at a time).
template <int FILL>
__global__ void __launch_bounds__(256) remainder_kernel(int32_t n, const int32_t* __restrict__ row_ptr, const int32_t* __restrict__ col,
                                                        const float* __restrict__ jval, int32_t n_kblocks,
                                                        const int32_t* __restrict__ kb_cnt, const int32_t* __restrict__ kb_idx,
                                                        int32_t* __restrict__ rem_ptr, int32_t* __restrict__ rem_col,
                                                        float* __restrict__ rem_val) {
  const int32_t a = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (a >= n) return;
  const int lane = threadIdx.x & 31;
  const int32_t tn = a / kBK;
  const int32_t* list = kb_idx + size_t(tn) * n_kblocks;
  const int32_t cnt = kb_cnt[tn];
  int32_t outp = FILL ? rem_ptr[a] : 0;
  for (int32_t e0 = row_ptr[a]; e0 < row_ptr[a + 1]; e0 += 32) {
    const int32_t e = e0 + lane;
    bool rem = false;
    int pos;
    if (e < row_ptr[a + 1]) rem = !tile_listed(list, cnt, col[e] / kBK, pos);
    const uint32_t m = __ballot_sync(0xffffffffu, rem);
    if (FILL && rem) {
      const int32_t o = outp + __popc(m & ((1u << lane) - 1u));
      rem_col[o] = col[e];
      rem_val[o] = jval[e];
    }
    outp += __popc(m);
  }
  if (!FILL && lane == 0) rem_ptr[a] = outp;
}

// y += c1[instance] * sum over the row's remainder entries of J x_old  -- one warp per row, lanes across replicas
// (float4), rows without remainder entries cost one row_ptr read.  Runs BEFORE the tile step of the same bSB step, on the
// fp32 x that step will then update in place; the tile step's fma(c1, F_tiles, fma(-c2, x, y)) completes the sum.
__device__ __forceinline__ float4 sgn4(float4 v) {
  return make_float4(v.x >= 0.f ? 1.f : -1.f, v.y >= 0.f ? 1.f : -1.f, v.z >= 0.f ? 1.f : -1.f, v.w >= 0.f ? 1.f : -1.f);
}
template <bool dsb>
__global__ void __launch_bounds__(256) remainder_step_kernel(int32_t n, int32_t R, const int32_t* __restrict__ rem_ptr,
                                                             const int32_t* __restrict__ rem_col, const float* __restrict__ rem_val,
                                                             const float* __restrict__ c1row_plain, const float* __restrict__ x,
                                                             float* __restrict__ y) {
  const int32_t a = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (a >= n) return;
  const int32_t e0 = rem_ptr[a], e1 = rem_ptr[a + 1];
  if (e0 == e1) return;
  const int lane = threadIdx.x & 31;
  const float c1 = c1row_plain[a];
  for (int32_t r = lane * 4; r < R; r += 128) {
    if (r + 4 <= R && (R & 3) == 0) {
      float4 F = make_float4(0.f, 0.f, 0.f, 0.f);
      int32_t e = e0;
      for (; e + 4 <= e1; e += 4) {                      // four independent gathers in flight, summed in ascending order
        float v[4];
        float4 xv[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          v[q] = __ldg(rem_val + e + q);
          xv[q] = *reinterpret_cast<const float4*>(x + size_t(__ldg(rem_col + e + q)) * R + r);
          if (dsb) xv[q] = sgn4(xv[q]);
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          F.x = fmaf(v[q], xv[q].x, F.x); F.y = fmaf(v[q], xv[q].y, F.y); F.z = fmaf(v[q], xv[q].z, F.z); F.w = fmaf(v[q], xv[q].w, F.w);
        }
      }
      for (; e < e1; ++e) {
        const float v = __ldg(rem_val + e);
        float4 xv = *reinterpret_cast<const float4*>(x + size_t(__ldg(rem_col + e)) * R + r);
        if (dsb) xv = sgn4(xv);
        F.x = fmaf(v, xv.x, F.x); F.y = fmaf(v, xv.y, F.y); F.z = fmaf(v, xv.z, F.z); F.w = fmaf(v, xv.w, F.w);
      }
      float4* py = reinterpret_cast<float4*>(y + size_t(a) * R + r);
      float4 yv = *py;
      yv.x = fmaf(c1, F.x, yv.x); yv.y = fmaf(c1, F.y, yv.y); yv.z = fmaf(c1, F.z, yv.z); yv.w = fmaf(c1, F.w, yv.w);
      *py = yv;
    } else {
      for (int32_t rr = r; rr < min(r + 4, R); ++rr) {
        float F = 0.f;
        for (int32_t e = e0; e < e1; ++e) {
          const float xj = x[size_t(__ldg(rem_col + e)) * R + rr];
          F = fmaf(__ldg(rem_val + e), dsb ? (xj >= 0.f ? 1.f : -1.f) : xj, F);
        }
        y[size_t(a) * R + rr] = fmaf(c1, F, y[size_t(a) * R + rr]);
      }
    }
  }
}

// One warp per row: scatter the row's entries into their tiles.  Tile (tn, kb) is block blk_ptr[tn] + (rank of kb in the
// ascending list kb_idx[tn][0 .. kb_cnt[tn])).  J_hi = fp16(J scale), J_lo = fp16(J scale - J_hi).
__global__ void __launch_bounds__(256) block_fill_kernel(int32_t n, const int32_t* __restrict__ row_ptr, const int32_t* __restrict__ col,
                                                         const float* __restrict__ jval, int32_t n_kblocks,
                                                         const int32_t* __restrict__ kb_cnt, const int32_t* __restrict__ kb_idx,
                                                         const int32_t* __restrict__ blk_ptr, const float* __restrict__ scale,
                                                         __half* __restrict__ jh, __half* __restrict__ jl) {
  const int32_t a = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (a >= n) return;
  const int lane = threadIdx.x & 31;
  const int32_t tn = a / kBK;
  const int32_t* list = kb_idx + size_t(tn) * n_kblocks;
  const int32_t cnt = kb_cnt[tn], base = blk_ptr[tn];
  const float sc = scale[0];
  for (int32_t e = row_ptr[a] + lane; e < row_ptr[a + 1]; e += 32) {
    const int32_t c = col[e], kb = c / kBK;
    int lo;
    if (!tile_listed(list, cnt, kb, lo)) continue;         // remainder entry (handled by remainder_step_kernel)
    const size_t idx = (size_t(base + lo) * kBK + size_t(a % kBK)) * kBK + size_t(c % kBK);
    const float vs = jval[e] * sc;
    const __half h = __float2half_rn(vs);
    jh[idx] = h;
    if (jl) jl[idx] = __float2half_rn(vs - __half2float(h));
  }
}

// ------------------------------------------------------------------------------------------- host side
// Kernel variant of a launch: RING (fp32 state through the TMA ring) x HINTS (L2 eviction priorities) x X16 (state16).
typedef void (*StepKernel)(const CUtensorMap, const CUtensorMap, const CUtensorMap, const CUtensorMap, const CUtensorMap,
                           const CUtensorMap, const CUtensorMap, const CUtensorMap, const DenseArgs);
StepKernel step_kernel_of(const DenseArgs& a) {
  const bool hints = a.pol_keep != ptx::kEvictNormal;
  if (a.x16) {
    if (a.pair_lines) {
      if (a.yldg) return hints ? dense_step_kernel<true, true, true, true, true, false> : dense_step_kernel<true, false, true, true, true, false>;
      return hints ? dense_step_kernel<true, true, true, true, false, false> : dense_step_kernel<true, false, true, true, false, false>;
    }
    if (a.yldg && a.xw32) return hints ? dense_step_kernel<true, true, true, false, true, true> : dense_step_kernel<true, false, true, false, true, true>;
    if (a.yldg) return hints ? dense_step_kernel<true, true, true, false, true, false> : dense_step_kernel<true, false, true, false, true, false>;
    return hints ? dense_step_kernel<true, true, true, false, false, false> : dense_step_kernel<true, false, true, false, false, false>;
  }
  if (a.ring) return hints ? dense_step_kernel<true, true, false, false, false, false> : dense_step_kernel<true, false, false, false, false, false>;
  return hints ? dense_step_kernel<false, true, false, false, false, false> : dense_step_kernel<false, false, false, false, false, false>;
}

// One launch of the step kernel.  Per-step launches carry the programmatic-stream-serialization attribute (see the
// kernel: griddepcontrol.wait); a fused launch (its CTAs wait for each other's tiles) is a COOPERATIVE launch, so the
// driver guarantees that all of its CTAs are co-resident whatever else runs on the device.
qhap_status launch_step(int grid, cudaStream_t stream, const CUtensorMap& tj, const CUtensorMap& tjl, const CUtensorMap& th,
                        const CUtensorMap& tl, const CUtensorMap& toh, const CUtensorMap& tol, const CUtensorMap& tsx,
                        const CUtensorMap& tsy, const DenseArgs& a) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(unsigned(grid));
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = kSmemBytes;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  if (a.fused) {
    attr[0].id = cudaLaunchAttributeCooperative;
    attr[0].val.cooperative = 1;
  } else {
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
  }
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  StepKernel kernel = step_kernel_of(a);
  // per device and cheap: set on every call (a process may drive several devices)
  QHAP_CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, int(kSmemBytes)));
  QHAP_CUDA_TRY(cudaLaunchKernelEx(&cfg, kernel, tj, tjl, th, tl, toh, tol, tsx, tsy, a));
  QHAP_LAUNCH_CHECK();
  return QHAP_OK;
}

// Shared-memory split between operand stages and the staging buffers of the fp16 copies: the operand feed (every tile
// re-reads ~6 k-blocks of x_hi, x_lo: 240 KB per tile at cfg1 against 160 KB of state) runs on the bytes in flight, so a
// single staging buffer is used whenever that buys another stage (fp32-x kernels; cfg1/cfg2: 2 -> 3 stages).  state16 always
// has two buffers (tile t + 1's own pair is loaded while tile t is updated) and a ring of half the size.
void choose_staging(DenseArgs& a, int stage_bytes, const qhap_bsb_tuning& t) {
  const int ring_bytes = a.x16 ? (a.yldg ? 0 : kRingBytes16) : (a.ring ? kRingBytes : 0);
  auto stages = [&](int bufs) {
    return std::min(kMaxStages, (kSmemBudget - (a.stage_out ? bufs * 2 * kStageX : 0) - ring_bytes) / stage_bytes);
  };
  int bufs = (t.dense_stg_bufs == 1 || t.dense_stg_bufs == 2) ? t.dense_stg_bufs : ((a.stage_out && stages(1) > stages(2) && stages(2) < 3) ? 1 : 2);
  if (a.x16 && t.dense_stg_bufs != 1) bufs = 2;
  a.stg_bufs = uint32_t(bufs);
  a.n_stages = stages(bufs);
  a.store_warp = (bufs == 1 || a.x16) ? 1u : 0u;        // launch_fused sets it too
}

// The arrays that are re-used (x in fp32 and the four fp16 copies: 12 B per (spin, replica); state16: the copies only, 8 B)
// get the evict_last priority and y evict_first when they fit the L2 with room for the y stream and the J tiles.
void set_l2_policies(DenseArgs& a, const qhap_bsb_tuning& t) {
  // state16: the copies stay in the L2 without help and the hints cost 1-9 % (cfg1 24.2 against 24.8, cfg2 28.0 against 30.7 us
  // per step), so automatic = off there
  const bool keep = t.l2_hints == 0 ? (!a.x16 && 12.0 * double(a.n) * double(a.R) <= 104e6) : t.l2_hints == 1;
  // q/16 of the keep set's lines are evict_last, the rest evict_first (createpolicy.fractional.L2::evict_last.L2::evict_first
  // with fraction q/16 encodes as (0x150 | (q - 1)) << 52; q = 16 is kEvictLast for every line)
  const int q = (t.l2_keep_16ths >= 1 && t.l2_keep_16ths <= 16) ? t.l2_keep_16ths : 16;
  a.pol_keep = keep ? (q == 16 ? ptx::kEvictLast : (uint64_t(0x150u | uint32_t(q - 1)) << 52)) : ptx::kEvictNormal;
  a.pol_stream = keep ? ptx::kEvictFirst : ptx::kEvictNormal;
  // (measured with state16: the meeting costs cfg1 26.6 against 25.6 us per step, so it stays with the fp32-x kernels)
  a.epi_sync = t.dense_epi_sync == 0 ? ((keep && !a.x16) ? 1u : 0u) : (t.dense_epi_sync == 1 ? 1u : 0u);
}

// Grid of a fused launch, or 0 = one launch per step.  Fused launches need: TMA-stored copies and tile rows == k-blocks
// (BN == kBK), k-block lists, at least two tiles per CTA and step (state prefetch distance: grid <= tiles / 2), and ALL CTAs
// co-resident -- the launch is cooperative, and the grid is capped by what the occupancy API says fits this device.
// Worth it while a CTA has few tiles per step (launch gap, pipeline fill and drain per step); with ~50 tiles per CTA and
// step (cfg3) the boundary is amortised and lock-step launches keep the L2 reuse between neighbouring CTAs.
int fused_grid(const DenseArgs& a, const qhap_bsb_params& p, const qhap_bsb_tuning& t) {
  const int64_t n_tiles = int64_t(a.n_tiles_m) * a.n_tiles_n;          // boxes
  if (t.step_launch != 0 || !a.stage_out || a.BN != kBK || a.kb_cnt == nullptr || p.steps_run < 2) return 0;
  int per_sm = 0, coop = 0, dev = 0;
  StepKernel kernel = step_kernel_of(a);
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) != cudaSuccess || !coop ||
      cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, int(kSmemBytes)) != cudaSuccess ||
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kThreads, kSmemBytes) != cudaSuccess || per_sm < 1) {
    (void)cudaGetLastError();
    return 0;
  }
  const int64_t grid = std::min<int64_t>(int64_t(sm_count()) * per_sm, n_tiles / 2);
  if (grid < 1 || ceil_div(n_tiles, grid) > 16) return 0;
  return int(grid);
}

void pair_plan_loads(int32_t n_tiles_n, int32_t n_tiles_m, int grid, int32_t P, int64_t& mx, int64_t& mn);

// All steps of the call in as few launches as the 32-bit virtual tile index allows (one, at every BASELINE size).
// tm_h / tm_l: the two buffers of split copies; buffer `cur` holds the current x.  Returns the buffer that holds x after.
qhap_status launch_fused(int grid, cudaStream_t stream, const CUtensorMap& tj, const CUtensorMap& tjl, const CUtensorMap (&tm_h)[2],
                         const CUtensorMap (&tm_l)[2], const CUtensorMap& tsx, const CUtensorMap& tsy, DenseArgs a,
                         const qhap_bsb_params& p, uint32_t* done, int& cur) {
  const int64_t n_tiles = int64_t(a.n_tiles_m) * a.n_tiles_n;          // boxes (done[] has one counter per box)
  a.fused = 1;
  a.store_warp = 1;
  a.tile_stride = int32_t(ceil_div(int64_t(a.n_slots), grid) * grid);
  a.fence_every = uint32_t(std::max<int64_t>(1, int64_t(a.n_slots) / grid - 1));
  {
    int64_t mx, mn;                               // boxes per CTA and step
    pair_plan_loads(a.n_tiles_n, a.n_tiles_m, grid, a.pair_lines, mx, mn);
    a.early_reload = (a.x16 && mn >= 3) ? 1 : 0;
  }
  a.steps_total = p.steps_total; a.dt = p.dt; a.a0 = p.a0;
  a.c3 = float(p.dt * p.a0);
  a.c2 = 0.f;
  a.done = done;
  a.xh_out = nullptr; a.xl_out = nullptr;          // fused launches store through the tensor maps only (stage_out)
  const int32_t max_steps = int32_t(std::max<int64_t>(1, (int64_t(1) << 30) / a.tile_stride));
  for (int32_t k = p.step_begin; k < p.step_begin + p.steps_run;) {
    a.n_steps = std::min(max_steps, p.step_begin + p.steps_run - k);
    a.k0 = k;
    QHAP_CUDA_TRY(cudaMemsetAsync(done, 0, sizeof(uint32_t) * size_t(n_tiles), stream));
    QHAP_TRY(launch_step(grid, stream, tj, tjl, tm_h[cur], tm_l[cur], tm_h[cur ^ 1], tm_l[cur ^ 1], tsx, tsy, a));
    cur ^= (a.n_steps & 1);
    k += a.n_steps;
  }
  return QHAP_OK;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      p = nullptr;
    return reinterpret_cast<EncodeTiledFn>(p);
  }();
  return fn;
}

// 2-D fp16 tensor [outer][inner] with row pitch `pitch` elements; box {64, box_outer}; 128-byte swizzle; OOB -> 0.
qhap_status make_map(CUtensorMap* m, const void* base, uint64_t inner, uint64_t outer, uint64_t pitch, uint32_t box_outer) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) {
    set_error("cuTensorMapEncodeTiled not available from the driver");
    return QHAP_ERR_CUDA;
  }
  const cuuint64_t dims[2] = {inner, outer};
  const cuuint64_t strides[1] = {pitch * 2};
  const cuuint32_t box[2] = {uint32_t(kBK), box_outer};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    set_error("cuTensorMapEncodeTiled failed with CUresult %d (base %p inner %llu outer %llu pitch %llu)", int(r), base,
              (unsigned long long)inner, (unsigned long long)outer, (unsigned long long)pitch);
    return QHAP_ERR_CUDA;
  }
  return QHAP_OK;
}

// fp32 state [n][R] (replica index contiguous): box = one work item of a warp, 32 replicas x kChunk spins, no swizzle, OOB -> 0.
qhap_status make_state_map(CUtensorMap* m, const float* base, int32_t n, int32_t R) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) {
    set_error("cuTensorMapEncodeTiled not available from the driver");
    return QHAP_ERR_CUDA;
  }
  const cuuint64_t dims[2] = {cuuint64_t(R), cuuint64_t(n)};
  const cuuint64_t strides[1] = {cuuint64_t(R) * 4};
  const cuuint32_t box[2] = {32, uint32_t(kChunk)};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(base), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    set_error("cuTensorMapEncodeTiled (state) failed with CUresult %d", int(r));
    return QHAP_ERR_CUDA;
  }
  return QHAP_OK;
}

// state ring usable: tile one box wide, row pitch a multiple of 16 bytes, 16-byte aligned bases -- and worth its 64 KB:
// with a single replica tile (R <= 128) every J tile comes from DRAM exactly once and the third operand stage that the
// ring would displace matters more (measured on cfg4: 146.8 us without the ring, 160.1 us with it)
bool ring_ok(int32_t BN, int32_t R, const float* x, const float* y) {
  return BN == kBK && R % 4 == 0 && R > kBM && ((reinterpret_cast<uintptr_t>(x) | reinterpret_cast<uintptr_t>(y)) & 15) == 0;
}

int32_t pitch_of(int32_t n) { return int32_t(ceil_div(n, 64) * 64); }

// Tile width: full GEMM -> minimise waves x width over the persistent grid; tile_skip -> 64 (one swizzle box wide: the
// step is then bound by the epilogue's state traffic, many small tiles balance best and the fp16 copies can leave
// through TMA stores; measured on cfg1: 43 us at 64, 54-56 us at 96..256).
int32_t choose_bn(int32_t n, int32_t R, bool tile_skip, int32_t forced) {
  if (forced >= kChunk * (kEpiWarps / 4) && forced <= kMaxBN && forced % 16 == 0) return forced;
  if (n <= 32) return 32;
  if (tile_skip) return kBK;
  const int64_t tm = ceil_div(R, kBM), sms = sm_count();
  int32_t best = 128;
  double best_cost = 1e300;
  for (int32_t bn : {64, 96, 128, 160, 192, 224, 256}) {
    const int64_t tiles = tm * ceil_div(n, bn);
    const double cost = double(ceil_div(tiles, sms)) * (bn + 4);   // + fixed per-tile overhead
    if (cost < best_cost - 1e-9 || (cost < best_cost + 1e-9 && bn > best)) { best_cost = cost; best = bn; }
  }
  return best;
}

}  // namespace

namespace {
// Workspace layout of the dense path -- ONE walk, used by the size query (measure mode) and by the solve.
struct DenseWs {
  __half* xh[2];
  __half* xl[2];
  int32_t* kb_cnt;
  int32_t* kb_idx;
  int32_t* pk_cnt;
  int32_t* pk_idx;
  int32_t* flags;
  uint32_t* done;
};
DenseWs carve_dense(Workspace& ws, int32_t n, int32_t R) {
  DenseWs w;
  const size_t copy = size_t(R) * pitch_of(n);
  w.xh[0] = ws.take<__half>(copy); w.xl[0] = ws.take<__half>(copy);
  w.xh[1] = ws.take<__half>(copy); w.xl[1] = ws.take<__half>(copy);
  const size_t n_kb = size_t(ceil_div(n, kBK)), n_tn_max = size_t(ceil_div(n, 32));
  w.kb_cnt = ws.take<int32_t>(n_tn_max);
  w.kb_idx = ws.take<int32_t>(n_tn_max * n_kb);
  w.pk_cnt = ws.take<int32_t>(n_kb / 2 + 1);                 // paired tiles (64-wide boxes only)
  w.pk_idx = ws.take<int32_t>((n_kb / 2 + 1) * n_kb);
  w.flags = ws.take<int32_t>(n_tn_max * n_kb);
  w.done = ws.take<uint32_t>(n_tn_max * size_t(ceil_div(R, kBM)));   // fused steps
  return w;
}

// Paired tiles: pairs per replica tile.  Slots go to CTAs round robin (slot % grid), pairs first; the step lasts as long as
// the most loaded CTA (in boxes), so: the largest number of pairs that does not raise that maximum above what single boxes
// give, ceil(boxes / grid) -- or, when min_boxes > 0 (fused launches: state prefetch distance), leaves a CTA with fewer
// than min_boxes boxes per step.
void pair_plan_loads(int32_t n_tiles_n, int32_t n_tiles_m, int grid, int32_t P, int64_t& mx, int64_t& mn) {   // boxes per CTA: max, min
  const int64_t np = int64_t(P) * n_tiles_m, ns = int64_t(n_tiles_n - 2 * P) * n_tiles_m;
  mx = 0; mn = INT64_MAX;
  for (int c = 0; c < grid; ++c) {
    const int64_t pc = np / grid + (c < np % grid ? 1 : 0);
    const int64_t c0 = ((c - np) % grid + grid) % grid;            // first single i with (np + i) % grid == c
    const int64_t sc = c0 < ns ? (ns - c0 + grid - 1) / grid : 0;
    mx = std::max(mx, 2 * pc + sc);
    mn = std::min(mn, 2 * pc + sc);
  }
}
int32_t choose_pair_lines(int32_t n_tiles_n, int32_t n_tiles_m, int grid, int min_boxes) {
  const int64_t target = ceil_div(int64_t(n_tiles_n) * n_tiles_m, grid);
  for (int32_t P = n_tiles_n / 2; P > 0; --P) {
    int64_t mx, mn;
    pair_plan_loads(n_tiles_n, n_tiles_m, grid, P, mx, mn);
    if (mx <= target && mn >= min_boxes) return P;
  }
  return 0;
}

// state16 is usable when the tile is one swizzle box wide with TMA-stored copies, the y ring's boxes are legal (row pitch a
// multiple of 16 bytes, aligned base) and nothing outside the step kernel needs the fp32 x between steps (no remainder
// gather, no dSB sign copies).
bool x16_ok(const DenseArgs& a, const float* y, bool has_rem, const qhap_bsb_params& p, const qhap_bsb_tuning& t) {
  return t.state16 != 2 && a.stage_out && a.BN == kBK && a.R % 4 == 0 && (reinterpret_cast<uintptr_t>(y) & 15) == 0 &&
         (!has_rem || t.y_ring != 1) &&      // with a remainder CSR: the plain-y loop, which also writes the fp32 x (DenseArgs::xw32)
         p.force_mode == 0;
}
}  // namespace

size_t dense_workspace_bytes(int32_t n, int32_t ld, int32_t R) {
  (void)ld;
  Workspace ws(nullptr);
  carve_dense(ws, n, R);
  return ws.used();
}

qhap_status dense_solve_steps(const CsrView& g, const void* dense_J, int32_t ld, int32_t dtype, int32_t R, const float* c1_dev,
                              const qhap_bsb_params& p, float* x, float* y, void* ws_ptr, size_t ws_bytes, cudaStream_t stream) {
  const int32_t n = g.n;
  const qhap_bsb_tuning t = tuning_of(p);
  QHAP_REQUIRE(dtype == QHAP_DENSE_FP16, "dense path takes J in fp16");
  QHAP_REQUIRE(uint64_t(g.n) * uint64_t(R) < (1ull << 32), "dense path: n * replicas must be below 2^32");
  QHAP_REQUIRE((reinterpret_cast<uintptr_t>(dense_J) & 15) == 0, "dense_J must be 16-byte aligned");
  Workspace ws(ws_ptr, ws_bytes);
  const DenseWs w = carve_dense(ws, n, R);
  if (ws.overflow) {
    set_error("dense workspace too small: %zu < %zu", ws_bytes, ws.used());
    return QHAP_ERR_WORKSPACE;
  }
  const int32_t n_k = pitch_of(n);
  const int32_t n_kb = int32_t(ceil_div(n, kBK));

  const bool skip = p.tile_skip != 0;
  const int32_t BN = choose_bn(n, R, skip, t.dense_bn);
  DenseArgs a;
  a.n = n; a.R = R; a.n_k = n_k; a.BN = BN;
  // fp16 copies through TMA stores: the tile must be exactly one 64-column box wide (tile_skip's width); the two
  // staging buffers (2 x 32 KB) come out of the operand-stage budget
  a.stage_out = (BN == kBK) ? 1 : 0;
  a.dsb = p.force_mode == 1 ? 1 : 0;
  a.x16 = x16_ok(a, y, false, p, t) ? 1 : 0;
  // y by plain loads (its own twice-unrolled epilogue loop, and the ring's 32 KB become an operand stage) unless the caller
  // asks for the ring: measured faster on every config (cfg1 24.2 -> 22.7 us per step with single boxes)
  a.yldg = (a.x16 && t.y_ring != 1) ? 1 : 0;
  a.ring = (a.x16 || ring_ok(BN, R, x, y)) ? 1 : 0;
  a.sacc = (t.split_acc != 2 && BN <= 128 && !a.dsb) ? 1 : 0;
  choose_staging(a, BN * kBK * 2 + 2 * kStageX, t);
  a.n_tiles_m = int32_t(ceil_div(R, kBM));
  a.inv_tm = a.n_tiles_m > 1 ? uint32_t((uint64_t(1) << 32) / uint64_t(a.n_tiles_m)) + 1u : 0u;
  QHAP_REQUIRE(ceil_div(n, 32) * int64_t(a.n_tiles_m) * a.n_tiles_m < (int64_t(1) << 32), "tile index arithmetic: too many replica tiles for this n");
  a.n_tiles_n = int32_t(ceil_div(n, BN));
  a.n_kblocks = n_kb;
  a.kb_cnt = skip ? w.kb_cnt : nullptr;
  a.kb_idx = skip ? w.kb_idx : nullptr;
  a.c1 = c1_dev; a.c1_per_row = 0; a.j_terms = 1; a.blk_ptr = nullptr;
  a.x = x; a.y = y;
  a.xw32 = 0; a.early_reload = 0; a.pair_lines = 0; a.n_slots = a.n_tiles_m * a.n_tiles_n; a.pk_cnt = w.pk_cnt; a.pk_idx = w.pk_idx;
  a.pk_ptr = nullptr; a.pk_kb = nullptr; a.pk_l = nullptr; a.pk_r = nullptr;
  set_l2_policies(a, t); a.n_steps = 1; a.fused = 0; a.fence_every = 1; a.k0 = 0; a.steps_total = p.steps_total; a.dt = p.dt; a.a0 = p.a0; a.done = nullptr;

  CUtensorMap tm_j, tm_h[2], tm_l[2], tm_sx, tm_sy;
  QHAP_TRY(make_state_map(&tm_sx, x, n, a.ring ? R : 4));
  QHAP_TRY(make_state_map(&tm_sy, y, n, a.ring ? R : 4));
  QHAP_TRY(make_map(&tm_j, dense_J, uint64_t(ld), uint64_t(ld), uint64_t(ld), uint32_t(BN)));
  for (int b = 0; b < 2; ++b) {
    QHAP_TRY(make_map(&tm_h[b], w.xh[b], uint64_t(n), uint64_t(R), uint64_t(n_k), kBM));
    QHAP_TRY(make_map(&tm_l[b], w.xl[b], uint64_t(n), uint64_t(R), uint64_t(n_k), kBM));
  }

  const dim3 tgrid(unsigned(ceil_div(n_k, 32)), unsigned(ceil_div(R, 32)));
  split_x_kernel<<<tgrid, 256, 0, stream>>>(n, R, n_k, a.x16 ? 2 : a.dsb, x, w.xh[0], w.xl[0]);
  QHAP_LAUNCH_CHECK();
  if (skip) {
    QHAP_CUDA_TRY(cudaMemsetAsync(w.flags, 0, sizeof(int32_t) * size_t(a.n_tiles_n) * n_kb, stream));
    kb_flag_kernel<<<int(ceil_div(int64_t(n) * 32, 256)), 256, 0, stream>>>(n, g.row_ptr, g.col, BN, n_kb, w.flags);
    QHAP_LAUNCH_CHECK();
    kb_list_kernel<<<a.n_tiles_n, 32, 0, stream>>>(n_kb, BN, w.flags, w.kb_cnt, w.kb_idx);
    QHAP_LAUNCH_CHECK();
  }

  // Paired tiles (DenseArgs::pair_lines): state16 with two staging buffers on the tile_skip lists.  y then comes by plain
  // loads (the ring's 32 KB go to the third 48 KB operand stage) unless the caller insists on the ring.
  const int gf = fused_grid(a, p, t);
  if (a.x16 && skip && BN == kBK && a.stg_bufs == 2 && t.pair_tiles != 2) {
    const int g0 = gf ? gf : int(std::min<int64_t>(a.n_slots, sm_count()));
    const int32_t P = choose_pair_lines(a.n_tiles_n, a.n_tiles_m, g0, gf ? 2 : 0);
    if (P > 0) {
      DenseArgs b = a;
      b.pair_lines = P;
      b.n_slots = P * a.n_tiles_m + (a.n_tiles_n - 2 * P) * a.n_tiles_m;
      if (t.y_ring != 1) b.yldg = 1;
      choose_staging(b, 2 * BN * kBK * 2 + 2 * kStageX, t);
      if (b.n_stages >= 2 && b.stg_bufs == 2) {
        a = b;
        pair_list_kernel<<<P, 32, 0, stream>>>(n_kb, w.flags, w.pk_cnt, w.pk_idx);
        QHAP_LAUNCH_CHECK();
      }
    }
  }
  const int grid = int(std::min<int64_t>(a.n_slots, sm_count()));
  a.tile_stride = int32_t(ceil_div(int64_t(a.n_slots), grid) * grid);
  int cur = 0;
  if (gf) {
    QHAP_TRY(launch_fused(gf, stream, tm_j, tm_j, tm_h, tm_l, tm_sx, tm_sy, a, p, w.done, cur));
  } else {
    for (int32_t k = p.step_begin; k < p.step_begin + p.steps_run; ++k) {
      const double a_k = p.steps_total > 1 ? p.a0 * double(k) / double(p.steps_total - 1) : 0.0;   // R10b
      a.c2 = float(p.dt * (p.a0 - a_k));
      a.c3 = float(p.dt * p.a0);
      a.xh_out = w.xh[cur ^ 1];
      a.xl_out = w.xl[cur ^ 1];
      QHAP_TRY(launch_step(grid, stream, tm_j, tm_j, tm_h[cur], tm_l[cur], tm_h[cur ^ 1], tm_l[cur ^ 1], tm_sx, tm_sy, a));
      cur ^= 1;
    }
  }
  if (a.x16) {
    merge_x_kernel<<<tgrid, 256, 0, stream>>>(n, R, n_k, w.xh[cur], w.xl[cur], x);
    QHAP_LAUNCH_CHECK();
  }
  return QHAP_OK;
}

}  // namespace qhap

// ------------------------------------------------------------------------------------------------------------------
// Block path: the same tcgen05 step on a BLOCK-COMPRESSED J built from the CSR (no n x n matrix): only the 64 x 64 tiles
// that hold a non-zero are stored ([blocks x 64][64] fp16, J_hi and -- for fp32 weights -- J_lo), one TMA box each.
// For banded graphs (reads sorted by start, SNPs in genome order, block-diagonal batches of them) that is a few tiles
// per 64 rows; a graph whose tiles would exceed the capacity below (long-range Pore-C edges) is refused and belongs on
// the CSR path.  Batches: c1 is looked up per row (instances may end inside a tile).
namespace qhap {

namespace {
// capacity of the tile arrays: 16x the CSR's own entries, plus one (possibly empty) tile per 64 rows
int64_t block_capacity(int32_t n, int64_t nnz) { return 16 * nnz / (kBK * kBK) + ceil_div(n, kBK) + 1; }
// first threshold (entries per tile) tried when not all tiles fit; see block_solve_steps
int32_t tile_threshold(int32_t R, int32_t j_terms) {
  const double tile = 8192.0 * j_terms + 32768.0 * double(ceil_div(R, kBM));
  const double entry = 1.2 * (8.0 + 4.0 * R);
  int32_t thr = 16;
  while (thr < kBK * kBK && double(thr) * 1.4142 < tile / entry) thr *= 2;      // nearest power of two on a log scale, at least 16
  return thr;
}
}  // namespace

namespace {
// Workspace layout of the block path -- ONE walk, used by the size query (measure mode) and by the solve.
struct BlockWs {
  __half* xh[2];
  __half* xl[2];
  int32_t *kb_cnt, *blk_ptr, *kb_idx, *flags;
  int32_t *pk_ptr, *pk_kb, *pk_l, *pk_r;      // pairs (single-term J without a remainder): union lists, back to back
  float *c1row, *c1plain;
  int32_t *rem_ptr, *rem_col;
  float* rem_val;
  uint32_t* scal;          // absmax bits, scale
  int64_t* totals;         // total blocks, overflow
  int64_t* scan_scratch;
  uint32_t* done;
  __half *jh, *jl;
  int64_t cap_blocks;
};
BlockWs carve_block(Workspace& ws, int32_t n, int64_t nnz, int32_t R) {
  BlockWs w;
  const size_t copy = size_t(R) * pitch_of(n);
  w.xh[0] = ws.take<__half>(copy); w.xl[0] = ws.take<__half>(copy);
  w.xh[1] = ws.take<__half>(copy); w.xl[1] = ws.take<__half>(copy);
  const size_t n_t = size_t(ceil_div(n, kBK));
  w.kb_cnt = ws.take<int32_t>(n_t + 1);
  w.blk_ptr = ws.take<int32_t>(n_t + 1);
  w.kb_idx = ws.take<int32_t>(n_t * n_t);
  w.flags = ws.take<int32_t>(n_t * n_t);
  w.c1row = ws.take<float>(size_t(n));
  w.c1plain = ws.take<float>(size_t(n));
  w.rem_ptr = ws.take<int32_t>(size_t(n) + 1);
  w.rem_col = ws.take<int32_t>(size_t(nnz));
  w.rem_val = ws.take<float>(size_t(nnz));
  w.scal = ws.take<uint32_t>(4);
  w.totals = ws.take<int64_t>(2);
  w.scan_scratch = ws.take<int64_t>(size_t(ceil_div(int64_t(n), 4096)) + 1);
  w.done = ws.take<uint32_t>(n_t * size_t(ceil_div(R, kBM)));   // fused steps
  w.cap_blocks = block_capacity(n, nnz);
  w.pk_ptr = ws.take<int32_t>(n_t / 2 + 2);
  w.pk_kb = ws.take<int32_t>(size_t(w.cap_blocks));
  w.pk_l = ws.take<int32_t>(size_t(w.cap_blocks));
  w.pk_r = ws.take<int32_t>(size_t(w.cap_blocks));
  const size_t cap = size_t(w.cap_blocks + 1) * kBK * kBK;          // + one all-zero tile for the pairs
  w.jh = ws.take<__half>(cap);
  w.jl = ws.take<__half>(cap);
  return w;
}
}  // namespace

size_t block_workspace_bytes(int32_t n, int64_t nnz, int32_t R) {
  Workspace ws(nullptr);
  carve_block(ws, n, nnz, R);
  return ws.used();
}

qhap_status block_solve_steps(const CsrView& g, const float* jval, int32_t weight_mode, int32_t R, int32_t n_inst,
                              const int32_t* inst_ptr_dev, const float* c1_dev, const qhap_bsb_params& p, float* x, float* y,
                              void* ws_ptr, size_t ws_bytes, cudaStream_t stream) {
  const int32_t n = g.n;
  const qhap_bsb_tuning t = tuning_of(p);
  QHAP_REQUIRE(uint64_t(n) * uint64_t(R) < (1ull << 32), "block path: n * replicas must be below 2^32");
  Workspace ws(ws_ptr, ws_bytes);
  const BlockWs w = carve_block(ws, n, g.nnz, R);
  if (ws.overflow) {
    set_error("block workspace too small: %zu < %zu", ws_bytes, ws.used());
    return QHAP_ERR_WORKSPACE;
  }
  const int32_t n_k = pitch_of(n);
  const int32_t n_t = int32_t(ceil_div(n, kBK));
  __half* const* xh = w.xh;
  __half* const* xl = w.xl;
  int32_t *kb_cnt = w.kb_cnt, *blk_ptr = w.blk_ptr, *kb_idx = w.kb_idx, *flags = w.flags;
  float *c1row = w.c1row, *c1plain = w.c1plain;
  int32_t *rem_ptr = w.rem_ptr, *rem_col = w.rem_col;
  float* rem_val = w.rem_val;
  uint32_t* scal = w.scal;
  int64_t *totals = w.totals, *scan_scratch = w.scan_scratch;
  uint32_t* done = w.done;
  const int64_t cap_blocks = w.cap_blocks;
  __half *jh = w.jh, *jl = w.jl;
  const bool two_terms = weight_mode == QHAP_WEIGHT_FX;      // integer counts are exact in fp16 (|J| <= 2048 checked below)

  // tile occupancy -> tile lists -> block offsets.  All tiles are kept if they fit the capacity (banded graphs); otherwise
  // only tiles with at least thr entries (tile_threshold, then doubled) are kept and the rest of the entries (long-range edges) become a
  // remainder CSR that a small gather kernel adds into y before each tile step.  One host synchronisation per attempt.
  QHAP_CUDA_TRY(cudaMemsetAsync(flags, 0, sizeof(int32_t) * size_t(n_t) * n_t, stream));
  QHAP_CUDA_TRY(cudaMemsetAsync(scal, 0, sizeof(uint32_t) * 4, stream));
  tile_count_kernel<<<int(ceil_div(int64_t(n) * 32, 256)), 256, 0, stream>>>(n, g.row_ptr, g.col, n_t, flags);
  QHAP_LAUNCH_CHECK();
  if (g.nnz > 0) {
    absmax_kernel<<<int(std::min<int64_t>(ceil_div(g.nnz, 256), int64_t(sm_count()) * 8)), 256, 0, stream>>>(g.nnz, jval, scal);
    QHAP_LAUNCH_CHECK();
  }
  int64_t total_blocks = 0;
  uint32_t amax_bits = 0;
  // Which tiles to keep when they do not all fit: a kept tile costs its 8 KB per J term plus a 32 KB x k-block per replica tile,
  // an entry left to the remainder CSR (8 + 4 R) bytes of latency-bound gather (weighted 1.2) -- break-even entries per tile, as a
  // power of two.  Measured: cfg4 (R = 128, two J terms) 210.6 us per step at 16, 195.7 at 32 and at 64, 203.8 at 128; cfg1 with
  // Pore-C fragments (R = 1,024, one term) 285.6 at 32, 262.0 at 64.  Both get 64.  Doubled until the tiles fit.
  const int32_t thr0 = tile_threshold(R, two_terms ? 2 : 1);
  int32_t thr = 1;
  for (;; thr = (thr == 1 ? thr0 : thr * 2)) {
    tile_list_kernel<<<n_t, 32, 0, stream>>>(n_t, flags, thr, kb_cnt, kb_idx);
    QHAP_LAUNCH_CHECK();
    QHAP_TRY(exclusive_scan_i32(kb_cnt, blk_ptr, n_t, totals, reinterpret_cast<int32_t*>(totals + 1), stream));
    QHAP_CUDA_TRY(cudaMemcpyAsync(&total_blocks, totals, sizeof(int64_t), cudaMemcpyDeviceToHost, stream));
    QHAP_CUDA_TRY(cudaMemcpyAsync(&amax_bits, scal, sizeof(uint32_t), cudaMemcpyDeviceToHost, stream));
    QHAP_CUDA_TRY(cudaStreamSynchronize(stream));
    if (total_blocks <= cap_blocks) break;
    if (thr > kBK * kBK) {
      set_error("block path: %lld tiles exceed the capacity %lld", (long long)total_blocks, (long long)cap_blocks);
      return QHAP_ERR_RANGE;
    }
  }
  const bool has_rem = thr > 1;
  if (has_rem) {
    const int rb = int(ceil_div(int64_t(n) * 32, 256));
    remainder_kernel<0><<<rb, 256, 0, stream>>>(n, g.row_ptr, g.col, jval, n_t, kb_cnt, kb_idx, rem_ptr, rem_col, rem_val);
    QHAP_LAUNCH_CHECK();
    QHAP_TRY(exclusive_scan_i32(rem_ptr, rem_ptr, n, totals, reinterpret_cast<int32_t*>(totals + 1), stream, scan_scratch));
    remainder_kernel<1><<<rb, 256, 0, stream>>>(n, g.row_ptr, g.col, jval, n_t, kb_cnt, kb_idx, rem_ptr, rem_col, rem_val);
    QHAP_LAUNCH_CHECK();
  }
  float amax;
  memcpy(&amax, &amax_bits, sizeof(float));
  if (!two_terms && amax > 2048.0f) {
    set_error("block path: |J| = %g is not exactly representable in fp16 (> 2048)", double(amax));
    return QHAP_ERR_RANGE;
  }
  float* scale = reinterpret_cast<float*>(scal + 1);
  block_scale_kernel<<<int(ceil_div(std::max(n, 1), 256)), 256, 0, stream>>>(n, n_inst, inst_ptr_dev, c1_dev, scal, two_terms ? 0 : 1,
                                                                            scale, c1row, c1plain);
  QHAP_LAUNCH_CHECK();
  QHAP_CUDA_TRY(cudaMemsetAsync(jh, 0, sizeof(__half) * size_t(total_blocks + 1) * kBK * kBK, stream));   // + the zero tile
  if (two_terms) QHAP_CUDA_TRY(cudaMemsetAsync(jl, 0, sizeof(__half) * size_t(total_blocks) * kBK * kBK, stream));
  block_fill_kernel<<<int(ceil_div(int64_t(n) * 32, 256)), 256, 0, stream>>>(n, g.row_ptr, g.col, jval, n_t, kb_cnt, kb_idx, blk_ptr,
                                                                            scale, jh, two_terms ? jl : nullptr);
  QHAP_LAUNCH_CHECK();

  DenseArgs a;
  a.n = n; a.R = R; a.n_k = n_k; a.BN = kBK;
  a.stage_out = 1;
  a.dsb = p.force_mode == 1 ? 1 : 0;
  a.x16 = x16_ok(a, y, has_rem, p, t) ? 1 : 0;
  // y by plain loads unless the caller asks for the ring (see dense_solve_steps; read graphs here: cfg1 25.1 -> 23.6 us)
  a.yldg = (a.x16 && t.y_ring != 1) ? 1 : 0;
  a.ring = (a.x16 || ring_ok(kBK, R, x, y)) ? 1 : 0;
  a.j_terms = two_terms ? 2 : 1;
  a.sacc = (t.split_acc != 2 && !a.dsb) ? 1 : 0;
  choose_staging(a, a.j_terms * kBK * kBK * 2 + 2 * kStageX, t);
  a.n_tiles_m = int32_t(ceil_div(R, kBM));
  a.inv_tm = a.n_tiles_m > 1 ? uint32_t((uint64_t(1) << 32) / uint64_t(a.n_tiles_m)) + 1u : 0u;
  QHAP_REQUIRE(ceil_div(n, 32) * int64_t(a.n_tiles_m) * a.n_tiles_m < (int64_t(1) << 32), "tile index arithmetic: too many replica tiles for this n");
  a.n_tiles_n = n_t;
  a.n_kblocks = n_t;
  a.kb_cnt = kb_cnt; a.kb_idx = kb_idx; a.blk_ptr = blk_ptr;
  a.xw32 = (a.x16 && has_rem) ? 1 : 0;
  a.early_reload = 0;
  a.pk_ptr = nullptr; a.pk_kb = nullptr; a.pk_l = nullptr; a.pk_r = nullptr;
  a.pair_lines = 0; a.n_slots = a.n_tiles_m * a.n_tiles_n; a.pk_cnt = nullptr; a.pk_idx = nullptr;
  a.c1 = c1row; a.c1_per_row = 1;
  if (n_inst == 1 && !two_terms && !has_rem) {      // one instance, unit scale: every row has the same factor c1 2^-15 -- the dense path's form (the kernel next to a remainder CSR is built for per-row factors)
    a.c1 = c1plain; a.c1_per_row = 0;   // (bit for bit: c1row[i] = c1 2^-15 / 1), without the per-item loads of the row factors
  }
  a.x = x; a.y = y;
  set_l2_policies(a, t); a.n_steps = 1; a.fused = 0; a.fence_every = 1; a.k0 = 0; a.steps_total = p.steps_total; a.dt = p.dt; a.a0 = p.a0; a.done = nullptr;

  CUtensorMap tm_jh, tm_jl, tm_h[2], tm_l[2], tm_sx, tm_sy;
  QHAP_TRY(make_state_map(&tm_sx, x, n, a.ring ? R : 4));
  QHAP_TRY(make_state_map(&tm_sy, y, n, a.ring ? R : 4));
  const uint64_t brows = uint64_t(total_blocks + 1) * kBK;
  QHAP_TRY(make_map(&tm_jh, jh, kBK, brows, kBK, kBK));
  QHAP_TRY(make_map(&tm_jl, two_terms ? jl : jh, kBK, brows, kBK, kBK));
  for (int b = 0; b < 2; ++b) {
    QHAP_TRY(make_map(&tm_h[b], xh[b], uint64_t(n), uint64_t(R), uint64_t(n_k), kBM));
    QHAP_TRY(make_map(&tm_l[b], xl[b], uint64_t(n), uint64_t(R), uint64_t(n_k), kBM));
  }
  const dim3 tgrid(unsigned(ceil_div(n_k, 32)), unsigned(ceil_div(R, 32)));
  split_x_kernel<<<tgrid, 256, 0, stream>>>(n, R, n_k, a.x16 ? 2 : a.dsb, x, xh[0], xl[0]);
  QHAP_LAUNCH_CHECK();
  if (a.xw32) {                       // the remainder gather of the first step must see the pair's value, not the caller's fp32 x
    merge_x_kernel<<<tgrid, 256, 0, stream>>>(n, R, n_k, xh[0], xl[0], x);
    QHAP_LAUNCH_CHECK();
  }
  // the remainder gather reads the fp32 x of the whole graph between two tile steps: a grid-wide step boundary
  const int gf = has_rem ? 0 : fused_grid(a, p, t);
  // Paired tiles as on the dense path, for one J term (read graphs) without a remainder: the union lists carry,
  // per k-block, the tile of the left and of the right box; a box that does not list the k-block gets the all-zero tile.
  if (a.x16 && !has_rem && !two_terms && a.stg_bufs == 2 && t.pair_tiles != 2 && n_inst == 1) {
    const int g0 = gf ? gf : int(std::min<int64_t>(a.n_slots, sm_count()));
    const int32_t P = choose_pair_lines(a.n_tiles_n, a.n_tiles_m, g0, gf ? 2 : 0);
    if (P > 0) {
      DenseArgs b = a;
      b.pair_lines = P;
      b.n_slots = P * a.n_tiles_m + (a.n_tiles_n - 2 * P) * a.n_tiles_m;
      if (t.y_ring != 1) b.yldg = 1;
      choose_staging(b, 2 * kBK * kBK * 2 + 2 * kStageX, t);
      if (b.n_stages >= 2 && b.stg_bufs == 2) {
        a = b;
        const int pb = int(ceil_div(P, 128));
        pair_merge_kernel<false><<<pb, 128, 0, stream>>>(P, n_t, kb_cnt, kb_idx, blk_ptr, int32_t(total_blocks), w.pk_ptr, w.pk_kb, w.pk_l, w.pk_r);
        QHAP_LAUNCH_CHECK();
        QHAP_TRY(exclusive_scan_i32(w.pk_ptr, w.pk_ptr, P, totals, reinterpret_cast<int32_t*>(totals + 1), stream, scan_scratch));
        pair_merge_kernel<true><<<pb, 128, 0, stream>>>(P, n_t, kb_cnt, kb_idx, blk_ptr, int32_t(total_blocks), w.pk_ptr, w.pk_kb, w.pk_l, w.pk_r);
        QHAP_LAUNCH_CHECK();
        a.pk_ptr = w.pk_ptr; a.pk_kb = w.pk_kb; a.pk_l = w.pk_l; a.pk_r = w.pk_r;
      }
    }
  }
  const int grid = int(std::min<int64_t>(a.n_slots, sm_count()));
  a.tile_stride = int32_t(ceil_div(int64_t(a.n_slots), grid) * grid);
  int cur = 0;
  if (gf) {
    QHAP_TRY(launch_fused(gf, stream, tm_jh, tm_jl, tm_h, tm_l, tm_sx, tm_sy, a, p, done, cur));
  } else {
    for (int32_t k = p.step_begin; k < p.step_begin + p.steps_run; ++k) {
      const double a_k = p.steps_total > 1 ? p.a0 * double(k) / double(p.steps_total - 1) : 0.0;   // R10b
      a.c2 = float(p.dt * (p.a0 - a_k));
      a.c3 = float(p.dt * p.a0);
      a.xh_out = xh[cur ^ 1];
      a.xl_out = xl[cur ^ 1];
      if (has_rem) {
        const int rb = int(ceil_div(int64_t(n) * 32, 256));
        if (a.dsb) remainder_step_kernel<true><<<rb, 256, 0, stream>>>(n, R, rem_ptr, rem_col, rem_val, c1plain, x, y);
        else remainder_step_kernel<false><<<rb, 256, 0, stream>>>(n, R, rem_ptr, rem_col, rem_val, c1plain, x, y);
        QHAP_LAUNCH_CHECK();
      }
      QHAP_TRY(launch_step(grid, stream, tm_jh, tm_jl, tm_h[cur], tm_l[cur], tm_h[cur ^ 1], tm_l[cur ^ 1], tm_sx, tm_sy, a));
      cur ^= 1;
    }
  }
  if (a.x16) {
    merge_x_kernel<<<tgrid, 256, 0, stream>>>(n, R, n_k, xh[cur], xl[cur], x);
    QHAP_LAUNCH_CHECK();
  }
  return QHAP_OK;
}

}  // namespace qhap

// Host-only query of the paired-tile plan (no device needed): what dense_solve_steps would choose for this shape.
extern "C" qhap_status qhap_plan_pair_tiles(int32_t n_boxes, int32_t n_replica_tiles, int32_t grid, int32_t min_boxes,
                                            int32_t* pairs_per_line, int32_t* max_boxes_per_cta, int32_t* min_boxes_per_cta) {
  using namespace qhap;
  QHAP_REQUIRE(n_boxes >= 1 && n_replica_tiles >= 1 && grid >= 1 && min_boxes >= 0, "bad sizes");
  QHAP_REQUIRE(pairs_per_line && max_boxes_per_cta && min_boxes_per_cta, "output pointers must not be NULL");
  QHAP_REQUIRE(int64_t(grid) <= int64_t(n_boxes) * n_replica_tiles, "grid larger than the number of boxes");
  const int32_t P = choose_pair_lines(n_boxes, n_replica_tiles, grid, min_boxes);
  int64_t mx, mn;
  pair_plan_loads(n_boxes, n_replica_tiles, grid, P, mx, mn);
  *pairs_per_line = P;
  *max_boxes_per_cta = int32_t(mx);
  *min_boxes_per_cta = int32_t(mn);
  return QHAP_OK;
}
