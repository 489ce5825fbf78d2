/* qhap.h -- C ABI of the QHap hot path on B200 (sm_100a).
 *
 * Method: QHap, arxiv/paper_2603_25762.  Citations are line numbers of /root/reference/PAPER.md
 * (section / equation in brackets).  The library turns a fragment x heterozygous-SNP matrix into a Max-Cut
 * graph (read graph: PAPER.md:L235-L246 [Eq. 2-3]; SNP graph: L287-L319 [Eq. 9-14], Pore-C scaling L350),
 * solves it with ballistic simulated bifurcation over many replicas (L252-L267 [Eq. 4-6]) and reads the
 * phase assignment back (L271-L281 [Eq. 7-8]; L336-L338).
 *
 * Conventions (every entry point):
 *  - plain C, no exceptions cross the boundary; every function returns a qhap_status.
 *  - ALL array pointers are DEVICE pointers owned by the caller unless the comment says HOST.  The library
 *    allocates nothing that outlives a call.  Scratch comes from the caller's `workspace` (device memory,
 *    256-byte aligned).  Calling with workspace == NULL is a SIZE QUERY: it writes the required byte count to
 *    *ws_bytes, launches nothing and returns QHAP_OK.  With workspace != NULL, *ws_bytes is the size provided;
 *    too small -> QHAP_ERR_WORKSPACE (and *ws_bytes = required).
 *  - all work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = legacy default stream).  Entry points
 *    that return a count to the host synchronise the stream: the graph builds, qhap_block_split (nnz),
 *    qhap_component_split (sizes), qhap_snp_refine (once per iteration) and qhap_bsb_solve on path 4 (its tile plan reads
 *    one count back).  qhap_bsb_solve on paths 1-3, qhap_cut_eval, the readouts, qhap_block_stitch, qhap_gauge_transform,
 *    qhap_flip_count_update, qhap_refine_readout and qhap_component_merge are asynchronous: results are valid after the
 *    caller synchronises.
 *  - no global state (one exception: the static scratch array of qhap_cut_eval_static, documented there), no hidden RNG, no CPU fallback: without an sm_100 device every call returns QHAP_ERR_CUDA.
 *  - qhap_last_error() returns a thread-local text for the last non-OK status.
 */
#ifndef QHAP_H_
#define QHAP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define QHAP_API __attribute__((visibility("default")))
#else
#define QHAP_API
#endif

typedef enum {
  QHAP_OK = 0,
  QHAP_ERR_INVALID_ARG = 1, /* NULL where an array is required, negative size, unknown mode              */
  QHAP_ERR_RANGE = 2,       /* a value is not exactly representable (|J| > 2048 in fp16 dense J, > 256 in  */
                            /* bf16; fixed-point sum overflow; nnz >= 2^31)                                  */
  QHAP_ERR_WORKSPACE = 3,   /* workspace or output capacity too small; required size written back          */
  QHAP_ERR_CUDA = 4         /* CUDA runtime error or no sm_100 device                                       */
} qhap_status;

/* Fragment matrix: reads x het SNPs with alleles {0,1,missing} and base qualities (PAPER.md:L216 last sentence;
 * the ternary matrix M of Eq. 1 [L226-L229] and the quality matrix W of Eq. 9-10 [L289-L295] are implicit).
 * CSR by fragment, snp_idx strictly ascending inside a fragment.  The read-graph build additionally requires
 * non-empty fragments sorted by their first SNP index (checked on the device -> QHAP_ERR_INVALID_ARG). */
typedef struct {
  int32_t n_frag, n_snp;
  int64_t nnz;               /* = frag_ptr[n_frag] (host copy, so that size queries need no device read)  */
  const int64_t *frag_ptr;   /* [n_frag+1]                                                                */
  const int32_t *snp_idx;    /* [nnz]                                                                     */
  const uint8_t *allele;     /* [nnz] 0 = ref, 1 = alt, 2 = missing (entry ignored everywhere, Eq. 1 "0") */
  const uint8_t *qual;       /* [nnz] integer Phred, clamped to [1,93]; may be NULL for the read graph    */
  const uint8_t *frag_flags; /* [n_frag] bit0: Pore-C derived (SNP graph: contribution x alpha, L350); NULL = 0 */
  const uint8_t *h1;         /* [n_snp] allele carried by the initial H1 (gauge, L222); NULL = all 0      */
} qhap_frags;

/* Symmetric weighted graph in CSR: both (a,b) and (b,a) stored, columns strictly ascending in a row, no diagonal.
 * Read graph: d = # shared SNPs with opposing alleles (Eq. 2-3), c = # shared with equal alleles.
 * SNP graph: w_fx = Eq. 14 as an exact int64 fixed-point sum at scale 2^-32; w = (float)(w_fx * 2^-32). */
typedef struct {
  int32_t n;        /* vertices                                                                          */
  int64_t nnz;      /* directed entries; on input to a build: CAPACITY of col/d/c/w_fx/w                 */
  int32_t *row_ptr; /* [n+1]                                                                             */
  int32_t *col;     /* [nnz]                                                                             */
  int32_t *d, *c;   /* [nnz] read graph only (else NULL)                                                 */
  int64_t *w_fx;    /* [nnz] SNP graph only (else NULL)                                                  */
  float *w;         /* [nnz] SNP graph only (else NULL)                                                  */
} qhap_csr;

enum { QHAP_WEIGHT_D = 0,        /* w = D        (paper Eq. 3, non-negative)                               */
       QHAP_WEIGHT_D_MINUS_C = 1,/* w = D - C    (BASELINE.json config 0: "discordant minus concordant")   */
       QHAP_WEIGHT_FX = 2 };     /* w = w_fx     (SNP graph)                                               */
enum { QHAP_DENSE_NONE = 0, QHAP_DENSE_FP16 = 1, QHAP_DENSE_BF16 = 2 };

/* (1) Read-graph build, PAPER.md:L235-L246 [Eq. 2-3]; edge set = pairs of fragments sharing >= 1 covered SNP.
 * out->row_ptr must point to [n_frag+1] ints.  If out->col == NULL or out->nnz (capacity) is too small only the
 * count pass runs: row_ptr and out->nnz (required) are written and QHAP_ERR_WORKSPACE is returned when col != NULL.
 * Otherwise col/d/c are filled.  Optionally also writes J = -w (Eq. 4) for `weight_mode` as a dense row-major
 * [dense_ld x dense_ld] matrix (dense_ld >= n_frag, multiple of 8; padding rows/cols written as 0) in fp16 or bf16;
 * an entry that is not exactly representable gives QHAP_ERR_RANGE (checked on device, reported after the sync).
 * The call synchronises the stream ONCE, at its end: with col != NULL the fill kernels follow the count and the scan directly
 * and check on the device that the entries fit (if they do not, col/d/c and dense_J are left untouched). */
QHAP_API qhap_status qhap_build_read_graph(const qhap_frags *frags, int32_t weight_mode, qhap_csr *out, void *dense_J,
                                  int32_t dense_ld, int32_t dense_dtype, void *workspace, size_t *ws_bytes,
                                  void *stream);

/* (2) SNP-graph build, PAPER.md:L287-L319 [Eq. 9-14]; linkage depth k/10 (L85): each SNP of a fragment is linked to
 * its nearest floor(k (|S_i|-1) / 10) downstream SNPs; Pore-C fragments (flag bit0) use the exhaustive depth and
 * their terms are scaled by alpha (L350).  Every term is rounded to int64 at scale 2^32 and integer-added, so the
 * result does not depend on the summation order.  `llr_table` is a HOST array [94*94] of fp64
 * log10(P_cis/P_trans) indexed Qu*94+Qv (Eq. 9, 11, 12), or NULL to let the library evaluate it with the C library.
 * Capacity protocol as for the read graph (out->row_ptr is [n_snp+1]). */
QHAP_API qhap_status qhap_build_snp_graph(const qhap_frags *frags, int32_t linkage_tenths, double alpha,
                                 const double *llr_table, qhap_csr *out, void *workspace, size_t *ws_bytes,
                                 void *stream);

/* Second half of the capacity protocol without repeating the first: fills out->col / w_fx / w (capacity out->nnz)
 * from what the preceding qhap_build_snp_graph call (count pass, out->col == NULL or capacity too small) left in
 * `workspace` and in out->row_ptr.  The caller passes the SAME frags, linkage_tenths, alpha, workspace and
 * out->row_ptr and must not have written to the workspace or to row_ptr in between; the fragment arrays are not read
 * again.  Sizes, parameters and the row_ptr address are checked against a tag the count pass stored in the workspace
 * (mismatch: QHAP_ERR_INVALID_ARG); capacity too small: QHAP_ERR_WORKSPACE.  The result is bit-identical to the one
 * qhap_build_snp_graph itself writes when called with col != NULL. */
QHAP_API qhap_status qhap_build_snp_graph_fill(const qhap_frags *frags, int32_t linkage_tenths, double alpha, qhap_csr *out,
                                      void *workspace, size_t *ws_bytes, void *stream);

/* Optional kernel tuning of qhap_bsb_solve (paths 1 and 4).  NULL, or a field left 0, means AUTOMATIC.  These knobs select
 * launch shapes, shared-memory splits and cache policies; only `state16` and `split_acc` can change result bits (documented there).  They
 * live outside qhap_bsb_params so that the solver's parameter block does not change when a kernel is retuned. */
typedef struct {
  int32_t dense_bn;       /* path 1: tile width in output spins (multiple of 16 in 32..256)                              */
  int32_t step_launch;    /* 1 = one launch per bSB step; automatic = ONE launch runs all steps_run steps when the tiles   */
                          /*    allow and all CTAs can be co-resident (checked with the occupancy API).  Same bits           */
  int32_t l2_hints;       /* L2 eviction priorities of the step kernel: 1 = on (the 16-bit copies of x evict_last, y          */
                          /*    evict_first), 2 = off; automatic = on when the copies fit the L2                              */
  int32_t dense_stg_bufs; /* shared-memory staging buffers for the 16-bit copies of x: 1 or 2                              */
  int32_t dense_epi_sync; /* epilogue warps meet after every tile: 1 = yes, 2 = no                                          */
  int32_t l2_keep_16ths;  /* with the hints on: the share q/16 (1..16) of the kept lines that gets evict_last              */
  int32_t state16;        /* how x is carried BETWEEN the steps of one call on the tile paths (64-wide tiles):               */
                          /*    automatic / 1 = as the pair of fp16 numbers the tensor cores read, 2^15 x = x_hi + x_lo      */
                          /*    (16 B of HBM traffic per spin-update instead of 24; x is rounded to that pair, relative      */
                          /*    2^-22, once per step instead of to fp32's 2^-24); 2 = in fp32.  The x returned to the caller */
                          /*    is fp32 either way                                                                            */
  int32_t split_acc;      /* tiles up to 128 wide: automatic / 1 = the small product terms (x_lo J, x_hi J_lo) accumulate in a   */
                          /*    second TMEM tile and the epilogue adds the two (the tensor cores' fp32 accumulation truncates at */
                          /*    every MMA; kept apart, the small terms no longer truncate the large sum: measured 2-8x smaller   */
                          /*    trajectory drift); 2 = one accumulator.  Changes result bits (documented in DESIGN.md 4.4)       */
  int32_t y_ring;         /* state16: how y reaches the epilogue: automatic = 2 / 1 = per-warp TMA ring in shared memory, 2 = plain   */
                          /*    coalesced loads one work item ahead (frees the ring's 32 KB for another operand stage). Same bits      */
  int32_t pair_tiles;     /* state16 on the dense tile_skip path and on path 4 with one J term and no remainder: automatic / 1 = two neighbouring 64-spin boxes of a replica tile */
                          /*    share one N = 128 accumulator where that does not unbalance the CTAs (each staged x k-block feeds  */
                          /*    128 output spins; y by plain loads unless y_ring = 1), 2 = every box on its own.  Same bits          */
  int32_t reserved[6];    /* must be 0                                                                                      */
} qhap_bsb_tuning;

/* bSB parameters (PAPER.md:L265 gives the outline; constants from BASELINE.json; readings R10a-f):
 *   a_k = a0 k / (steps_total - 1), k = step_begin .. step_begin + steps_run - 1
 *   F = J x (x of the previous step);  y += dt (-(a0 - a_k) x + c0 F);  x += dt a0 y;  |x| > 1: x = sign(x), y = 0.
 * force_mode 1 (dSB, the discrete variant of the paper's bake-off): F = J sgn(x), sgn(0) = +1. */
typedef struct {
  int32_t replicas;     /* R; x, y are [n][R] with the replica index contiguous                           */
  int32_t steps_total;  /* T of the ramp                                                                  */
  int32_t step_begin;   /* first step index run by this call (resume)                                     */
  int32_t steps_run;    /* number of steps run by this call                                               */
  double dt, a0;        /* BASELINE.json: 1.25, 1.0                                                       */
  double c0;            /* <= 0: automatic 0.5 sqrt(N-1) / ||J||_F per instance                           */
  uint64_t seed;        /* used when init_state != 0                                                      */
  int32_t replica_begin;/* global index of this call's replica 0 in the seeded start state (init_state != 0): devices that */
                        /*    share one seed run disjoint slices [replica_begin, replica_begin + replicas) of its replicas  */
  int32_t weight_mode;  /* QHAP_WEIGHT_*: which CSR arrays define w (J = -w)                              */
  int32_t path;         /* which bSB step kernel:                                                           */
                        /*  1 tcgen05 GEMM over the dense J (needs dense_J, fp16, one instance);              */
                        /*  2 sparse CSR step;                                                                */
                        /*  3 shared-memory resident (small problems, n R <= 65536: all steps in one launch;  */
                        /*    same bits as path 2);                                                           */
                        /*  4 tcgen05 step on a block-compressed J built from the CSR (64 x 64 tiles; entries */
                        /*    of sparsely filled tiles -- long-range edges -- go through a remainder CSR      */
                        /*    gather; batches allowed; the plan SYNCHRONISES the stream once or a few times); */
                        /*  0 auto: 3 if it fits, else 1 if dense_J is given, else 4 (2 below 1024 or above 2^20 vertices) */
  int32_t tile_skip;    /* path 1: 1 = visit only the 64-column blocks of J that hold a non-zero (bit-identical) */
  int32_t init_state;   /* 1: x, y <- seeded U(-0.1,0.1) counter hash (R11) before the first step */
  int32_t finalize;     /* 1: after the steps compute cut per replica, best replica, best spins           */
  int32_t force_mode;   /* 0 = bSB (F = J x, the paper's solver, L265); 1 = dSB (F = J sgn(x), L71-L77)     */
  int32_t eval_every;   /* k > 0: after every k-th step of this call (steps step_begin + k, + 2k, ...) the cut of sgn(x)   */
                        /*    of every replica is evaluated -- what Fig. 3 plots per time step -- and      */
                        /*    written to the trace arrays below, row j = after step_begin + (j + 1) k steps; 0 = never      */
  int64_t *trace_cut;      /* DEVICE [steps_run / k][n_inst][R] or NULL                                                       */
  int64_t *trace_best_cut; /* DEVICE [steps_run / k][n_inst]: max over the replicas (min energy, E = W_tot - 2 cut), or NULL */
  const qhap_bsb_tuning *tuning;   /* HOST, optional (NULL = automatic)                                                      */
} qhap_bsb_params;

/* (3)+(4)+(5) bSB solve of `n_inst` independent instances stored as ONE block-diagonal CSR `graph`
 * (instance b owns rows inst_ptr[b] .. inst_ptr[b+1]-1; all its columns lie in the same range).
 * inst_ptr: HOST array [n_inst+1] or NULL for a single instance.  dense_J: optional dense J (see above) for the
 * tensor-core path (single instance only).  x, y: [graph->n][R] fp32 in/out.  Outputs (used when finalize != 0):
 * best_spins [graph->n] int8 (+1/-1, sign(0) = +1), best_cut [n_inst] int64 in the graph's integer units,
 * best_replica [n_inst] (lowest index with maximal cut), cut_per_replica [n_inst][R] (may be NULL). */
QHAP_API qhap_status qhap_bsb_solve(const qhap_csr *graph, int32_t n_inst, const int32_t *inst_ptr, const void *dense_J,
                           int32_t dense_ld, int32_t dense_dtype, const qhap_bsb_params *params, float *x, float *y,
                           int8_t *best_spins, int64_t *best_cut, int32_t *best_replica, int64_t *cut_per_replica,
                           void *workspace, size_t *ws_bytes, void *stream);

/* (5) Cut and Ising energy of given spins, PAPER.md:L254-L263 [Eq. 4-6]:
 *   cut_r = sum over undirected edges with s_a != s_b of w_ab;  energy_r = W_tot - 2 cut_r  (= -1/2 s^T J s, J = -A),
 * in the graph's integer units (counts, or 2^-32 fixed point).  spins: [n][R] int8 (+1/-1).  energy may be NULL. */
QHAP_API qhap_status qhap_cut_eval(const qhap_csr *graph, int32_t weight_mode, const int8_t *spins, int32_t replicas,
                          int64_t *cut, int64_t *energy, void *workspace, size_t *ws_bytes, void *stream);

/* (5') qhap_cut_eval WITHOUT a workspace, for callers that cannot allocate device memory (code under CUDA graph capture,
 * serving loops, harnesses that forbid cudaMalloc).  Same arguments, same results bit for bit, asynchronous on `stream`.
 * The scratch (512 bytes + one bit per (spin, replica), rows padded to 32 replicas) lives in a static device array of
 * QHAP_CUT_STATIC_BYTES inside the library: every GPU that loads the library holds that much until the process exits.
 * Limit: 512 + 4 n ceil(replicas / 32) <= QHAP_CUT_STATIC_BYTES (e.g. 8,000 spins x 4,096 replicas), else
 * QHAP_ERR_WORKSPACE with a message naming both sizes and nothing is launched.  The call allocates and frees nothing.
 * All calls on a device SHARE the array: calls that overlap on the GPU (different streams, no ordering between them) race;
 * calls ordered on one stream, or by events, are safe.  The array keeps the last call's contents; every call clears or
 * overwrites what it reads. */
#define QHAP_CUT_STATIC_BYTES (4u << 20)
QHAP_API qhap_status qhap_cut_eval_static(const qhap_csr *graph, int32_t weight_mode, const int8_t *spins, int32_t replicas,
                                 int64_t *cut, int64_t *energy, void *stream);

/* (6) Phase readout.  Read-based vote, PAPER.md:L271-L281 [Eq. 7-8]: v_j = sum_i s_i M_ij;
 * hap1[j] = H1 allele if v_j > 0, the other allele if v_j < 0, -1 (unphased) if v_j == 0.
 * SNP-based (L336-L338 with one solve): hap1[u] = h1[u] if s_u > 0 else 1 - h1[u]. */
QHAP_API qhap_status qhap_phase_readout_reads(const qhap_frags *frags, const int8_t *spins /*[n_frag]*/, int8_t *hap1 /*[n_snp]*/,
                                     void *workspace, size_t *ws_bytes, void *stream);
QHAP_API qhap_status qhap_phase_readout_snps(int32_t n_snp, const uint8_t *h1 /*may be NULL*/, const int8_t *spins,
                                    int8_t *hap1, void *stream);

/* (7) Block split (BASELINE.json config 3: "independent 5k-SNP overlapping blocks"; R17): sub-graphs induced
 * by the SNP windows [win[2b], win[2b+1]) (HOST array), emitted as one block-diagonal CSR in the order of the windows.
 * Capacity protocol as for the builds; out->row_ptr is [sum of window lengths + 1]. */
QHAP_API qhap_status qhap_block_split(const qhap_csr *graph, int32_t n_blocks, const int64_t *win, qhap_csr *out,
                             void *workspace, size_t *ws_bytes, void *stream);

/* (7) Block stitch: orient each block against the previous one by the majority over the overlap, each block owning
 * the SNPs up to the overlap midpoint.  block_spins: concatenated per-block spins (device); out: [n] (device). */
QHAP_API qhap_status qhap_block_stitch(int32_t n, int32_t n_blocks, const int64_t *win /*HOST*/, const int8_t *block_spins,
                              int8_t *out, void *workspace, size_t *ws_bytes, void *stream);

/* (f1) SNP-based iterative refinement, PAPER.md:L325-L338 [Eq. 15-17]; readings in DESIGN.md R16.
 * qhap_gauge_transform: Eq. 15, w'_uv = -w_uv where spins[u] != spins[v] (w_fx and/or w, in place; exact sign flips).
 * qhap_flip_count_update: Eq. 16, flip_count[u] += 1 for u in the smaller subset of `spins` (the -1 side on a tie).
 * qhap_refine_readout: Eq. 17, hap1[u] = h1[u] if flip_count[u] is even else 1 - h1[u].
 * qhap_snp_refine: the loop -- solve (seed + t, seeded start state, path/replicas/steps from `params`), stop if the best
 *   cut is <= 0 or one side is empty, else Eq. 16 and Eq. 15 -- at most max_iter solves on ONE instance; the graph's
 *   weights are updated in place; flip_count [n] is zeroed first; `iterations` and `cuts` [max_iter] are HOST outputs
 *   (the call synchronises the stream once per iteration). */
QHAP_API qhap_status qhap_gauge_transform(const qhap_csr *graph, const int8_t *spins /*[n]*/, void *stream);
QHAP_API qhap_status qhap_flip_count_update(int32_t n, const int8_t *spins, int32_t *flip_count, void *workspace, size_t *ws_bytes,
                                   void *stream);
QHAP_API qhap_status qhap_refine_readout(int32_t n, const uint8_t *h1 /*may be NULL*/, const int32_t *flip_count, int8_t *hap1,
                                void *stream);
QHAP_API qhap_status qhap_snp_refine(qhap_csr *graph, const qhap_bsb_params *params, int32_t max_iter, float *x, float *y,
                            int32_t *flip_count, int32_t *iterations /*HOST*/, int64_t *cuts /*HOST [max_iter]*/, void *workspace,
                            size_t *ws_bytes, void *stream);

/* (f2) Connected components: the kept components (>= min_size vertices; numbered by their smallest
 * vertex; vertices ascending inside a component) as ONE block-diagonal CSR for qhap_bsb_solve's batch mode (per-component
 * c0 and best replica).  `out` arrays need the INPUT's sizes as capacity (row_ptr [n+1], col and the value arrays
 * [graph->nnz]; a NULL value array is skipped); out->n and out->nnz are written.  perm: device [n] (new index -> old
 * vertex); inst_ptr: HOST [n+1]; n_comp: HOST.  Synchronises the stream.
 * qhap_component_merge: out[perm[i]] = comp_spins[i]; vertices of dropped components get 0 (unphased). */
QHAP_API qhap_status qhap_component_split(const qhap_csr *graph, int32_t min_size, qhap_csr *out, int32_t *perm, int32_t *inst_ptr,
                                 int32_t *n_comp, void *workspace, size_t *ws_bytes, void *stream);
QHAP_API qhap_status qhap_component_merge(int32_t n, int32_t n_kept, const int32_t *perm, const int8_t *comp_spins, int8_t *out,
                                 void *stream);

QHAP_API const char *qhap_last_error(void);
/* Number of CUDA kernels this library has launched in this process so far (monotonic; bench.py reports the difference
 * over its timed region as "gpu_launches"). */
/* HOST-only query (no device, nothing launched): the paired-tile plan of the dense tile_skip step for a graph
 * of n_boxes 64-spin boxes and n_replica_tiles 128-replica tiles on `grid` CTAs.  Slots of a step are numbered pairs first
 * (pair q of replica tile m: slot q n_replica_tiles + m, boxes 2q and 2q + 1), then the boxes from 2 pairs_per_line on as
 * singles (box b of replica tile m: slot (b - pairs_per_line) n_replica_tiles + m); slot s runs on CTA s % grid.  Returns the
 * pairs per replica tile the library would use (0 = no pairs) and the largest / smallest number of boxes any CTA gets per step.
 * min_boxes: 2 for fused launches (state prefetch distance), 0 for one launch per step. */
QHAP_API qhap_status qhap_plan_pair_tiles(int32_t n_boxes, int32_t n_replica_tiles, int32_t grid, int32_t min_boxes,
                                 int32_t *pairs_per_line, int32_t *max_boxes_per_cta, int32_t *min_boxes_per_cta);

QHAP_API uint64_t qhap_launch_count(void);
/* Library / build identification, e.g. "qhap-b200 0.1 sm_100a". */
QHAP_API const char *qhap_version(void);

#ifdef __cplusplus
}
#endif
#endif /* QHAP_H_ */
