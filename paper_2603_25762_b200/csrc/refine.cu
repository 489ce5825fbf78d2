// (f1) SNP-based iterative refinement, PAPER.md:L325-L338 [Eq. 15-17]: solve -> stop if the cut is non-positive or one side
// is empty -> C(p_u) += 1 on the smaller subset (Eq. 16) -> w_uv <- w_uv s_u s_v (Eq. 15, an exact sign flip of the
// fixed-point and fp32 weights) -> solve again; Eq. 17 reads the haplotype from the parity of C.  Readings: DESIGN.md R16.
#include <vector>

#include "kernels.cuh"

using namespace qhap;

namespace {

// One warp per row: flip the sign of the entries that cross the partition.
__global__ void __launch_bounds__(256) gauge_kernel(int32_t n, const int32_t* __restrict__ row_ptr, const int32_t* __restrict__ col,
                                                    const int8_t* __restrict__ spins, int64_t* __restrict__ w_fx, float* __restrict__ w) {
  const int32_t a = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (a >= n) return;
  const int lane = threadIdx.x & 31;
  const int8_t sa = spins[a];
  for (int32_t e = row_ptr[a] + lane; e < row_ptr[a + 1]; e += 32) {
    if (spins[col[e]] != sa) {
      if (w_fx) w_fx[e] = -w_fx[e];
      if (w) w[e] = -w[e];
    }
  }
}

// counts[0] = number of +1 spins (integer atomics: order independent)
__global__ void __launch_bounds__(256) count_pos_kernel(int32_t n, const int8_t* __restrict__ spins, int32_t* __restrict__ counts) {
  int32_t c = 0;
  for (int32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) c += spins[i] > 0;
  c = warp_sum(c);
  if ((threadIdx.x & 31) == 0 && c) atomicAdd(counts, c);
}

// C(p_u) += 1 on the smaller subset; the -1 side on a tie (R16)
__global__ void __launch_bounds__(256) flip_count_kernel(int32_t n, const int8_t* __restrict__ spins, const int32_t* __restrict__ counts,
                                                         int32_t* __restrict__ flip_count) {
  const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int32_t n_pos = counts[0], n_neg = n - n_pos;
  const bool small_is_pos = n_pos < n_neg;
  if ((spins[i] > 0) == small_is_pos) flip_count[i] += 1;
}

__global__ void __launch_bounds__(256) refine_readout_kernel(int32_t n, const uint8_t* __restrict__ h1, const int32_t* __restrict__ flip_count,
                                                             int8_t* __restrict__ hap1) {
  const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint8_t h = h1 ? h1[i] : 0;
  hap1[i] = (flip_count[i] & 1) ? int8_t(1 - h) : int8_t(h);
}

}  // namespace

extern "C" qhap_status qhap_gauge_transform(const qhap_csr* graph, const int8_t* spins, void* stream_v) {
  QHAP_REQUIRE(graph && graph->n >= 0, "graph must not be NULL");
  QHAP_TRY(require_device());
  if (graph->n == 0 || graph->nnz == 0) return QHAP_OK;
  QHAP_REQUIRE(spins && graph->row_ptr && graph->col && (graph->w_fx || graph->w), "spins, row_ptr, col and a weight array are required");
  gauge_kernel<<<int(ceil_div(int64_t(graph->n) * 32, 256)), 256, 0, static_cast<cudaStream_t>(stream_v)>>>(
      graph->n, graph->row_ptr, graph->col, spins, graph->w_fx, graph->w);
  QHAP_LAUNCH_CHECK();
  return QHAP_OK;
}

extern "C" qhap_status qhap_flip_count_update(int32_t n, const int8_t* spins, int32_t* flip_count, void* workspace, size_t* ws_bytes,
                                              void* stream_v) {
  QHAP_REQUIRE(n >= 0, "bad size");
  Workspace ws(workspace);
  int32_t* counts = ws.take<int32_t>(4);
  qhap_status st;
  if (workspace_protocol(ws, workspace, ws_bytes, &st)) return st;
  QHAP_TRY(require_device());
  if (n == 0) return QHAP_OK;
  QHAP_REQUIRE(spins && flip_count, "spins and flip_count must not be NULL");
  cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
  QHAP_CUDA_TRY(cudaMemsetAsync(counts, 0, sizeof(int32_t) * 4, stream));
  count_pos_kernel<<<int(std::min<int64_t>(ceil_div(n, 256), 1024)), 256, 0, stream>>>(n, spins, counts);
  QHAP_LAUNCH_CHECK();
  flip_count_kernel<<<int(ceil_div(n, 256)), 256, 0, stream>>>(n, spins, counts, flip_count);
  QHAP_LAUNCH_CHECK();
  return QHAP_OK;
}

extern "C" qhap_status qhap_refine_readout(int32_t n, const uint8_t* h1, const int32_t* flip_count, int8_t* hap1, void* stream_v) {
  QHAP_REQUIRE(n >= 0, "bad size");
  QHAP_TRY(require_device());
  if (n == 0) return QHAP_OK;
  QHAP_REQUIRE(flip_count && hap1, "flip_count and hap1 must not be NULL");
  refine_readout_kernel<<<int(ceil_div(n, 256)), 256, 0, static_cast<cudaStream_t>(stream_v)>>>(n, h1, flip_count, hap1);
  QHAP_LAUNCH_CHECK();
  return QHAP_OK;
}

namespace {
struct RefineWs {
  int8_t* spins;
  int64_t* cut;
  int32_t* rep;
  int32_t* counts;
  void* solve;
  size_t solve_bytes;
};
}  // namespace

// The loop of PAPER.md:L325-L333 around qhap_bsb_solve (single instance).  Every iteration starts from the seeded
// state of seed + t (R11, R16).  The termination test needs the best cut and the subset sizes on the host:
// one stream synchronisation per iteration.
extern "C" qhap_status qhap_snp_refine(qhap_csr* graph, const qhap_bsb_params* params, int32_t max_iter, float* x, float* y,
                                       int32_t* flip_count, int32_t* iterations, int64_t* cuts, void* workspace, size_t* ws_bytes,
                                       void* stream_v) {
  QHAP_REQUIRE(graph && params && max_iter >= 1, "graph, params and max_iter >= 1 are required");
  const int32_t n = graph->n;
  qhap_bsb_params p = *params;
  p.weight_mode = QHAP_WEIGHT_FX;
  p.init_state = 1; p.finalize = 1; p.step_begin = 0; p.steps_run = p.steps_total;
  size_t solve_bytes = 0;
  QHAP_TRY(qhap_bsb_solve(graph, 1, nullptr, nullptr, 0, QHAP_DENSE_NONE, &p, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr,
                          &solve_bytes, stream_v));
  Workspace ws(workspace);
  RefineWs r;
  r.spins = ws.take<int8_t>(size_t(std::max(n, 1)));
  r.cut = ws.take<int64_t>(1);
  r.rep = ws.take<int32_t>(1);
  r.counts = ws.take<int32_t>(4);
  r.solve_bytes = solve_bytes;
  r.solve = ws.take<char>(solve_bytes);
  qhap_status st;
  if (workspace_protocol(ws, workspace, ws_bytes, &st)) return st;
  QHAP_TRY(require_device());
  QHAP_REQUIRE(x && y && flip_count && iterations && cuts, "x, y, flip_count, iterations (host) and cuts (host) must not be NULL");
  QHAP_REQUIRE(graph->w_fx && graph->w, "the SNP graph's w_fx and w are required (both are updated in place)");
  cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
  QHAP_CUDA_TRY(cudaMemsetAsync(flip_count, 0, sizeof(int32_t) * size_t(n), stream));
  *iterations = 0;
  for (int32_t t = 0; t < max_iter; ++t) {
    p.seed = params->seed + uint64_t(t);
    size_t sb = r.solve_bytes;
    QHAP_TRY(qhap_bsb_solve(graph, 1, nullptr, nullptr, 0, QHAP_DENSE_NONE, &p, x, y, r.spins, r.cut, r.rep, nullptr, r.solve, &sb, stream_v));
    QHAP_CUDA_TRY(cudaMemsetAsync(r.counts, 0, sizeof(int32_t) * 4, stream));
    if (n > 0) {
      count_pos_kernel<<<int(std::min<int64_t>(ceil_div(n, 256), 1024)), 256, 0, stream>>>(n, r.spins, r.counts);
      QHAP_LAUNCH_CHECK();
    }
    int64_t cut = 0;
    int32_t n_pos = 0;
    QHAP_CUDA_TRY(cudaMemcpyAsync(&cut, r.cut, sizeof(int64_t), cudaMemcpyDeviceToHost, stream));
    QHAP_CUDA_TRY(cudaMemcpyAsync(&n_pos, r.counts, sizeof(int32_t), cudaMemcpyDeviceToHost, stream));
    QHAP_CUDA_TRY(cudaStreamSynchronize(stream));
    cuts[t] = cut;
    *iterations = t + 1;
    if (cut <= 0 || n_pos == 0 || n_pos == n) break;          // L333: non-positive cut or a single subset
    flip_count_kernel<<<int(ceil_div(n, 256)), 256, 0, stream>>>(n, r.spins, r.counts, flip_count);   // Eq. 16
    QHAP_LAUNCH_CHECK();
    gauge_kernel<<<int(ceil_div(int64_t(n) * 32, 256)), 256, 0, stream>>>(n, graph->row_ptr, graph->col, r.spins, graph->w_fx, graph->w);   // Eq. 15
    QHAP_LAUNCH_CHECK();
  }
  return QHAP_OK;
}
