// (f2) Connected components and per-component batching, PAPER.md:L248, L319 (the paper solves every connected component
// of the graph separately).  Canonical form (R14): components numbered by their smallest vertex, vertices in
// ascending order inside a component, components with fewer than min_size vertices dropped.  Output: the kept
// components as ONE block-diagonal CSR + perm (new index -> old vertex) + a host inst_ptr, i.e. exactly the batch
// format qhap_bsb_solve takes (per-component c0 and best replica).
// Labels: min-label hooking + pointer jumping (every vertex ends with the smallest vertex of its component as parent;
// integer atomicMin only -> the result does not depend on the execution order).  The grouping of the vertices by label runs
// on the device too: component sizes (integer atomics), two exclusive scans over the roots (offsets and component
// numbers, both in ascending root order), one stable radix sort of the vertices by component number (library primitive:
// cub::DeviceRadixSort) and index arithmetic.  The host only reads back the counts and inst_ptr.
#include <algorithm>

#include <cub/device/device_radix_sort.cuh>

#include "kernels.cuh"

using namespace qhap;

namespace {

__global__ void __launch_bounds__(256) cc_init_kernel(int32_t n, int32_t* __restrict__ parent) {
  const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) parent[i] = i;
}

// One warp per vertex u: m = min over neighbours v of parent[v]; hook parent[u] and the root parent[parent[u]] to m.
__global__ void __launch_bounds__(256) cc_hook_kernel(int32_t n, const int32_t* __restrict__ row_ptr, const int32_t* __restrict__ col,
                                                      int32_t* __restrict__ parent, int32_t* __restrict__ changed) {
  const int32_t u = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (u >= n) return;
  const int lane = threadIdx.x & 31;
  int32_t m = 0x7fffffff;
  for (int32_t e = row_ptr[u] + lane; e < row_ptr[u + 1]; e += 32) m = min(m, parent[col[e]]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = min(m, __shfl_xor_sync(0xffffffffu, m, o));
  if (lane == 0) {
    const int32_t pu = parent[u];
    if (m < pu) {
      atomicMin(parent + pu, m);
      atomicMin(parent + u, m);
      *changed = 1;
    }
  }
}

__global__ void __launch_bounds__(256) cc_jump_kernel(int32_t n, int32_t* __restrict__ parent, int32_t* __restrict__ changed) {
  const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int32_t p = parent[i], gp = parent[p];
  if (gp != p) {
    while (parent[gp] != gp) gp = parent[gp];     // parents only decrease towards the root: terminates
    parent[i] = gp;
    *changed = 1;
  }
}

// size[label] += 1 for every vertex
__global__ void __launch_bounds__(256) cc_size_kernel(int32_t n, const int32_t* __restrict__ parent, int32_t* __restrict__ size) {
  const int32_t v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v < n) atomicAdd(size + parent[v], 1);
}

// per root r (ascending): cnt[r] = size of the component if it is kept, ind[r] = 1 if it is kept
__global__ void __launch_bounds__(256) cc_keep_kernel(int32_t n, int32_t min_size, const int32_t* __restrict__ parent,
                                                      const int32_t* __restrict__ size, int32_t* __restrict__ cnt, int32_t* __restrict__ ind) {
  const int32_t r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n) return;
  const bool keep = parent[r] == r && size[r] >= min_size;
  cnt[r] = keep ? size[r] : 0;
  ind[r] = keep ? 1 : 0;
}

// sort key of vertex v = number of its component among the kept ones (dropped: INT_MAX); inst[number] = offset of the component
__global__ void __launch_bounds__(256) cc_key_kernel(int32_t n, int32_t min_size, const int32_t* __restrict__ parent,
                                                     const int32_t* __restrict__ size, const int32_t* __restrict__ start,
                                                     const int32_t* __restrict__ cidx, int32_t* __restrict__ key, int32_t* __restrict__ val,
                                                     int32_t* __restrict__ inst) {
  const int32_t v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= n) return;
  const int32_t r = parent[v];
  const bool keep = size[r] >= min_size;
  key[v] = keep ? cidx[r] : 0x7fffffff;
  val[v] = v;
  if (keep && r == v) inst[cidx[r]] = start[r];
  if (v == 0) inst[cidx[n]] = start[n];                 // cidx[n] = number of kept components, start[n] = kept vertices
}

// perm[i] = i-th vertex in (component, vertex) order; inv[v] = its new index, -1 for dropped vertices
__global__ void __launch_bounds__(256) cc_perm_kernel(int32_t n, const int32_t* __restrict__ m_dev, const int32_t* __restrict__ sorted,
                                                      int32_t* __restrict__ perm, int32_t* __restrict__ inv) {
  const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int32_t v = sorted[i];
  if (i < *m_dev) { perm[i] = v; inv[v] = i; } else inv[v] = -1;
}

__global__ void __launch_bounds__(256) cc_degree_kernel(int32_t m, const int32_t* __restrict__ perm, const int32_t* __restrict__ row_ptr,
                                                        int32_t* __restrict__ out_cnt) {
  const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < m) out_cnt[i] = row_ptr[perm[i] + 1] - row_ptr[perm[i]];
}

// One warp per new row: copy the old row's entries, columns renumbered through inv (all neighbours are kept).
__global__ void __launch_bounds__(256) cc_fill_kernel(int32_t m, const int32_t* __restrict__ perm, const int32_t* __restrict__ inv,
                                                      const int32_t* __restrict__ row_ptr, const int32_t* __restrict__ col,
                                                      const int32_t* __restrict__ d, const int32_t* __restrict__ c,
                                                      const int64_t* __restrict__ w_fx, const float* __restrict__ w,
                                                      const int32_t* __restrict__ new_ptr, int32_t* __restrict__ ocol, int32_t* __restrict__ od,
                                                      int32_t* __restrict__ oc, int64_t* __restrict__ ow_fx, float* __restrict__ ow) {
  const int32_t i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (i >= m) return;
  const int lane = threadIdx.x & 31;
  const int32_t v = perm[i], e0 = row_ptr[v], len = row_ptr[v + 1] - e0, o0 = new_ptr[i];
  for (int32_t k = lane; k < len; k += 32) {
    ocol[o0 + k] = inv[col[e0 + k]];
    if (d && od) od[o0 + k] = d[e0 + k];
    if (c && oc) oc[o0 + k] = c[e0 + k];
    if (w_fx && ow_fx) ow_fx[o0 + k] = w_fx[e0 + k];
    if (w && ow) ow[o0 + k] = w[e0 + k];
  }
}

__global__ void __launch_bounds__(256) cc_merge_kernel(int32_t m, const int32_t* __restrict__ perm, const int8_t* __restrict__ spins,
                                                       int8_t* __restrict__ out) {
  const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < m) out[perm[i]] = spins[i];
}

}  // namespace

// out arrays need the INPUT's sizes as capacity (row_ptr [n+1], col/d/c/w_fx/w [graph->nnz]; a NULL value array is
// skipped); perm: device [n]; inst_ptr: HOST [n+1]; n_comp: HOST.  out->n, out->nnz are written.  Synchronises the stream
// (label convergence test per round, labels to the host, perm back).
extern "C" qhap_status qhap_component_split(const qhap_csr* graph, int32_t min_size, qhap_csr* out, int32_t* perm, int32_t* inst_ptr,
                                            int32_t* n_comp, void* workspace, size_t* ws_bytes, void* stream_v) {
  QHAP_REQUIRE(graph && out && graph->n >= 0 && graph->nnz >= 0 && min_size >= 1, "bad arguments");
  const int32_t n = graph->n;
  Workspace ws(workspace);
  int32_t* parent = ws.take<int32_t>(size_t(n) + 1);
  int32_t* inv = ws.take<int32_t>(size_t(n) + 1);
  int32_t* flag = ws.take<int32_t>(4);
  int64_t* totals = ws.take<int64_t>(4);
  int64_t* scan_scratch = ws.take<int64_t>(size_t(ceil_div(int64_t(graph->n), 4096)) + 1);
  int32_t* size = ws.take<int32_t>(size_t(n) + 1);
  int32_t* cnt = ws.take<int32_t>(size_t(n) + 1);       // kept sizes per root, then their exclusive scan (start)
  int32_t* cidx = ws.take<int32_t>(size_t(n) + 1);      // kept indicator per root, then its exclusive scan (component number)
  int32_t* key = ws.take<int32_t>(size_t(n) + 1);
  int32_t* val = ws.take<int32_t>(size_t(n) + 1);
  int32_t* key2 = ws.take<int32_t>(size_t(n) + 1);
  int32_t* val2 = ws.take<int32_t>(size_t(n) + 1);
  int32_t* inst_dev = ws.take<int32_t>(size_t(n) + 2);
  // scratch of the radix sort: CUB's own query, which launches nothing (a bound is used should the query fail, e.g. without a device)
  size_t sort_bytes = 0;
  if (cub::DeviceRadixSort::SortPairs(nullptr, sort_bytes, key, key2, val, val2, std::max(n, 1)) != cudaSuccess) {
    (void)cudaGetLastError();
    sort_bytes = size_t(1) << 20;
  }
  sort_bytes = std::max(sort_bytes, size_t(1) << 16);
  char* sort_tmp = ws.take<char>(sort_bytes);
  qhap_status st;
  if (workspace_protocol(ws, workspace, ws_bytes, &st)) return st;
  QHAP_TRY(require_device());
  QHAP_REQUIRE(perm && inst_ptr && n_comp && out->row_ptr, "perm, inst_ptr (host), n_comp (host) and out->row_ptr must not be NULL");
  QHAP_REQUIRE(n == 0 || (graph->row_ptr && (graph->nnz == 0 || (graph->col && out->col))), "graph / out arrays must not be NULL");
  cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
  *n_comp = 0;
  inst_ptr[0] = 0;
  out->n = 0; out->nnz = 0;
  if (n == 0) {
    QHAP_CUDA_TRY(cudaMemsetAsync(out->row_ptr, 0, sizeof(int32_t), stream));
    return QHAP_OK;
  }
  const int vb = int(ceil_div(n, 256)), wb = int(ceil_div(int64_t(n) * 32, 256));
  cc_init_kernel<<<vb, 256, 0, stream>>>(n, parent);
  QHAP_LAUNCH_CHECK();
  for (int round = 0; round < 64; ++round) {            // O(log n) rounds in practice; 64 is a safety bound
    QHAP_CUDA_TRY(cudaMemsetAsync(flag, 0, sizeof(int32_t), stream));
    cc_hook_kernel<<<wb, 256, 0, stream>>>(n, graph->row_ptr, graph->col, parent, flag);
    QHAP_LAUNCH_CHECK();
    cc_jump_kernel<<<vb, 256, 0, stream>>>(n, parent, flag);
    QHAP_LAUNCH_CHECK();
    int32_t changed = 0;
    QHAP_CUDA_TRY(cudaMemcpyAsync(&changed, flag, sizeof(int32_t), cudaMemcpyDeviceToHost, stream));
    QHAP_CUDA_TRY(cudaStreamSynchronize(stream));
    if (!changed) break;
    QHAP_REQUIRE(round < 63, "connected components did not converge");
  }
  // group the vertices by label (= smallest vertex of the component): ascending label, ascending vertex inside a component
  QHAP_CUDA_TRY(cudaMemsetAsync(size, 0, sizeof(int32_t) * (size_t(n) + 1), stream));
  cc_size_kernel<<<vb, 256, 0, stream>>>(n, parent, size);
  QHAP_LAUNCH_CHECK();
  cc_keep_kernel<<<vb, 256, 0, stream>>>(n, min_size, parent, size, cnt, cidx);
  QHAP_LAUNCH_CHECK();
  QHAP_TRY(exclusive_scan_i32(cnt, cnt, n, totals, reinterpret_cast<int32_t*>(totals + 3), stream, scan_scratch));       // start[r]; total = kept vertices
  QHAP_TRY(exclusive_scan_i32(cidx, cidx, n, totals + 1, reinterpret_cast<int32_t*>(totals + 3), stream, scan_scratch));  // number[r]; total = kept components
  cc_key_kernel<<<vb, 256, 0, stream>>>(n, min_size, parent, size, cnt, cidx, key, val, inst_dev);
  QHAP_LAUNCH_CHECK();
  {
    size_t bytes = sort_bytes;
    QHAP_CUDA_TRY(cub::DeviceRadixSort::SortPairs(sort_tmp, bytes, key, key2, val, val2, n, 0, 32, stream));   // stable: vertices stay ascending
    count_launches(3);
  }
  cc_perm_kernel<<<vb, 256, 0, stream>>>(n, cnt + n, val2, perm, inv);
  QHAP_LAUNCH_CHECK();
  int64_t counts[2] = {0, 0};
  QHAP_CUDA_TRY(cudaMemcpyAsync(counts, totals, sizeof(counts), cudaMemcpyDeviceToHost, stream));
  QHAP_CUDA_TRY(cudaStreamSynchronize(stream));
  const int32_t m = int32_t(counts[0]), nc = int32_t(counts[1]);
  QHAP_CUDA_TRY(cudaMemcpyAsync(inst_ptr, inst_dev, sizeof(int32_t) * (size_t(nc) + 1), cudaMemcpyDeviceToHost, stream));
  *n_comp = nc;
  out->n = m;
  if (m == 0) {
    QHAP_CUDA_TRY(cudaMemsetAsync(out->row_ptr, 0, sizeof(int32_t), stream));
    QHAP_CUDA_TRY(cudaStreamSynchronize(stream));
    inst_ptr[0] = 0;
    return QHAP_OK;
  }
  cc_degree_kernel<<<int(ceil_div(m, 256)), 256, 0, stream>>>(m, perm, graph->row_ptr, out->row_ptr);
  QHAP_LAUNCH_CHECK();
  QHAP_TRY(exclusive_scan_i32(out->row_ptr, out->row_ptr, m, totals, reinterpret_cast<int32_t*>(totals + 1), stream, scan_scratch));
  cc_fill_kernel<<<int(ceil_div(int64_t(m) * 32, 256)), 256, 0, stream>>>(m, perm, inv, graph->row_ptr, graph->col, graph->d, graph->c,
                                                                         graph->w_fx, graph->w, out->row_ptr, out->col, out->d, out->c,
                                                                         out->w_fx, out->w);
  QHAP_LAUNCH_CHECK();
  int64_t total = 0;
  QHAP_CUDA_TRY(cudaMemcpyAsync(&total, totals, sizeof(int64_t), cudaMemcpyDeviceToHost, stream));
  QHAP_CUDA_TRY(cudaStreamSynchronize(stream));          // nnz and inst_ptr are on the host now
  out->nnz = total;
  return QHAP_OK;
}

// out[perm[i]] = comp_spins[i]; vertices of dropped components get 0 (unphased).
extern "C" qhap_status qhap_component_merge(int32_t n, int32_t n_kept, const int32_t* perm, const int8_t* comp_spins, int8_t* out,
                                            void* stream_v) {
  QHAP_REQUIRE(n >= 0 && n_kept >= 0 && n_kept <= n, "bad sizes");
  QHAP_TRY(require_device());
  if (n == 0) return QHAP_OK;
  QHAP_REQUIRE(out && (n_kept == 0 || (perm && comp_spins)), "arrays must not be NULL");
  cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
  QHAP_CUDA_TRY(cudaMemsetAsync(out, 0, size_t(n), stream));
  if (n_kept > 0) {
    cc_merge_kernel<<<int(ceil_div(n_kept, 256)), 256, 0, stream>>>(n_kept, perm, comp_spins, out);
    QHAP_LAUNCH_CHECK();
  }
  return QHAP_OK;
}
