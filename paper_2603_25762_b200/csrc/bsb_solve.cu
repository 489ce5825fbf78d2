// C entry points qhap_bsb_solve and qhap_cut_eval: argument checks, workspace carving, step loop, finalisation.
// Every arithmetic step runs in the kernels of bsb_sparse.cu / bsb_dense.cu / cut_eval.cu.
#include <vector>

#include "kernels.cuh"

using namespace qhap;

namespace {

struct SolveWs {
  int32_t* inst_ptr;
  float* jval;
  double* sumsq;      // [n_inst + n]: per-instance sums, then per-row partials
  float* c1;
  float* x_alt;
  int64_t* cut;
  int64_t* wtot;
  int64_t* best_cut;
  int32_t* best_replica;
  uint32_t* bits;     // packed signs for the cut evaluation
  void* dense;
  size_t dense_bytes;
};

SolveWs carve(Workspace& ws, int32_t n, int64_t nnz, int32_t n_inst, int32_t R, bool dense, int32_t ld, bool block = false) {
  SolveWs s;
  s.inst_ptr = ws.take<int32_t>(size_t(n_inst) + 1);
  s.jval = ws.take<float>(size_t(nnz));
  s.sumsq = ws.take<double>(size_t(n_inst) + size_t(n));
  s.c1 = ws.take<float>(size_t(n_inst));
  s.x_alt = (dense || block) ? nullptr : ws.take<float>(size_t(n) * R);
  s.cut = ws.take<int64_t>(size_t(n_inst) * R);
  s.wtot = ws.take<int64_t>(size_t(n_inst));
  s.best_cut = ws.take<int64_t>(size_t(n_inst));
  s.best_replica = ws.take<int32_t>(size_t(n_inst));
  s.bits = ws.take<uint32_t>(cut_bits_words(n, R));
  s.dense_bytes = dense ? dense_workspace_bytes(n, ld, R) : (block ? block_workspace_bytes(n, nnz, R) : 0);
  s.dense = (dense || block) ? static_cast<void*>(ws.take<char>(s.dense_bytes)) : nullptr;
  return s;
}

}  // namespace

// One contiguous run of bSB steps [pc.step_begin, pc.step_begin + pc.steps_run) on the chosen path.
static qhap_status run_steps(const CsrView& g, int path, int32_t res_rc, const void* dense_J, int32_t dense_ld, int32_t dense_dtype,
                             int32_t n_inst, const SolveWs& s, const qhap_bsb_params& pc, float* x, float* y, cudaStream_t stream) {
  const int32_t n = g.n, R = pc.replicas;
  if (pc.steps_run <= 0 || n == 0) return QHAP_OK;
  if (path == 1) return dense_solve_steps(g, dense_J, dense_ld, dense_dtype, R, s.c1, pc, x, y, s.dense, s.dense_bytes, stream);
  if (path == 4) return block_solve_steps(g, s.jval, pc.weight_mode, R, n_inst, s.inst_ptr, s.c1, pc, x, y, s.dense, s.dense_bytes, stream);
  if (path == 3) return resident_solve_steps(g, s.jval, R, res_rc, n_inst, s.inst_ptr, s.c1, pc, x, y, stream);
  float* cur = x;
  float* alt = s.x_alt;
  if (pc.steps_run & 1) {   // an odd number of ping-pong steps must end in the caller's x
    QHAP_CUDA_TRY(cudaMemcpyAsync(alt, x, sizeof(float) * size_t(n) * R, cudaMemcpyDeviceToDevice, stream));
    cur = s.x_alt; alt = x;
  }
  for (int32_t k = pc.step_begin; k < pc.step_begin + pc.steps_run; ++k) {
    const double a_k = pc.steps_total > 1 ? pc.a0 * double(k) / double(pc.steps_total - 1) : 0.0;   // R10b
    StepConsts sc;
    sc.c2 = float(pc.dt * (pc.a0 - a_k));
    sc.c3 = float(pc.dt * pc.a0);
    QHAP_TRY(sparse_step(g, s.jval, R, n_inst, s.inst_ptr, s.c1, sc, pc.force_mode, cur, alt, y, stream));
    std::swap(cur, alt);
  }
  return QHAP_OK;
}

extern "C" qhap_status qhap_bsb_solve(const qhap_csr* graph, int32_t n_inst, const int32_t* inst_ptr, const void* dense_J,
                                      int32_t dense_ld, int32_t dense_dtype, const qhap_bsb_params* p, float* x, float* y,
                                      int8_t* best_spins, int64_t* best_cut, int32_t* best_replica,
                                      int64_t* cut_per_replica, void* workspace, size_t* ws_bytes, void* stream_v) {
  QHAP_REQUIRE(graph && p, "graph and params must not be NULL");
  QHAP_REQUIRE(graph->n >= 0 && graph->nnz >= 0 && n_inst >= 1, "bad sizes");
  QHAP_REQUIRE(p->replicas >= 1 && p->steps_total >= 1 && p->step_begin >= 0 && p->steps_run >= 0 &&
                   p->step_begin + p->steps_run <= p->steps_total,
               "bad replica/step counts");
  QHAP_REQUIRE(p->weight_mode >= 0 && p->weight_mode <= 2, "bad weight_mode");
  QHAP_REQUIRE(p->force_mode == 0 || p->force_mode == 1, "force_mode must be 0 (bSB) or 1 (dSB)");
  QHAP_REQUIRE(p->eval_every >= 0, "eval_every must be >= 0");
  QHAP_REQUIRE(p->replica_begin >= 0, "replica_begin must be >= 0");
  QHAP_REQUIRE(n_inst == 1 || inst_ptr, "inst_ptr (host) is required for n_inst > 1");
  if (p->tuning)
    for (int32_t v : p->tuning->reserved) QHAP_REQUIRE(v == 0, "qhap_bsb_tuning.reserved must be 0");
  int path = p->path;
  const int32_t res_rc = (path == 0 || path == 3) ? resident_plan(graph->n, graph->nnz, p->replicas) : 0;
  // auto: small problems -> shared-memory resident; a dense J was built -> tcgen05 over it; otherwise the tcgen05 step on the
  // block-compressed J (hybrid with a remainder CSR for non-banded graphs), except for tiny graphs where the CSR step is as good
  if (path == 0) path = res_rc > 0 ? 3 : ((dense_J && n_inst == 1) ? 1 : ((graph->n >= 1024 && graph->n <= (1 << 20)) ? 4 : 2));   // path 4's tile-occupancy table is (n / 64)^2 ints
  QHAP_REQUIRE(path >= 1 && path <= 4, "path must be 0, 1, 2, 3 or 4");
  QHAP_REQUIRE(path != 3 || res_rc > 0, "resident path: problem too large for shared memory (needs n R <= 65536)");
  if (path == 1) {
    QHAP_REQUIRE(dense_J && n_inst == 1, "dense path needs dense_J and a single instance");
    QHAP_REQUIRE(dense_dtype == QHAP_DENSE_FP16, "dense path takes J in fp16 (exact to |J| <= 2048)");
    QHAP_REQUIRE(dense_ld >= graph->n && dense_ld % 8 == 0, "dense_ld must be >= n and a multiple of 8");
  }
  const int32_t n = graph->n, R = p->replicas;
  Workspace ws(workspace, (workspace && ws_bytes) ? *ws_bytes : ~size_t(0));
  SolveWs s = carve(ws, n, graph->nnz, n_inst, R, path == 1, dense_ld, path == 4);
  qhap_status st;
  if (workspace_protocol(ws, workspace, ws_bytes, &st)) return st;
  QHAP_TRY(require_device());
  QHAP_REQUIRE((x && y) || graph->n == 0, "x and y must not be NULL");
  QHAP_REQUIRE(n == 0 || (graph->row_ptr && (graph->nnz == 0 || graph->col)), "graph arrays must not be NULL");
  if (p->weight_mode == QHAP_WEIGHT_FX) QHAP_REQUIRE(graph->nnz == 0 || graph->w_fx, "w_fx required for weight_mode 2");
  else QHAP_REQUIRE(graph->nnz == 0 || (graph->d && (p->weight_mode == 0 || graph->c)), "d (and c) required for weight_mode 0/1");
  cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
  const CsrView g = view_of(*graph);

  if (n_inst > 1) {
    QHAP_REQUIRE(inst_ptr[0] == 0 && inst_ptr[n_inst] == n, "inst_ptr must start at 0 and end at graph->n");
    for (int b = 0; b < n_inst; ++b) QHAP_REQUIRE(inst_ptr[b] <= inst_ptr[b + 1], "inst_ptr must be non-decreasing");
    QHAP_CUDA_TRY(cudaMemcpyAsync(s.inst_ptr, inst_ptr, sizeof(int32_t) * (size_t(n_inst) + 1), cudaMemcpyHostToDevice, stream));
  } else {
    const int32_t one[2] = {0, n};
    QHAP_CUDA_TRY(cudaMemcpyAsync(s.inst_ptr, one, sizeof(one), cudaMemcpyHostToDevice, stream));
  }
  QHAP_TRY(materialize_jval(g, p->weight_mode, n_inst, s.inst_ptr, s.jval, s.sumsq, stream));
  QHAP_TRY(compute_c1(n, n_inst, s.inst_ptr, s.sumsq, p->dt, p->c0, s.c1, stream));
  if (p->init_state && p->step_begin == 0) QHAP_TRY(init_state(n, R, p->seed, p->replica_begin, x, y, stream));

  // eval_every = k: the steps run in pieces of k, each followed by a cut evaluation of sgn(x) (Fig. 3)
  const bool tracing = p->eval_every > 0 && (p->trace_cut || p->trace_best_cut);
  qhap_bsb_params pc = *p;
  int32_t k = p->step_begin, row = 0;
  const int32_t k_end = p->step_begin + p->steps_run;
  while (k < k_end) {
    pc.step_begin = k;
    pc.steps_run = tracing ? std::min(p->eval_every, k_end - k) : k_end - k;
    QHAP_TRY(run_steps(g, path, res_rc, dense_J, dense_ld, dense_dtype, n_inst, s, pc, x, y, stream));
    k += pc.steps_run;
    if (tracing && pc.steps_run == p->eval_every) {
      int64_t* cut = p->trace_cut ? p->trace_cut + size_t(row) * n_inst * R : s.cut;
      QHAP_TRY(cut_from_x(g, p->weight_mode, x, R, n_inst, s.inst_ptr, cut, s.wtot, s.bits, stream));
      if (p->trace_best_cut)
        QHAP_TRY(cut_finalize(n_inst, R, cut, s.wtot, nullptr, p->trace_best_cut + size_t(row) * n_inst, s.best_replica, stream));
      ++row;
    }
  }
  if (p->finalize) {
    QHAP_REQUIRE(best_spins && best_cut && best_replica, "best_spins, best_cut, best_replica must not be NULL when finalize != 0");
    int64_t* cut = cut_per_replica ? cut_per_replica : s.cut;
    QHAP_TRY(cut_from_x(g, p->weight_mode, x, R, n_inst, s.inst_ptr, cut, s.wtot, s.bits, stream));
    QHAP_TRY(cut_finalize(n_inst, R, cut, s.wtot, nullptr, best_cut, best_replica, stream));
    QHAP_TRY(gather_best_spins(n, R, x, n_inst, s.inst_ptr, best_replica, best_spins, stream));
  }
  return QHAP_OK;
}

extern "C" qhap_status qhap_cut_eval(const qhap_csr* graph, int32_t weight_mode, const int8_t* spins, int32_t replicas,
                                     int64_t* cut, int64_t* energy, void* workspace, size_t* ws_bytes, void* stream_v) {
  QHAP_REQUIRE(graph, "graph must not be NULL");
  QHAP_REQUIRE(graph->n >= 0 && graph->nnz >= 0 && replicas >= 1, "bad sizes");
  QHAP_REQUIRE(weight_mode >= 0 && weight_mode <= 2, "bad weight_mode");
  Workspace ws(workspace);
  int64_t* wtot = ws.take<int64_t>(1);
  int32_t* inst_ptr = ws.take<int32_t>(2);
  uint32_t* bits = ws.take<uint32_t>(cut_bits_words(graph->n, replicas));
  qhap_status st;
  if (workspace_protocol(ws, workspace, ws_bytes, &st)) return st;
  QHAP_TRY(require_device());
  QHAP_REQUIRE(spins && cut, "spins and cut must not be NULL");
  QHAP_REQUIRE(graph->n == 0 || (graph->row_ptr && (graph->nnz == 0 || graph->col)), "graph arrays must not be NULL");
  if (weight_mode == QHAP_WEIGHT_FX) QHAP_REQUIRE(graph->nnz == 0 || graph->w_fx, "w_fx required for weight_mode 2");
  else QHAP_REQUIRE(graph->nnz == 0 || (graph->d && (weight_mode == 0 || graph->c)), "d (and c) required for weight_mode 0/1");
  cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
  const CsrView g = view_of(*graph);
  QHAP_TRY(cut_from_spins(g, weight_mode, spins, replicas, 1, inst_ptr, cut, wtot, bits, stream));
  QHAP_TRY(cut_finalize(1, replicas, cut, wtot, energy, nullptr, nullptr, stream));
  return QHAP_OK;
}
