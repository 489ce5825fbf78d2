// Internal launcher interface between the translation units of libqhap (device pointers everywhere).
#pragma once

#include <algorithm>

#include "common.cuh"

namespace qhap {

struct CsrView {
  int32_t n = 0;
  int64_t nnz = 0;
  const int32_t* row_ptr = nullptr;
  const int32_t* col = nullptr;
  const int32_t* d = nullptr;
  const int32_t* c = nullptr;
  const int64_t* w_fx = nullptr;
  const float* w = nullptr;
};

inline CsrView view_of(const qhap_csr& g) {
  CsrView v;
  v.n = g.n; v.nnz = g.nnz; v.row_ptr = g.row_ptr; v.col = g.col; v.d = g.d; v.c = g.c; v.w_fx = g.w_fx; v.w = g.w;
  return v;
}

// Tuning knobs of a solve (qhap.h qhap_bsb_tuning): the caller's block, or all zeros = automatic.
inline qhap_bsb_tuning tuning_of(const qhap_bsb_params& p) {
  qhap_bsb_tuning t = {};
  if (p.tuning) t = *p.tuning;
  return t;
}

// bSB step constants, evaluated on the host in fp64 and rounded once to fp32 (R10):
//   y' = fma(c1, F, fma(-c2, x, y)), x' = fma(c3, y', x);  c1 = dt c0 (per instance), c2 = dt (a0 - a_k), c3 = dt a0.
struct StepConsts {
  float c2, c3;
};

// ---- cut_eval.cu
// `bits`: scratch of cut_bits_words(n, R) uint32 (the signs packed to one bit per (spin, replica))
size_t cut_bits_words(int32_t n, int32_t R);
qhap_status cut_from_spins(const CsrView& g, int mode, const int8_t* spins, int32_t R, int32_t n_inst,
                           const int32_t* inst_ptr_dev, int64_t* cut, int64_t* wtot, uint32_t* bits, cudaStream_t stream);
qhap_status cut_from_x(const CsrView& g, int mode, const float* x, int32_t R, int32_t n_inst,
                       const int32_t* inst_ptr_dev, int64_t* cut, int64_t* wtot, uint32_t* bits, cudaStream_t stream);
qhap_status cut_finalize(int32_t n_inst, int32_t R, const int64_t* cut, const int64_t* wtot, int64_t* energy,
                         int64_t* best_cut, int32_t* best_replica, cudaStream_t stream);
qhap_status gather_best_spins(int32_t n, int32_t R, const float* x, int32_t n_inst, const int32_t* inst_ptr_dev,
                              const int32_t* best_replica, int8_t* best_spins, cudaStream_t stream);

// ---- bsb_sparse.cu
// jval[e] = -(float)w_e;  sumsq[inst] = sum of w_e^2 over the instance's directed entries (fp64, deterministic order).
qhap_status materialize_jval(const CsrView& g, int mode, int32_t n_inst, const int32_t* inst_ptr_dev, float* jval,
                             double* sumsq, cudaStream_t stream);
// c1[inst] = (float)(dt * c0_inst), c0_inst = c0 > 0 ? c0 : 0.5 sqrt(N_inst - 1) / sqrt(sumsq[inst])  (1.0 if undefined)
qhap_status compute_c1(int32_t n, int32_t n_inst, const int32_t* inst_ptr_dev, const double* sumsq, double dt, double c0,
                       float* c1, cudaStream_t stream);
qhap_status init_state(int64_t n, int32_t R, uint64_t seed, int32_t replica_begin, float* x, float* y, cudaStream_t stream);
// one bSB step on the CSR path: x_out, y (in place) from x_in; force_mode 1 (dSB): F = J sgn(x_in)
qhap_status sparse_step(const CsrView& g, const float* jval, int32_t R, int32_t n_inst, const int32_t* inst_ptr_dev,
                        const float* c1, StepConsts k, int32_t force_mode, const float* x_in, float* x_out, float* y,
                        cudaStream_t stream);

// ---- bsb_dense.cu
size_t dense_workspace_bytes(int32_t n, int32_t ld, int32_t R);
qhap_status dense_solve_steps(const CsrView& g, const void* dense_J, int32_t ld, int32_t dtype, int32_t R,
                              const float* c1_dev, const qhap_bsb_params& p, float* x, float* y, void* ws, size_t ws_bytes,
                              cudaStream_t stream);

// block-compressed J built from the CSR (64 x 64 fp16 tiles that hold a non-zero), same tcgen05 step; batches allowed
size_t block_workspace_bytes(int32_t n, int64_t nnz, int32_t R);
qhap_status block_solve_steps(const CsrView& g, const float* jval, int32_t weight_mode, int32_t R, int32_t n_inst,
                              const int32_t* inst_ptr_dev, const float* c1_dev, const qhap_bsb_params& p, float* x, float* y,
                              void* ws, size_t ws_bytes, cudaStream_t stream);

// ---- bsb_resident.cu: whole solve in shared memory for small problems (one CTA owns all spins of RC replicas)
int32_t resident_plan(int32_t n, int64_t nnz, int32_t R);   // replicas per CTA, 0 = not applicable
qhap_status resident_solve_steps(const CsrView& g, const float* jval, int32_t R, int32_t RC, int32_t n_inst,
                                 const int32_t* inst_ptr_dev, const float* c1, const qhap_bsb_params& p, float* x, float* y,
                                 cudaStream_t stream);

// ---- graph_read.cu / graph_snp.cu / readout.cu are reached through their C entry points only.

}  // namespace qhap
