// (4') Shared-memory-resident bSB solve for small problems (BASELINE.json config 0: 150 spins x 64 replicas x 1,000
// dependent steps, where a launch per step costs more than the step -- SURVEY.md 7 H7 / 8(d) "cfg0: latency").
// Replicas are independent trajectories, so a CTA that owns ALL spins of a few replicas needs nobody
// else's state: x (double-buffered, Jacobi), y, the CSR of J and the per-row c1 live in shared memory for the whole
// call, the steps are separated by __syncthreads only, and the grid is ceil(R / RC) CTAs with no inter-CTA traffic.
// Same recurrence and the same fp32 operation order as the CSR step kernel (bsb_sparse.cu; R10a-f):
//   F = sum_e J_e x_old[col_e] in ascending e;  y' = fma(c1, F, fma(-c2, x, y));  x' = fma(c3, y', x);  wall.
#include "kernels.cuh"

namespace qhap {

namespace {

constexpr int kResThreads = 256;

struct ResidentArgs {
  int32_t n, R, RC, n_inst;
  int64_t nnz;
  const int32_t* row_ptr;
  const int32_t* col;
  const float* jval;
  const int32_t* inst_ptr;
  const float* c1;
  float* x;
  float* y;
  int32_t steps_total, step_begin, steps_run;
  int32_t dsb;                 // 1: F = J sgn(x) (dSB), sgn(0) = +1
  double dt, a0;
};

__global__ void __launch_bounds__(kResThreads) bsb_resident_kernel(const ResidentArgs a) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int n = a.n, RC = a.RC;
  float* xs0 = reinterpret_cast<float*>(smem);
  float* xs1 = xs0 + size_t(n) * RC;
  float* ys = xs1 + size_t(n) * RC;
  float* c1row = ys + size_t(n) * RC;
  float* jv = c1row + n;
  int32_t* cl = reinterpret_cast<int32_t*>(jv + a.nnz);
  int32_t* rp = cl + a.nnz;
  const int r0 = blockIdx.x * RC;
  const int rc = min(RC, a.R - r0);            // replicas owned by this CTA

  for (int64_t e = threadIdx.x; e < a.nnz; e += kResThreads) { jv[e] = a.jval[e]; cl[e] = a.col[e]; }
  for (int i = threadIdx.x; i <= n; i += kResThreads) rp[i] = a.row_ptr[i];
  for (int i = threadIdx.x; i < n; i += kResThreads) {
    int inst = 0;
    if (a.n_inst > 1) {
      int lo = 0, hi = a.n_inst;
      while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (a.inst_ptr[mid] <= i) lo = mid; else hi = mid;
      }
      inst = lo;
    }
    c1row[i] = a.c1[inst];
  }
  for (int p = threadIdx.x; p < n * RC; p += kResThreads) {
    const int i = p / RC, l = p % RC;
    const bool ok = l < rc;
    xs0[p] = ok ? a.x[size_t(i) * a.R + r0 + l] : 0.f;
    ys[p] = ok ? a.y[size_t(i) * a.R + r0 + l] : 0.f;
  }
  __syncthreads();

  float* cur = xs0;
  float* nxt = xs1;
  const int l = threadIdx.x % RC, slot = threadIdx.x / RC, slots = kResThreads / RC;
  const float c3 = float(a.dt * a.a0);
  for (int32_t k = a.step_begin; k < a.step_begin + a.steps_run; ++k) {
    // the same fp64 expressions the host evaluates for the per-launch kernels, rounded once to fp32 (R10b)
    const double a_k = a.steps_total > 1 ? a.a0 * double(k) / double(a.steps_total - 1) : 0.0;
    const float c2 = float(a.dt * (a.a0 - a_k));
    for (int i = slot; i < n; i += slots) {
      float F = 0.f;
      const int e1 = rp[i + 1];
      if (a.dsb) {
        for (int e = rp[i]; e < e1; ++e) F = fmaf(jv[e], cur[cl[e] * RC + l] >= 0.f ? 1.0f : -1.0f, F);
      } else {
        for (int e = rp[i]; e < e1; ++e) F = fmaf(jv[e], cur[cl[e] * RC + l], F);
      }
      const float xo = cur[i * RC + l];
      float yn = fmaf(c1row[i], F, fmaf(-c2, xo, ys[i * RC + l]));
      float xn = fmaf(c3, yn, xo);
      if (fabsf(xn) > 1.0f) {                  // inelastic wall, strict inequality (R10d)
        xn = copysignf(1.0f, xn);
        yn = 0.0f;
      }
      ys[i * RC + l] = yn;
      nxt[i * RC + l] = xn;
    }
    __syncthreads();
    float* t = cur; cur = nxt; nxt = t;
  }
  for (int p = threadIdx.x; p < n * RC; p += kResThreads) {
    const int i = p / RC, ll = p % RC;
    if (ll < rc) {
      a.x[size_t(i) * a.R + r0 + ll] = cur[p];
      a.y[size_t(i) * a.R + r0 + ll] = ys[p];
    }
  }
}

size_t resident_smem_bytes(int32_t n, int64_t nnz, int32_t RC) {
  return size_t(n) * RC * 12 + size_t(n) * 4 + size_t(nnz) * 8 + size_t(n + 1) * 4 + 16;
}

}  // namespace

// Replicas per CTA for the resident kernel, or 0 if the problem does not fit / is not worth it.  Heuristic: the
// per-launch kernels win as soon as one step is much longer than a launch (large n R); the resident kernel needs the
// whole CSR and 12 B per (spin, replica) in <= 200 KB of shared memory.
int32_t resident_plan(int32_t n, int64_t nnz, int32_t R) {
  if (n <= 0 || R <= 0 || int64_t(n) * R > (1 << 16)) return 0;
  for (int32_t rc : {1, 2, 4, 8}) {            // fewest replicas per CTA (shortest step) that still fits the chip in two waves
    if (resident_smem_bytes(n, nnz, rc) <= 200 * 1024 && ceil_div(R, rc) <= 2 * int64_t(sm_count())) return rc;
  }
  return 0;
}

qhap_status resident_solve_steps(const CsrView& g, const float* jval, int32_t R, int32_t RC, int32_t n_inst,
                                 const int32_t* inst_ptr_dev, const float* c1, const qhap_bsb_params& p, float* x, float* y,
                                 cudaStream_t stream) {
  if (g.n == 0 || R == 0 || p.steps_run == 0) return QHAP_OK;
  QHAP_REQUIRE(RC >= 1 && kResThreads % RC == 0, "resident path: bad replica group");
  const size_t smem = resident_smem_bytes(g.n, g.nnz, RC);
  QHAP_REQUIRE(smem <= 200 * 1024, "resident path: problem does not fit in shared memory");
  QHAP_CUDA_TRY(cudaFuncSetAttribute(bsb_resident_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));   // per device
  ResidentArgs a;
  a.n = g.n; a.R = R; a.RC = RC; a.n_inst = n_inst; a.nnz = g.nnz;
  a.row_ptr = g.row_ptr; a.col = g.col; a.jval = jval; a.inst_ptr = inst_ptr_dev; a.c1 = c1;
  a.x = x; a.y = y;
  a.steps_total = p.steps_total; a.step_begin = p.step_begin; a.steps_run = p.steps_run;
  a.dt = p.dt; a.a0 = p.a0; a.dsb = p.force_mode == 1 ? 1 : 0;
  bsb_resident_kernel<<<int(ceil_div(R, RC)), kResThreads, smem, stream>>>(a);
  QHAP_LAUNCH_CHECK();
  return QHAP_OK;
}

}  // namespace qhap
