// (4) Sparse bSB step: F = CSR(J) X with the replica index as the coalesced, vectorised inner dimension, fused with
// the y/x update, the a(t) ramp and the inelastic wall.  PAPER.md:L252-L265 [Eq. 4], L323, L340; constants and the
// recurrence: BASELINE.json + DESIGN.md R10a-f:
//   F = J x_old;  y' = y + dt(-(a0 - a_k) x + c0 F);  x' = x + dt a0 y';  |x'| > 1: x' = sign(x'), y' = 0.
// Also: J value materialisation (J = -w, Eq. 4), ||J||_F^2 per instance, c1 = dt c0, seeded initial state (R11).
#include "kernels.cuh"

namespace qhap {

namespace {

// ------------------------------------------------------------------------------------------- J values
// One warp per row: jval[e] = -(float) w_e; rowsq[a] = sum_e w_e^2 (fp64, fixed lane order -> deterministic).
__global__ void __launch_bounds__(256) jval_kernel(int32_t n, const int32_t* __restrict__ row_ptr,
                                                   const int32_t* __restrict__ d, const int32_t* __restrict__ c,
                                                   const int64_t* __restrict__ w_fx, const float* __restrict__ w, int mode,
                                                   float* __restrict__ jval, double* __restrict__ rowsq) {
  const int32_t a = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (a >= n) return;
  const int lane = threadIdx.x & 31;
  double ss = 0.0;
  for (int32_t e = row_ptr[a] + lane; e < row_ptr[a + 1]; e += 32) {
    float v;
    if (mode == QHAP_WEIGHT_FX) {
      v = w ? w[e] : float(double(w_fx[e]) * (1.0 / 4294967296.0));
    } else {
      v = float(edge_weight(mode, d, c, w_fx, e));
    }
    jval[e] = -v;
    ss += double(v) * double(v);
  }
  ss = warp_sum(ss);
  if (lane == 0) rowsq[a] = ss;
}

// One CTA per instance: sumsq[b] = sum of rowsq over the instance's rows (fixed tree -> deterministic).
__global__ void __launch_bounds__(256) inst_sumsq_kernel(int32_t n, int32_t n_inst, const int32_t* __restrict__ inst_ptr,
                                                         const double* __restrict__ rowsq, double* __restrict__ sumsq) {
  __shared__ double s[256];
  const int b = blockIdx.x;
  const int32_t a0 = n_inst > 1 ? inst_ptr[b] : 0, a1 = n_inst > 1 ? inst_ptr[b + 1] : n;
  double acc = 0.0;
  for (int32_t a = a0 + threadIdx.x; a < a1; a += 256) acc += rowsq[a];
  s[threadIdx.x] = acc;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) s[threadIdx.x] += s[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) sumsq[b] = s[0];
}

__global__ void c1_kernel(int32_t n, int32_t n_inst, const int32_t* __restrict__ inst_ptr,
                          const double* __restrict__ sumsq, double dt, double c0, float* __restrict__ c1) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= n_inst) return;
  const int32_t nb = n_inst > 1 ? inst_ptr[b + 1] - inst_ptr[b] : n;
  double c = c0;
  if (!(c0 > 0.0)) {
    const double ss = sumsq[b];
    c = (ss == 0.0 || nb < 2) ? 1.0 : 0.5 * sqrt(double(nb - 1)) / sqrt(ss);   // R10c
  }
  c1[b] = float(dt * c);
}

// ------------------------------------------------------------------------------------- initial state
__device__ __forceinline__ uint64_t splitmix64(uint64_t z) {
  z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
  z ^= z >> 27; z *= 0x94D049BB133111EBull;
  z ^= z >> 31;
  return z;
}

// x0, y0 ~ U(-0.1, 0.1): idx = (r n + i) 2 + {0: x, 1: y}; z = splitmix64(seed + GOLDEN (idx + 1)); u = z >> 40;
// value = fp32( fp64(2u + 1 - 2^24) * fp64(0.1 / 2^24) )   (R11; same formula as synth.bsb_init_state)
__global__ void __launch_bounds__(256) init_state_kernel(int64_t n, int32_t R, uint64_t seed, int32_t r0, float* __restrict__ x,
                                                         float* __restrict__ y) {
  const int64_t total = n * R;
  for (int64_t p = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; p < total; p += int64_t(gridDim.x) * blockDim.x) {
    const int64_t i = p / R, r = p % R;
    const uint64_t base = (uint64_t(r0 + r) * uint64_t(n) + uint64_t(i)) * 2ull;      // r0 + r: the GLOBAL replica index
#pragma unroll
    for (int which = 0; which < 2; ++which) {
      const uint64_t z = splitmix64(seed + 0x9E3779B97F4A7C15ull * (base + which + 1ull));
      const long long u = (long long)(z >> 40);
      const double v = double(2 * u + 1 - (1ll << 24)) * (0.1 / 16777216.0);
      (which == 0 ? x : y)[p] = __double2float_rn(v);
    }
  }
}

// ------------------------------------------------------------------------------------------ the step
// dSB: the force sees sgn(x), sgn(0) = sgn(-0) = +1 (R10e)
__device__ __forceinline__ float sgn1(float v) { return v >= 0.f ? 1.0f : -1.0f; }

template <int VEC>
struct Vec;
template <>
struct Vec<4> {
  using T = float4;
  static __device__ __forceinline__ void fma(float (&f)[4], float v, const float4& a) {
    f[0] = fmaf(v, a.x, f[0]); f[1] = fmaf(v, a.y, f[1]); f[2] = fmaf(v, a.z, f[2]); f[3] = fmaf(v, a.w, f[3]);
  }
  static __device__ __forceinline__ void unpack(float (&f)[4], const float4& a) { f[0] = a.x; f[1] = a.y; f[2] = a.z; f[3] = a.w; }
  static __device__ __forceinline__ float4 pack(const float (&f)[4]) { return make_float4(f[0], f[1], f[2], f[3]); }
  static __device__ __forceinline__ float4 sgn(const float4& a) { return make_float4(sgn1(a.x), sgn1(a.y), sgn1(a.z), sgn1(a.w)); }
};
template <>
struct Vec<2> {
  using T = float2;
  static __device__ __forceinline__ void fma(float (&f)[2], float v, const float2& a) {
    f[0] = fmaf(v, a.x, f[0]); f[1] = fmaf(v, a.y, f[1]);
  }
  static __device__ __forceinline__ void unpack(float (&f)[2], const float2& a) { f[0] = a.x; f[1] = a.y; }
  static __device__ __forceinline__ float2 pack(const float (&f)[2]) { return make_float2(f[0], f[1]); }
  static __device__ __forceinline__ float2 sgn(const float2& a) { return make_float2(sgn1(a.x), sgn1(a.y)); }
};
template <>
struct Vec<1> {
  using T = float;
  static __device__ __forceinline__ void fma(float (&f)[1], float v, const float& a) { f[0] = fmaf(v, a, f[0]); }
  static __device__ __forceinline__ void unpack(float (&f)[1], const float& a) { f[0] = a; }
  static __device__ __forceinline__ float pack(const float (&f)[1]) { return f[0]; }
  static __device__ __forceinline__ float sgn(const float& a) { return sgn1(a); }
};

// The fused update of one (spin, replica): returns x', writes y'.
__device__ __forceinline__ float bsb_update(float F, float x, float& y, float c1, float c2, float c3) {
  float yn = fmaf(c1, F, fmaf(-c2, x, y));
  float xn = fmaf(c3, yn, x);
  if (fabsf(xn) > 1.0f) {            // inelastic wall, strict inequality (R10d)
    xn = copysignf(1.0f, xn);
    yn = 0.0f;
  }
  y = yn;
  return xn;
}

constexpr int kRowsPerBlock = 32;   // consecutive rows share neighbours -> their x rows stay in L1
constexpr int kWarps = 8;

template <int VEC, bool DSB>
__global__ void __launch_bounds__(kWarps * 32) sparse_step_kernel(
    int32_t n, const int32_t* __restrict__ row_ptr, const int32_t* __restrict__ col, const float* __restrict__ jval,
    int32_t R, int32_t n_inst, const int32_t* __restrict__ inst_ptr, const float* __restrict__ c1v, float c2, float c3,
    const float* __restrict__ x_in, float* __restrict__ x_out, float* __restrict__ y) {
  using V = typename Vec<VEC>::T;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int chunks = (R + 32 * VEC - 1) / (32 * VEC);
  const int64_t n_tiles = (int64_t(n) + kRowsPerBlock - 1) / kRowsPerBlock;
  for (int64_t work = blockIdx.x; work < n_tiles * chunks; work += gridDim.x) {
    const int chunk = int(work / n_tiles);                 // chunk-major: neighbouring CTAs work on neighbouring rows
    const int32_t a_begin = int32_t(work % n_tiles) * kRowsPerBlock;
    const int r = chunk * 32 * VEC + lane * VEC;
    const bool active = r < R;
    for (int32_t a = a_begin + warp; a < min(n, a_begin + kRowsPerBlock); a += kWarps) {
      const int32_t e0 = row_ptr[a], e1 = row_ptr[a + 1];
      float F[VEC];
#pragma unroll
      for (int k = 0; k < VEC; ++k) F[k] = 0.f;
      if (active) {
        int32_t e = e0;
        for (; e + 4 <= e1; e += 4) {
          const int32_t b0 = __ldg(col + e), b1 = __ldg(col + e + 1), b2 = __ldg(col + e + 2), b3 = __ldg(col + e + 3);
          const float v0 = __ldg(jval + e), v1 = __ldg(jval + e + 1), v2 = __ldg(jval + e + 2), v3 = __ldg(jval + e + 3);
          V x0 = *reinterpret_cast<const V*>(x_in + size_t(b0) * R + r);
          V x1 = *reinterpret_cast<const V*>(x_in + size_t(b1) * R + r);
          V x2 = *reinterpret_cast<const V*>(x_in + size_t(b2) * R + r);
          V x3 = *reinterpret_cast<const V*>(x_in + size_t(b3) * R + r);
          if constexpr (DSB) { x0 = Vec<VEC>::sgn(x0); x1 = Vec<VEC>::sgn(x1); x2 = Vec<VEC>::sgn(x2); x3 = Vec<VEC>::sgn(x3); }
          Vec<VEC>::fma(F, v0, x0); Vec<VEC>::fma(F, v1, x1); Vec<VEC>::fma(F, v2, x2); Vec<VEC>::fma(F, v3, x3);
        }
        for (; e < e1; ++e) {
          V xv = *reinterpret_cast<const V*>(x_in + size_t(__ldg(col + e)) * R + r);
          if constexpr (DSB) xv = Vec<VEC>::sgn(xv);
          Vec<VEC>::fma(F, __ldg(jval + e), xv);
        }
        int inst = 0;
        if (n_inst > 1) {
          int lo = 0, hi = n_inst;
          while (hi - lo > 1) {
            int mid = (lo + hi) >> 1;
            if (__ldg(inst_ptr + mid) <= a) lo = mid; else hi = mid;
          }
          inst = lo;
        }
        const float c1 = __ldg(c1v + inst);
        float xs[VEC], ys[VEC];
        Vec<VEC>::unpack(xs, *reinterpret_cast<const V*>(x_in + size_t(a) * R + r));
        Vec<VEC>::unpack(ys, *reinterpret_cast<const V*>(y + size_t(a) * R + r));
#pragma unroll
        for (int k = 0; k < VEC; ++k) xs[k] = bsb_update(F[k], xs[k], ys[k], c1, c2, c3);
        *reinterpret_cast<V*>(x_out + size_t(a) * R + r) = Vec<VEC>::pack(xs);
        *reinterpret_cast<V*>(y + size_t(a) * R + r) = Vec<VEC>::pack(ys);
      }
    }
  }
}

}  // namespace

qhap_status materialize_jval(const CsrView& g, int mode, int32_t n_inst, const int32_t* inst_ptr_dev, float* jval,
                             double* sumsq, cudaStream_t stream) {
  if (g.n == 0) return QHAP_OK;
  // rowsq lives right after sumsq in the caller's buffer: sumsq has n_inst + n slots
  double* rowsq = sumsq + n_inst;
  jval_kernel<<<int(ceil_div(int64_t(g.n) * 32, 256)), 256, 0, stream>>>(g.n, g.row_ptr, g.d, g.c, g.w_fx, g.w, mode, jval,
                                                                         rowsq);
  QHAP_LAUNCH_CHECK();
  inst_sumsq_kernel<<<n_inst, 256, 0, stream>>>(g.n, n_inst, inst_ptr_dev, rowsq, sumsq);
  QHAP_LAUNCH_CHECK();
  return QHAP_OK;
}

qhap_status compute_c1(int32_t n, int32_t n_inst, const int32_t* inst_ptr_dev, const double* sumsq, double dt, double c0,
                       float* c1, cudaStream_t stream) {
  c1_kernel<<<int(ceil_div(n_inst, 128)), 128, 0, stream>>>(n, n_inst, inst_ptr_dev, sumsq, dt, c0, c1);
  QHAP_LAUNCH_CHECK();
  return QHAP_OK;
}

qhap_status init_state(int64_t n, int32_t R, uint64_t seed, int32_t replica_begin, float* x, float* y, cudaStream_t stream) {
  if (n * R == 0) return QHAP_OK;
  const int blocks = int(std::min<int64_t>(ceil_div(n * R, 256), int64_t(sm_count()) * 16));
  init_state_kernel<<<blocks, 256, 0, stream>>>(n, R, seed, replica_begin, x, y);
  QHAP_LAUNCH_CHECK();
  return QHAP_OK;
}

qhap_status sparse_step(const CsrView& g, const float* jval, int32_t R, int32_t n_inst, const int32_t* inst_ptr_dev,
                        const float* c1, StepConsts k, int32_t force_mode, const float* x_in, float* x_out, float* y,
                        cudaStream_t stream) {
  if (g.n == 0 || R == 0) return QHAP_OK;
  const bool al16 = ((reinterpret_cast<uintptr_t>(x_in) | reinterpret_cast<uintptr_t>(x_out) | reinterpret_cast<uintptr_t>(y)) & 15) == 0;
  const int vec = (R % 4 == 0 && R >= 128 && al16) ? 4 : ((R % 2 == 0 && al16) ? 2 : 1);
  const int chunks = int(ceil_div(R, 32 * vec));
  const int64_t work = ceil_div(g.n, kRowsPerBlock) * chunks;
  const int blocks = int(std::min<int64_t>(work, int64_t(sm_count()) * 8));
#define QHAP_STEP_ARGS g.n, g.row_ptr, g.col, jval, R, n_inst, inst_ptr_dev, c1, k.c2, k.c3, x_in, x_out, y
  if (force_mode == 1) {
    if (vec == 4) sparse_step_kernel<4, true><<<blocks, kWarps * 32, 0, stream>>>(QHAP_STEP_ARGS);
    else if (vec == 2) sparse_step_kernel<2, true><<<blocks, kWarps * 32, 0, stream>>>(QHAP_STEP_ARGS);
    else sparse_step_kernel<1, true><<<blocks, kWarps * 32, 0, stream>>>(QHAP_STEP_ARGS);
  } else {
    if (vec == 4) sparse_step_kernel<4, false><<<blocks, kWarps * 32, 0, stream>>>(QHAP_STEP_ARGS);
    else if (vec == 2) sparse_step_kernel<2, false><<<blocks, kWarps * 32, 0, stream>>>(QHAP_STEP_ARGS);
    else sparse_step_kernel<1, false><<<blocks, kWarps * 32, 0, stream>>>(QHAP_STEP_ARGS);
  }
#undef QHAP_STEP_ARGS
  QHAP_LAUNCH_CHECK();
  return QHAP_OK;
}

}  // namespace qhap
