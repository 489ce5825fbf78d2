// (6) Phase readout and (7) block stitch.
// Read-based vote, PAPER.md:L271-L281 [Eq. 7-8] (rule at L279 partly garbled; R13):
//   v_j = sum_i s_i M_ij = (c1+ - c1-) - (c2+ - c2-);  hap1[j] = H1 allele if v_j > 0, other allele if v_j < 0, -1 if 0.
// SNP-based, L336-L338 with a single solve: hap1[u] = h1[u] if s_u > 0 else 1 - h1[u].
// Block stitch (R17): o_0 = +1; o_b = sign of the agreement of block b with the oriented block b-1 over their
// overlap (ties -> +1); block b owns the SNPs between the overlap midpoints.
#include <vector>

#include "kernels.cuh"

namespace qhap {
namespace {

__global__ void __launch_bounds__(256) vote_kernel(int32_t n_frag, const int64_t* __restrict__ frag_ptr,
                                                   const int32_t* __restrict__ snp_idx, const uint8_t* __restrict__ allele,
                                                   const uint8_t* __restrict__ h1, const int8_t* __restrict__ spins,
                                                   int32_t* __restrict__ v) {
  const int32_t i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (i >= n_frag) return;
  const int lane = threadIdx.x & 31;
  const int s = spins[i];
  for (int64_t e = frag_ptr[i] + lane; e < frag_ptr[i + 1]; e += 32) {
    const uint8_t al = allele[e];
    if (al > 1) continue;
    const int32_t j = snp_idx[e];
    const int m = (al == (h1 ? h1[j] : uint8_t(0))) ? 1 : -1;   // Eq. 1
    atomicAdd(&v[j], s * m);                                   // integer: order independent
  }
}

__global__ void __launch_bounds__(256) vote_to_hap_kernel(int32_t n_snp, const int32_t* __restrict__ v,
                                                          const uint8_t* __restrict__ h1, int8_t* __restrict__ hap1) {
  const int32_t j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n_snp) return;
  const int8_t hj = h1 ? int8_t(h1[j]) : int8_t(0);
  hap1[j] = v[j] > 0 ? hj : (v[j] < 0 ? int8_t(1 - hj) : int8_t(-1));
}

__global__ void __launch_bounds__(256) snp_readout_kernel(int32_t n_snp, const uint8_t* __restrict__ h1,
                                                          const int8_t* __restrict__ spins, int8_t* __restrict__ hap1) {
  const int32_t u = blockIdx.x * blockDim.x + threadIdx.x;
  if (u >= n_snp) return;
  const int8_t hu = h1 ? int8_t(h1[u]) : int8_t(0);
  hap1[u] = spins[u] > 0 ? hu : int8_t(1 - hu);
}

// One CTA walks the blocks in order (the orientation of block b depends on that of block b-1).
__global__ void __launch_bounds__(256) stitch_orient_kernel(int32_t nb, const int64_t* __restrict__ win,
                                                            const int64_t* __restrict__ off, const int8_t* __restrict__ bs,
                                                            int32_t* __restrict__ orient) {
  __shared__ long long red[256];
  __shared__ int o_prev;
  if (threadIdx.x == 0) { orient[0] = 1; o_prev = 1; }
  __syncthreads();
  for (int32_t b = 1; b < nb; ++b) {
    long long agree = 0;
    for (int64_t i = win[2 * b] + threadIdx.x; i < win[2 * (b - 1) + 1]; i += blockDim.x)
      agree += (long long)(bs[off[b - 1] + (i - win[2 * (b - 1)])]) * bs[off[b] + (i - win[2 * b])];
    red[threadIdx.x] = agree;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
      if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
      __syncthreads();
    }
    if (threadIdx.x == 0) {
      const int ob = (o_prev * red[0] >= 0) ? 1 : -1;
      orient[b] = ob;
      o_prev = ob;
    }
    __syncthreads();
  }
}

__global__ void __launch_bounds__(256) stitch_write_kernel(int32_t n, int32_t nb, const int64_t* __restrict__ win,
                                                           const int64_t* __restrict__ off, const int8_t* __restrict__ bs,
                                                           const int32_t* __restrict__ orient, int8_t* __restrict__ out) {
  const int b = blockIdx.y;
  const int64_t lo = b == 0 ? 0 : (win[2 * b] + win[2 * (b - 1) + 1]) / 2;
  const int64_t hi = b == nb - 1 ? n : (win[2 * (b + 1)] + win[2 * b + 1]) / 2;
  for (int64_t i = lo + int64_t(blockIdx.x) * blockDim.x + threadIdx.x; i < hi; i += int64_t(gridDim.x) * blockDim.x)
    out[i] = int8_t(orient[b] * bs[off[b] + (i - win[2 * b])]);
}

}  // namespace
}  // namespace qhap

using namespace qhap;

extern "C" qhap_status qhap_phase_readout_reads(const qhap_frags* fr, const int8_t* spins, int8_t* hap1, void* workspace,
                                                size_t* ws_bytes, void* stream_v) {
  QHAP_REQUIRE(fr, "frags must not be NULL");
  QHAP_REQUIRE(fr->n_frag >= 0 && fr->n_snp >= 0, "negative sizes");
  Workspace ws(workspace);
  int32_t* v = ws.take<int32_t>(size_t(fr->n_snp));
  qhap_status st;
  if (workspace_protocol(ws, workspace, ws_bytes, &st)) return st;
  QHAP_TRY(require_device());
  QHAP_REQUIRE(fr->n_snp == 0 || hap1, "hap1 must not be NULL");
  QHAP_REQUIRE(fr->n_frag == 0 || (spins && fr->frag_ptr && fr->snp_idx && fr->allele), "spins and fragment arrays must not be NULL");
  cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
  if (fr->n_snp == 0) return QHAP_OK;
  QHAP_CUDA_TRY(cudaMemsetAsync(v, 0, sizeof(int32_t) * size_t(fr->n_snp), stream));
  if (fr->n_frag > 0) {
    vote_kernel<<<int(ceil_div(int64_t(fr->n_frag) * 32, 256)), 256, 0, stream>>>(fr->n_frag, fr->frag_ptr, fr->snp_idx,
                                                                              fr->allele, fr->h1, spins, v);
    QHAP_LAUNCH_CHECK();
  }
  vote_to_hap_kernel<<<int(ceil_div(fr->n_snp, 256)), 256, 0, stream>>>(fr->n_snp, v, fr->h1, hap1);
  QHAP_LAUNCH_CHECK();
  return QHAP_OK;
}

extern "C" qhap_status qhap_phase_readout_snps(int32_t n_snp, const uint8_t* h1, const int8_t* spins, int8_t* hap1,
                                               void* stream_v) {
  QHAP_REQUIRE(n_snp >= 0, "negative size");
  QHAP_TRY(require_device());
  QHAP_REQUIRE(n_snp == 0 || (spins && hap1), "spins and hap1 must not be NULL");
  if (n_snp == 0) return QHAP_OK;
  snp_readout_kernel<<<int(ceil_div(n_snp, 256)), 256, 0, static_cast<cudaStream_t>(stream_v)>>>(n_snp, h1, spins, hap1);
  QHAP_LAUNCH_CHECK();
  return QHAP_OK;
}

extern "C" qhap_status qhap_block_stitch(int32_t n, int32_t n_blocks, const int64_t* win, const int8_t* block_spins,
                                         int8_t* out, void* workspace, size_t* ws_bytes, void* stream_v) {
  QHAP_REQUIRE(n >= 0 && n_blocks >= 1 && win, "bad sizes or NULL windows");
  Workspace ws(workspace);
  int64_t* win_d = ws.take<int64_t>(2 * size_t(n_blocks));
  int64_t* off_d = ws.take<int64_t>(size_t(n_blocks) + 1);
  int32_t* orient = ws.take<int32_t>(size_t(n_blocks));
  qhap_status st;
  if (workspace_protocol(ws, workspace, ws_bytes, &st)) return st;
  QHAP_TRY(require_device());
  QHAP_REQUIRE(block_spins && out, "block_spins and out must not be NULL");
  std::vector<int64_t> off(size_t(n_blocks) + 1, 0);
  for (int b = 0; b < n_blocks; ++b) {
    QHAP_REQUIRE(win[2 * b] >= 0 && win[2 * b] <= win[2 * b + 1] && win[2 * b + 1] <= n, "window outside [0, n]");
    if (b > 0) QHAP_REQUIRE(win[2 * b] >= win[2 * (b - 1)] && win[2 * b] <= win[2 * (b - 1) + 1], "windows must be ordered and contiguous or overlapping");
    off[b + 1] = off[b] + (win[2 * b + 1] - win[2 * b]);
  }
  cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
  QHAP_CUDA_TRY(cudaMemcpyAsync(win_d, win, sizeof(int64_t) * 2 * size_t(n_blocks), cudaMemcpyHostToDevice, stream));
  QHAP_CUDA_TRY(cudaMemcpyAsync(off_d, off.data(), sizeof(int64_t) * (size_t(n_blocks) + 1), cudaMemcpyHostToDevice, stream));
  stitch_orient_kernel<<<1, 256, 0, stream>>>(n_blocks, win_d, off_d, block_spins, orient);
  QHAP_LAUNCH_CHECK();
  stitch_write_kernel<<<dim3(32, n_blocks), 256, 0, stream>>>(n, n_blocks, win_d, off_d, block_spins, orient, out);
  QHAP_LAUNCH_CHECK();
  QHAP_CUDA_TRY(cudaStreamSynchronize(stream));   // `off` is a host temporary
  return QHAP_OK;
}
