// (3) Dense bSB step on the tensor cores (tcgen05 / TMEM / TMA).  Placeholder until the kernel lands.
#include "kernels.cuh"

namespace qhap {

size_t dense_workspace_bytes(int32_t, int32_t, int32_t) { return 256; }

qhap_status dense_solve_steps(const CsrView&, const void*, int32_t, int32_t, int32_t, const float*, const qhap_bsb_params&,
                              float*, float*, void*, size_t, cudaStream_t) {
  set_error("dense tcgen05 path not built in this revision");
  return QHAP_ERR_INVALID_ARG;
}

}  // namespace qhap
