// hsg_zmarch_l32.cu — instantiations of the z-marching sweep kernel for L = 32 (hsg_zmarch.cuh, Tune<32>).
#include "hsg_zmarch_dispatch.cuh"

namespace hsg {
cudaError_t zmarch_launch_l32(const ZmarchArgs& a, cudaStream_t stream, int* n_launch, int sm_count) {
  return zmarch_launch_size<32>(a, stream, n_launch, sm_count);
}
}  // namespace hsg
