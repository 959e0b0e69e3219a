// hsg_zmarch_l8.cu — instantiations of the z-marching sweep kernel for L = 8 (hsg_zmarch.cuh, Tune<8>).
#include "hsg_zmarch_dispatch.cuh"

namespace hsg {
cudaError_t zmarch_launch_l8(const ZmarchArgs& a, cudaStream_t stream, int* n_launch, int sm_count) {
  return zmarch_launch_size<8>(a, stream, n_launch, sm_count);
}
}  // namespace hsg
