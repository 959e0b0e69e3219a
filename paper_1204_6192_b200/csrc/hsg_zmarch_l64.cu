// hsg_zmarch_l64.cu — instantiations of the z-marching sweep kernel for L = 64 (hsg_zmarch.cuh, Tune<64>).
#include "hsg_zmarch_dispatch.cuh"

namespace hsg {
cudaError_t zmarch_launch_l64(const ZmarchArgs& a, cudaStream_t stream, int* n_launch, int sm_count) {
  return zmarch_launch_size<64>(a, stream, n_launch, sm_count);
}
}  // namespace hsg
