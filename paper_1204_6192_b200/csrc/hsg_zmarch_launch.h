// hsg_zmarch_launch.h — host entry points of the z-marching sweep kernel, one per supported lattice size.  Each is defined
// in its own translation unit (hsg_zmarch_l8.cu, ..., hsg_zmarch_l64.cu) so that the sizes compile in parallel.
#pragma once
#include <cuda_runtime.h>
#include "hsg_layout.cuh"
#include "hsg_math.cuh"

namespace hsg {

struct ZmarchArgs {
  Geom g;
  float* spins;                 // [R][3N] private layout
  const float* jh;              // [D][6N]
  const int32_t* temp_of_slot;  // [R]
  const float* beta;            // [T]
  PhiloxKey key;
  unsigned long long k_hb;      // heat-bath sweep counter of the first HB sweep of this call
  int n_or, n_hb;
  double* e_slot;               // [R]    energy of every slot after the call, or nullptr
  double* m_slot;               // [R][3] magnetisation of every slot after the call
  int fast_math;                // heat-bath sweeps use the fast-math variant of the draw (HSG_FLAG_FAST_MATH)
};

// n_launch receives the number of kernel launches made (0 on error); sm_count = SMs of the current device
cudaError_t zmarch_launch_l8(const ZmarchArgs& a, cudaStream_t stream, int* n_launch, int sm_count);
cudaError_t zmarch_launch_l16(const ZmarchArgs& a, cudaStream_t stream, int* n_launch, int sm_count);
cudaError_t zmarch_launch_l32(const ZmarchArgs& a, cudaStream_t stream, int* n_launch, int sm_count);
cudaError_t zmarch_launch_l64(const ZmarchArgs& a, cudaStream_t stream, int* n_launch, int sm_count);

inline bool zmarch_supported(const Geom& g) { return g.L == 8 || g.L == 16 || g.L == 32 || g.L == 64; }

inline cudaError_t zmarch_launch(const ZmarchArgs& a, cudaStream_t stream, int* n_launch, int sm_count) {
  switch (a.g.L) {
    case 8: return zmarch_launch_l8(a, stream, n_launch, sm_count);
    case 16: return zmarch_launch_l16(a, stream, n_launch, sm_count);
    case 32: return zmarch_launch_l32(a, stream, n_launch, sm_count);
    case 64: return zmarch_launch_l64(a, stream, n_launch, sm_count);
    default: *n_launch = 0; return cudaErrorNotSupported;
  }
}

}  // namespace hsg
