// hsg_zmarch.cuh — fused z-marching sweep kernel (placeholder until the kernel lands).
#pragma once
#include "hsg_layout.cuh"
#include "hsg_math.cuh"

namespace hsg {

struct ZmarchArgs {
  Geom g;
  float* spins;
  const float* jh;
  const int32_t* temp_of_slot;
  const float* beta;
  PhiloxKey key;
  unsigned long long k_hb;
  int n_or, n_hb;
};

inline bool zmarch_supported(const Geom&) { return false; }
inline cudaError_t zmarch_launch(const ZmarchArgs&, cudaStream_t, int* n_launch) { *n_launch = 0; return cudaErrorNotSupported; }

}  // namespace hsg
