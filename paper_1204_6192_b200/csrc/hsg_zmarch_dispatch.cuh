// hsg_zmarch_dispatch.cuh — host side of the z-marching sweep kernel: launch configuration, the choice of G (systems per
// CTA) and the dispatch over the instantiations of zm::zmarch_kernel.  Included by the per-size translation units
// (hsg_zmarch_l8.cu ... hsg_zmarch_l64.cu).
#pragma once
#include "hsg_zmarch.cuh"

namespace hsg {

// ------------------------------------------------------------------------------------------------ host side
template <int L, int YS, int V, int G, bool FM = false>
inline cudaError_t zmarch_launch_t(const ZmarchArgs& a, cudaStream_t stream) {
  using C = zm::Cfg<L, YS, V, G>;
  // the attribute is per device: set it on every launch (a host-side table lookup) rather than remember per process,
  // so that contexts on several devices of one process work (hsg.h: "distinct contexts are independent")
  const cudaError_t e = cudaFuncSetAttribute(zm::zmarch_kernel<L, YS, V, G, FM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::smem_bytes);
  if (e != cudaSuccess) return e;
  if (C::NCL == 1) {
    zm::zmarch_kernel<L, YS, V, G, FM><<<a.g.R / G, C::NT, C::smem_bytes, stream>>>(a);
    return cudaGetLastError();
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(a.g.R / G * C::NCL));
  cfg.blockDim = dim3(C::NT);
  cfg.dynamicSmemBytes = C::smem_bytes;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = C::NCL; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, zm::zmarch_kernel<L, YS, V, G, FM>, a);
}

// hsg_sweep(n_or, n_hb) at lattice size L with G systems per CTA: one launch, or (VHB != V and both phases present) an
// over-relaxation launch followed by a heat-bath launch; E and m are reduced by whichever launch holds the final sweep
template <int L, int G>
inline cudaError_t zmarch_launch_g(const ZmarchArgs& a, cudaStream_t stream, int* n_launch) {
  using T = zm::Tune<L>;
  *n_launch = 1;
  if (T::VHB != T::V && a.n_hb > 0) {
    if (a.n_or > 0) {
      ZmarchArgs o = a;
      o.n_hb = 0; o.e_slot = nullptr;
      const cudaError_t e = zmarch_launch_t<L, T::YS, T::V, G>(o, stream);
      if (e != cudaSuccess) return e;
      *n_launch = 2;
    }
    ZmarchArgs h = a;
    h.n_or = 0;
    return a.fast_math ? zmarch_launch_t<L, T::YS, T::VHB, G, true>(h, stream) : zmarch_launch_t<L, T::YS, T::VHB, G>(h, stream);
  }
  // (only a launch that holds heat-bath sweeps has a fast-math form: over-relaxation is the reference arithmetic either way)
  if constexpr (T::VHB == T::V) {
    if (a.fast_math && a.n_hb > 0) return zmarch_launch_t<L, T::YS, T::V, G, true>(a, stream);
  }
  return zmarch_launch_t<L, T::YS, T::V, G>(a, stream);
}

// Systems per CTA: the G slots of a CTA must belong to one sample (G divides O*T); G shrinks while the grid would leave at
// least half of the SMs without a CTA, but not below one full warp per CTA where divisibility allows (L = 8: 16 threads per system).  (Measured on the paper's Table-1 workload, 256 systems of L = 32:
// 128 CTAs of G = 2 run 6.1 ps/update, 256 CTAs of G = 1 run 8.0 — a second wave costs more than 20 idle SMs.)
template <int L>
inline int zmarch_pick_g(const Geom& g, int sm_count) {
  using T = zm::Tune<L>;
  // threads of one system in the launch with the fewest threads per system (V >= VHB): a CTA keeps at least one full warp
  constexpr int TPS_MIN = T::YS * (L / 2 / T::V);
  int G = T::GMAX;
  while (G > 1 && (g.O * g.T) % G != 0) G >>= 1;
  while (G > 1 && (G / 2) * TPS_MIN >= 32 && 2 * (long long)(g.R / G) * (L / T::YS) <= sm_count) G >>= 1;
  return G;
}

template <int L, int G>
inline cudaError_t zmarch_dispatch_g(const ZmarchArgs& a, cudaStream_t stream, int* n_launch, int want_g) {
  if (want_g == G) return zmarch_launch_g<L, G>(a, stream, n_launch);
  if constexpr (G > 1) return zmarch_dispatch_g<L, G / 2>(a, stream, n_launch, want_g);
  *n_launch = 0;
  return cudaErrorNotSupported;
}

// body of the per-size entry points zmarch_launch_l<L> (hsg_zmarch_l8.cu ... hsg_zmarch_l64.cu: one translation unit per
// lattice size, compiled in parallel)
template <int L>
inline cudaError_t zmarch_launch_size(const ZmarchArgs& a, cudaStream_t stream, int* n_launch, int sm_count) {
  return zmarch_dispatch_g<L, zm::Tune<L>::GMAX>(a, stream, n_launch, zmarch_pick_g<L>(a.g, sm_count));
}

}  // namespace hsg
