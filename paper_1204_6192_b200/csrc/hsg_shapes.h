// hsg_shapes.h — host-side launch shapes of the plain (one thread per item) kernels of hsg_kernels.cuh / hsg_observables.cuh:
// how many blocks, how many threads, how many planes per block.  Used by hsg_api.cu for the launches (and by the host
// execution of these kernels in tests/test_kernels_on_host.py, so that the tests run the shapes the library launches).
#pragma once
#include "hsg_kernels.cuh"

namespace hsg {

inline unsigned blocks_for(long long n) { return (unsigned)((n + kThreads - 1) / kThreads); }

// planes per block of the reduction kernels: about 4 vector items per thread, at most L chunks per system
inline int reduce_zb(const Geom& g, int V) {
  const int ipp = 2 * g.L * (g.Lh / V);
  int zb = (4 * kThreads + ipp - 1) / ipp;
  if (zb < 1) zb = 1;
  if (zb > g.L) zb = g.L;
  return zb;
}
inline int vec_width(const Geom& g) { return (g.Lh % 4 == 0) ? 4 : (g.Lh % 2 == 0) ? 2 : 1; }

// a block takes a chunk of planes of one (sample[, pair], temperature): whole lattices up to L = 32, 16 planes beyond
inline void reduction_shape(const Geom& g, int V, int* ZB, int* n_chunks, int* nt) {
  *ZB = g.L > 32 ? 16 : g.L;
  *n_chunks = (g.L + *ZB - 1) / *ZB;
  int n = 32;
  while (n < kThreads && ((long long)*ZB * g.L * (g.Lh / V) >= 8LL * n || n < 2 * (g.Lh / V))) n *= 2;
  *nt = n;
}

}  // namespace hsg
