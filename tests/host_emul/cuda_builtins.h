// cuda_builtins.h — host stand-ins for the CUDA built-ins the plain kernels (hsg_kernels.cuh, hsg_observables.cuh) use
// directly, on the execution model of emu.h: one OS thread per CUDA thread, one block at a time (so `__shared__` arrays can
// be process-wide statics).  Include before the kernel headers.  tests/test_kernels_on_host.py.
#pragma once
#include <cmath>
#include <cstdint>
#include <cuda_runtime.h>
#include "emu.h"

struct EmuDim3 { unsigned x = 1, y = 1, z = 1; };
inline thread_local EmuDim3 threadIdx, blockIdx, blockDim, gridDim;

#define __shared__ static
inline void __syncthreads() { emu::cta_sync(); }
inline double __shfl_down_sync(unsigned, double v, int delta) {
  const int lane = (int)(emu::self.tid & 31u);
  return emu::shuffle<double>(v, lane + delta < 32 ? lane + delta : -1);
}
inline int min(int a, int b) { return a < b ? a : b; }
inline int max(int a, int b) { return a > b ? a : b; }
inline float __fdiv_rn(float a, float b) { return a / b; }
inline float __fsqrt_rn(float a) { return std::sqrt(a); }
inline unsigned long long atomicAdd(unsigned long long* p, unsigned long long v) { return __sync_fetch_and_add(p, v); }

struct float2 { float x, y; };
struct alignas(16) float4 { float x, y, z, w; };
inline float2 make_float2(float x, float y) { return float2{x, y}; }
inline float4 make_float4(float x, float y, float z, float w) { return float4{x, y, z, w}; }

namespace emu {
// kernel<<<grid, block>>>(args...) : blocks one after the other, the threads of a block concurrently
template <class F> void launch_grid(unsigned grid, unsigned block, F kernel) {
  for (unsigned b = 0; b < grid; ++b) {
    Launch ln(1, (int)block, 16, b, {});
    ln.run([=] {
      threadIdx.x = self.tid; blockIdx.x = b; blockDim.x = block; gridDim.x = grid;
      kernel();
    });
  }
}
}  // namespace emu
