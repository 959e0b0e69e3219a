// hsg_zmarch_ptx.cuh — every hardware-specific primitive of the z-marching sweep kernel (hsg_zmarch.cuh): the PTX wrappers
// (mbarrier, cp.async, cp.async.bulk, st.async, thread-block cluster, shared / streaming global access) and the few CUDA
// built-ins it uses (thread and block index, CTA barrier, warp shuffles, the dynamic shared-memory window).  The kernel itself
// is plain C++ over these, so that tests/test_zmarch_on_host.py can compile the very same kernel source for the host against
// a host restatement of THIS file (tests/host_emul/) and run it thread for thread.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "hsg_prim.cuh"

namespace hsg {
namespace zm {

// ---------------------------------------------------------------- CUDA built-ins
__device__ __forceinline__ unsigned tid_x() { return threadIdx.x; }
__device__ __forceinline__ unsigned ctaid_x() { return blockIdx.x; }
__device__ __forceinline__ int imin(int a, int b) { return min(a, b); }
__device__ __forceinline__ void cta_sync() { __syncthreads(); }
__device__ __forceinline__ void warp_sync() { __syncwarp(); }
__device__ __forceinline__ float shfl_idx(uint32_t lanes, float v, int src) { return __shfl_sync(lanes, v, src); }
__device__ __forceinline__ double shfl_down(uint32_t lanes, double v, int delta, int width) { return __shfl_down_sync(lanes, v, delta, width); }
// the CTA's dynamic shared memory, declared inside the kernel
#define HSG_DYN_SMEM(name) extern __shared__ __align__(128) unsigned char name[]

// ---------------------------------------------------------------- PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ uint64_t policy_evict_first() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ uint64_t policy_evict_last() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  return p;
}
// per-thread async copy of 4V bytes global -> shared (streaming: evict-first in L2)
template <int V> __device__ __forceinline__ void cp_async(uint32_t dst, const float* src, uint64_t pol);
template <> __device__ __forceinline__ void cp_async<2>(uint32_t dst, const float* src, uint64_t pol) {
  asm volatile("cp.async.ca.shared.global.L2::cache_hint [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "l"(pol) : "memory");
}
template <> __device__ __forceinline__ void cp_async<4>(uint32_t dst, const float* src, uint64_t pol) {
  asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "l"(pol) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// thread-block cluster helpers (strips of one lattice, see the header comment)
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ uint32_t mapa_u32(uint32_t cta_addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(cta_addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_arrive_relaxed() { asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ void st_cluster_f64(uint32_t addr, double v) {
  asm volatile("st.shared::cluster.f64 [%0], %1;" ::"r"(addr), "d"(v) : "memory");
}

// ---------------------------------------------------------------- V-wide vector access: V = 2 or 4 floats = V/2 packed pairs
// (hsg_math.cuh: F2 = two binary32 lanes in an aligned register pair; lane e&1 of pair e>>1 is compact site j0 + e)

// shared memory by 32-bit shared-window byte address (keeps all address arithmetic 32-bit)
template <int V> __device__ __forceinline__ void lds(F2 (&r)[V / 2], uint32_t a);
template <> __device__ __forceinline__ void lds<2>(F2 (&r)[1], uint32_t a) {
  asm volatile("ld.shared.b64 %0, [%1];" : "=l"(r[0].v) : "r"(a) : "memory");
}
template <> __device__ __forceinline__ void lds<4>(F2 (&r)[2], uint32_t a) {
  asm volatile("ld.shared.v2.b64 {%0,%1}, [%2];" : "=l"(r[0].v), "=l"(r[1].v) : "r"(a) : "memory");
}
template <int V> __device__ __forceinline__ void sts(uint32_t a, const F2 (&r)[V / 2]);
template <> __device__ __forceinline__ void sts<2>(uint32_t a, const F2 (&r)[1]) {
  asm volatile("st.shared.b64 [%0], %1;" ::"r"(a), "l"(r[0].v) : "memory");
}
template <> __device__ __forceinline__ void sts<4>(uint32_t a, const F2 (&r)[2]) {
  asm volatile("st.shared.v2.b64 [%0], {%1,%2};" ::"r"(a), "l"(r[0].v), "l"(r[1].v) : "memory");
}
// asynchronous store into the shared memory of another CTA of the cluster (addresses from mapa_u32); the bytes are
// counted on an mbarrier of THAT CTA, whose threads wait on it: no fence on either side
template <int V> __device__ __forceinline__ void st_async(uint32_t a, const F2 (&r)[V / 2], uint32_t bar);
template <> __device__ __forceinline__ void st_async<2>(uint32_t a, const F2 (&r)[1], uint32_t bar) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b64 [%0], %1, [%2];"
               ::"r"(a), "l"(r[0].v), "r"(bar) : "memory");
}
template <> __device__ __forceinline__ void st_async<4>(uint32_t a, const F2 (&r)[2], uint32_t bar) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.b64 [%0], {%1,%2}, [%3];"
               ::"r"(a), "l"(r[0].v), "l"(r[1].v), "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// bulk asynchronous copy global -> shared, `bytes` (a multiple of 16) counted on the mbarrier `bar` of this CTA
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const float* src, uint32_t bytes, uint32_t bar, uint64_t pol) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(pol) : "memory");
}
__device__ __forceinline__ void fence_mbarrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// streaming global access for the spins: each value is touched once per sweep
template <int V> __device__ __forceinline__ void ldg(F2 (&r)[V / 2], const float* p);
template <> __device__ __forceinline__ void ldg<2>(F2 (&r)[1], const float* p) {
  const float2 t = __ldcs(reinterpret_cast<const float2*>(p));
  r[0] = make_f2(t.x, t.y);
}
template <> __device__ __forceinline__ void ldg<4>(F2 (&r)[2], const float* p) {
  const float4 t = __ldcs(reinterpret_cast<const float4*>(p));
  r[0] = make_f2(t.x, t.y); r[1] = make_f2(t.z, t.w);
}
template <int V> __device__ __forceinline__ void stg(float* p, const F2 (&r)[V / 2]);
template <> __device__ __forceinline__ void stg<2>(float* p, const F2 (&r)[1]) {
  __stcs(reinterpret_cast<float2*>(p), make_float2(f2_lo(r[0]), f2_hi(r[0])));
}
template <> __device__ __forceinline__ void stg<4>(float* p, const F2 (&r)[2]) {
  __stcs(reinterpret_cast<float4*>(p), make_float4(f2_lo(r[0]), f2_hi(r[0]), f2_lo(r[1]), f2_hi(r[1])));
}


}  // namespace zm
}  // namespace hsg
