// Host restatement of paper_1204_6192_b200/csrc/hsg_zmarch_ptx.cuh for tests/test_zmarch_on_host.py: the same names and
// signatures, implemented on the execution model of emu.h (PTX semantics, see there).  Cache policies are ignored.
#pragma once
#include <cstdint>
#include <cstring>
#include <thread>
#include <cuda_runtime.h>
#include "hsg_prim.cuh"
#include "emu.h"

namespace hsg {
namespace zm {

// ---------------------------------------------------------------- CUDA built-ins
inline unsigned tid_x() { return emu::self.tid; }
inline unsigned ctaid_x() { return emu::self.cta->block_id; }
inline int imin(int a, int b) { return a < b ? a : b; }
inline void cta_sync() { emu::cta_sync(); }
inline void warp_sync() { emu::warp_sync(); }
inline float shfl_idx(uint32_t lanes, float v, int src) {
  if (!((lanes >> src) & 1u)) { std::fprintf(stderr, "emu: shuffle from lane %d outside the mask\n", src); std::abort(); }
  return emu::shuffle<float>(v, src);
}
inline double shfl_down(uint32_t, double v, int delta, int width) {
  const int lane = (int)(emu::self.tid & 31u);
  const int src = (lane % width) + delta < width ? lane + delta : -1;     // out of the segment: the caller's own value
  return emu::shuffle<double>(v, src);
}
#define HSG_DYN_SMEM(name) unsigned char* const name = emu::self.cta->smem

// ---------------------------------------------------------------- "PTX" wrappers
inline uint32_t smem_u32(const void* p) { return emu::addr_of(p); }
inline void mbar_init(uint64_t* bar, uint32_t count) { emu::self.cta->mbar(emu::addr_of(bar)).init((int)count); }
inline uint64_t policy_evict_first() { return 0; }
inline uint64_t policy_evict_last() { return 0; }
template <int V> inline void cp_async(uint32_t dst, const float* src, uint64_t) { emu::cp_async(dst, src, 4u * V); }
inline void cp_async_commit() { emu::cp_async_commit(); }
template <int N> inline void cp_async_wait() { emu::cp_async_wait(N); }

inline uint32_t cluster_ctarank() { return (uint32_t)emu::self.cta->rank; }
inline uint32_t mapa_u32(uint32_t cta_addr, uint32_t rank) { return (cta_addr & 0xFFFFFFu) | ((rank + 1u) << 24); }
inline void cluster_arrive() { emu::cluster_arrive(); }
inline void cluster_arrive_relaxed() { emu::cluster_arrive(); }
inline void cluster_wait() { emu::cluster_wait(); }
inline void st_cluster_f64(uint32_t addr, double v) { std::memcpy(emu::ptr_of(addr), &v, 8); }

template <int V> inline void lds(F2 (&r)[V / 2], uint32_t a) {
  if (a % (4u * V)) { std::fprintf(stderr, "emu: misaligned ld.shared\n"); std::abort(); }
  std::memcpy(&r[0], emu::ptr_of(a), 4u * V);
}
template <int V> inline void sts(uint32_t a, const F2 (&r)[V / 2]) {
  if (a % (4u * V)) { std::fprintf(stderr, "emu: misaligned st.shared\n"); std::abort(); }
  std::memcpy(emu::ptr_of(a), &r[0], 4u * V);
}
// st.async: remote store whose bytes are counted on an mbarrier of the destination CTA
template <int V> inline void st_async(uint32_t a, const F2 (&r)[V / 2], uint32_t bar) {
  if ((a & 0xFFFFFFu) % (4u * V) || (bar & 7u)) { std::fprintf(stderr, "emu: misaligned st.async or mbarrier\n"); std::abort(); }
  emu::Copy c{emu::ptr_of(a), nullptr, 4u * V, {0}, true};
  std::memcpy(c.imm, &r[0], 4u * V);
  emu::cta_of(bar)->mbar(bar & 0xFFFFFFu).transfer(c);
}
inline void mbar_expect_tx(uint32_t bar, uint32_t bytes) { emu::cta_of(bar)->mbar(bar & 0xFFFFFFu).arrive_expect_tx(bytes); }
inline void bulk_g2s(uint32_t dst, const float* src, uint32_t bytes, uint32_t bar, uint64_t) {
  if (bytes % 16u || dst % 16u || ((uintptr_t)src % 16u)) { std::fprintf(stderr, "emu: cp.async.bulk needs 16-byte alignment and size\n"); std::abort(); }
  emu::Copy c{emu::ptr_of(dst), (const unsigned char*)src, bytes, {0}, false};
  if ((dst & 0xFFFFFFu) + bytes > emu::self.cta->smem_bytes) { std::fprintf(stderr, "emu: bulk copy runs past the end of shared memory\n"); std::abort(); }
  emu::cta_of(bar)->mbar(bar & 0xFFFFFFu).transfer(c);
}
inline void fence_mbarrier_init() {}
inline void mbar_wait(uint32_t bar, uint32_t parity) {
  emu::Mbar& m = emu::cta_of(bar)->mbar(bar & 0xFFFFFFu);
  while (!m.test_wait(parity)) std::this_thread::yield();
}

template <int V> inline void ldg(F2 (&r)[V / 2], const float* p) { std::memcpy(&r[0], p, 4u * V); }
template <int V> inline void stg(float* p, const F2 (&r)[V / 2]) { std::memcpy(p, &r[0], 4u * V); }

}  // namespace zm
}  // namespace hsg
