// emu.h — a small thread-for-thread execution model of one thread-block cluster on the host, for
// tests/test_zmarch_on_host.py: every CUDA thread is an OS thread; CTA barriers, warp shuffles, mbarriers with transaction
// counts, per-thread cp.async groups, bulk copies, remote (cluster) shared-memory stores and the split cluster barrier are
// modelled with their PTX semantics.  It is test infrastructure and knows nothing about spins.
//
// Asynchronous copies have no fixed landing time on the hardware — only "not before the issue, not after the wait".  The model
// runs in one of two MODES, the two ends of that window:
//   EARLY : the bytes move at the moment the copy is issued   -> a slot that is overwritten while somebody still needs its old
//           contents (write-after-read hazard of a ring) shows up as wrong data;
//   LATE  : the bytes move (and the source is read) only when a thread waits for them -> a read of data that was never
//           waited for, or a source overwritten before the copy landed (read-after-write / premature-reuse hazards), shows up.
// A protocol that gives the oracle's bits in both modes has no hazard the window can expose at this granularity.
#pragma once
#include <algorithm>
#include <atomic>
#include <condition_variable>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <deque>
#include <map>
#include <mutex>
#include <thread>
#include <vector>
#include <pthread.h>

namespace emu {

enum Mode { EARLY = 0, LATE = 1 };
inline int mode = EARLY;

struct Copy {            // one asynchronous transfer: plain copy, or an immediate value (remote store)
  unsigned char* dst; const unsigned char* src; uint32_t bytes; unsigned char imm[16]; bool has_imm;
  void land() const { std::memcpy(dst, has_imm ? imm : src, bytes); }
};

struct Mbar {            // mbarrier.shared::cta.b64 with transaction count
  std::mutex m;
  uint64_t completed = 0;   // phases completed so far; the phase in flight has parity completed & 1
  int init_count = 0, pending = 0;
  long tx = 0;
  std::vector<Copy> deferred;               // LATE mode: transfers not yet landed
  void check() { if (pending == 0 && tx == 0) { ++completed; pending = init_count; } }
  void init(int count) { std::lock_guard<std::mutex> g(m); init_count = pending = count; tx = 0; completed = 0; deferred.clear(); }
  void arrive_expect_tx(uint32_t bytes) { std::lock_guard<std::mutex> g(m); tx += bytes; --pending; check(); }
  void transfer(const Copy& c) {           // a copy that completes `bytes` of the transaction count
    std::lock_guard<std::mutex> g(m);
    if (mode == EARLY) { c.land(); tx -= c.bytes; check(); }
    else { deferred.push_back(c); }
  }
  bool test_wait(uint32_t parity) {        // mbarrier.try_wait.parity
    std::lock_guard<std::mutex> g(m);
    for (const Copy& c : deferred) { c.land(); tx -= c.bytes; check(); }
    deferred.clear();
    return (completed & 1u) != parity;
  }
};

struct Warp {
  pthread_barrier_t bar; double buf[32]; int lanes;
};

struct Cluster;
struct Cta {
  Cluster* cluster; int rank, nthreads; unsigned block_id;
  unsigned char* smem; size_t smem_bytes;
  pthread_barrier_t bar;
  std::map<uint32_t, Mbar> mbars;          // by byte offset inside smem (created before the threads start: see Launch)
  std::vector<Warp> warps;
  Mbar& mbar(uint32_t off) { return mbars.at(off); }
};

struct Cluster {
  std::vector<Cta*> ctas;
  std::mutex m; std::condition_variable cv;
  long arrived = 0, phase = 0, total = 0;   // barrier.cluster: arrive / wait are split
};

struct Thread {           // per-thread state
  Cta* cta = nullptr; unsigned tid = 0;
  std::deque<std::vector<Copy>> groups;     // committed cp.async groups not yet waited for (LATE mode)
  std::vector<Copy> open;                   // cp.async copies since the last commit
  long cluster_waited = 0;
};
inline thread_local Thread self;

// ---- shared-window addresses: low 24 bits = byte offset, bits 24.. = 1 + rank of the owning CTA (0: this CTA)
inline uint32_t addr_of(const void* p) { return (uint32_t)((const unsigned char*)p - self.cta->smem); }
inline Cta* cta_of(uint32_t a) { const uint32_t r = a >> 24; return r == 0 ? self.cta : self.cta->cluster->ctas.at(r - 1); }
inline unsigned char* ptr_of(uint32_t a) {
  Cta* c = cta_of(a); const uint32_t off = a & 0xFFFFFFu;
  if (off >= c->smem_bytes) { std::fprintf(stderr, "emu: shared-memory address %u out of range\n", off); std::abort(); }
  return c->smem + off;
}

inline void cta_sync() { pthread_barrier_wait(&self.cta->bar); }
inline Warp& my_warp() { return self.cta->warps[self.tid >> 5]; }
inline void warp_sync() { pthread_barrier_wait(&my_warp().bar); }
template <class T> inline T shuffle(T v, int src_lane) {
  Warp& w = my_warp(); const int lane = self.tid & 31;
  std::memcpy(&w.buf[lane], &v, sizeof(T));
  pthread_barrier_wait(&w.bar);
  T r = v;
  if (src_lane >= 0 && src_lane < w.lanes) std::memcpy(&r, &w.buf[src_lane], sizeof(T));
  pthread_barrier_wait(&w.bar);
  return r;
}

// ---- per-thread cp.async
inline void cp_async(uint32_t dst, const void* src, uint32_t bytes) {
  Copy c{ptr_of(dst), (const unsigned char*)src, bytes, {0}, false};
  if ((dst & (bytes - 1)) != 0 || ((uintptr_t)src & (bytes - 1)) != 0) { std::fprintf(stderr, "emu: misaligned cp.async\n"); std::abort(); }
  if (mode == EARLY) c.land(); else self.open.push_back(c);
}
inline void cp_async_commit() { if (mode == LATE) { self.groups.push_back(self.open); self.open.clear(); } }
inline void cp_async_wait(int n_pending_allowed) {
  while ((int)self.groups.size() > n_pending_allowed) { for (const Copy& c : self.groups.front()) c.land(); self.groups.pop_front(); }
}

// ---- cluster barrier
inline void cluster_arrive() {
  Cluster* cl = self.cta->cluster; std::lock_guard<std::mutex> g(cl->m);
  if (++cl->arrived == cl->total) { cl->arrived = 0; ++cl->phase; cl->cv.notify_all(); }
}
inline void cluster_wait() {
  Cluster* cl = self.cta->cluster; std::unique_lock<std::mutex> g(cl->m);
  const long want = ++self.cluster_waited;
  cl->cv.wait(g, [&] { return cl->phase >= want; });
}

// ---- launching one cluster: kernel(tid) runs on nthreads x n_cta OS threads
struct Launch {
  Cluster cl; std::vector<Cta> ctas;
  Launch(int n_cta, int nthreads, size_t smem_bytes, unsigned first_block, const std::vector<uint32_t>& mbar_offsets) : ctas(n_cta) {
    cl.total = (long)n_cta * nthreads;
    for (int r = 0; r < n_cta; ++r) {
      Cta& c = ctas[r];
      c.cluster = &cl; c.rank = r; c.nthreads = nthreads; c.block_id = first_block + r; c.smem_bytes = smem_bytes;
      c.smem = (unsigned char*)std::aligned_alloc(128, (smem_bytes + 127) / 128 * 128);
      std::memset(c.smem, 0xCD, smem_bytes);                    // poison: stale reads do not look like spins
      pthread_barrier_init(&c.bar, nullptr, nthreads);
      for (uint32_t off : mbar_offsets) c.mbars[off];            // nodes exist before any thread runs (no concurrent insertion)
      const int nw = (nthreads + 31) / 32;
      c.warps = std::vector<Warp>(nw);
      for (int w = 0; w < nw; ++w) { c.warps[w].lanes = std::min(32, nthreads - 32 * w); pthread_barrier_init(&c.warps[w].bar, nullptr, c.warps[w].lanes); }
      cl.ctas.push_back(&c);
    }
  }
  ~Launch() { for (Cta& c : ctas) std::free(c.smem); }
  template <class F> void run(F kernel) {
    std::vector<std::thread> th;
    for (Cta& c : ctas)
      for (int t = 0; t < c.nthreads; ++t)
        th.emplace_back([&c, t, kernel] { self = Thread(); self.cta = &c; self.tid = (unsigned)t; kernel(); });
    for (auto& x : th) x.join();
  }
};

}  // namespace emu
