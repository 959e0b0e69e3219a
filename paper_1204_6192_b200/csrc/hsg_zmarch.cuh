// hsg_zmarch.cuh — the fused z-marching sweep kernel.
//
// One launch runs a whole hsg_sweep(n_or, n_hb) call (at L = 32 and 16 the heat-bath sweeps are a second launch with
// fewer sites per thread, see zmarch_launch_g).  A CTA owns G configuration slots of ONE disorder
// sample and marches them together through the lattice planes z = 0..L-1, updating colour 0 of plane k
// and then colour 1 of plane k-1 in step k, so that every spin is read once and written once per sweep
// and the result is exactly the global two-colour sweep of PAPER.md:141-146 (colour 1 of a plane is
// updated only after colour 0 of the planes k-2, k-1, k has its new values; colour 1 of plane 0 is
// deferred to the last step because it needs the new colour 0 of plane L-1).
//
//   * Thread ownership: thread (y, j0) of a system owns the V compact sites j0..j0+V-1 of row y in BOTH
//     colours and in every plane.  All its global loads and stores go to its own column, so no
//     inter-thread ordering of global memory is ever needed; the z neighbours of a site are the thread's
//     own registers from the neighbouring steps.
//   * Spin planes are streamed global -> shared memory by per-thread cp.async copies of the thread's OWN
//     column, DS steps ahead of their use (rings C1 = old colour-1 planes, C0 = old colour-0 planes).
//     Completion is tracked per thread by cp.async groups, which (unlike register loads, whose scoreboard is
//     shared with younger loads) lets a step wait for the oldest stage while DS-1 younger ones stay in flight.
//   * In-plane neighbours (rows y-1, y+1 and the one x neighbour outside the thread's V sites) are read
//     from shared memory: ring C1 holds the old colour-1 spins of plane k, X0 (double-buffered) the new
//     colour-0 spins of plane k-1; one barrier per step.
//   * Couplings and fields of the sample stream through shared-memory rings filled by bulk async copies
//     (cp.async.bulk, mbarrier completion) issued DJ steps ahead, and are shared by the G systems of the CTA
//     (PAPER.md:161's R_TO idea).  Eleven of the twelve arrays of a plane live for two steps (ring A); the +z
//     couplings of colour 0 live for three (ring B).  Issuing a bulk copy costs its warp tens of cycles and the
//     whole CTA waits for its slowest warp at the step barrier, so the copies of a plane are issued by lane 0 of
//     different warps (two for a whole plane, four for a strip).
//   * Lattices whose planes do not fit one SM's shared memory (L = 64) are split into L/YS strips of YS rows;
//     the strips of a system group are the CTAs of one thread-block cluster.  Every shared spin array then
//     carries halo rows: the old colour-1 halo rows are fetched from global memory by the edge threads (the owner
//     overwrites them only two cluster barriers later), the new colour-0 halo rows are pushed into the
//     neighbour CTA's shared memory (st.async, counted on an mbarrier of that CTA) by the thread that computed
//     them, and the step barrier becomes a __syncthreads plus a split, relaxed cluster barrier (step_end / step_wait).
//     The J/H layout is strip-major (hsg_layout.cuh): two bulk copies per strip and plane, plus the two Jy rows below the strip.
//   * In the final sweep of a call the kernel also reduces E and m of every system.
#pragma once
#include <cuda_runtime.h>
#include "hsg_layout.cuh"
#include "hsg_math.cuh"
#include "hsg_zmarch_launch.h"
#include "hsg_zmarch_ptx.cuh"

namespace hsg {

namespace zm {

// Settled tuning of the march per lattice size (ncu evidence: profiles/).
//   YS   rows per strip (= L: the whole plane in one CTA; < L: L/YS strips = CTAs of a thread-block cluster)
//   V    compact sites per thread in the over-relaxation phase, VHB in the heat-bath phase; VHB != V: the heat-bath
//        sweeps of a call run as a second launch with more, lighter threads (they are bound by instruction issue, the
//        over-relaxation sweeps by memory)
//   GMAX most systems of one sample a CTA marches together (they share the J/H rings)
//   DS / DJ  spin / J-H planes in flight ahead of the step that uses them
template <int L> struct Tune;
template <> struct Tune<8>  { static constexpr int YS = 8,  V = 2, VHB = 2, GMAX = 8, DS = 2, DJ = 2; };
template <> struct Tune<16> { static constexpr int YS = 16, V = 4, VHB = 2, GMAX = 8, DS = 2, DJ = 2; };
template <> struct Tune<32> { static constexpr int YS = 32, V = 4, VHB = 2, GMAX = 2, DS = 2, DJ = 2; };
template <> struct Tune<64> { static constexpr int YS = 16, V = 4, VHB = 4, GMAX = 2, DS = 2, DJ = 2; };
constexpr int kUnroll = 2;     // unroll factor of the main march loop (over-relaxation / heat bath)
constexpr int kUnrollHB = 2;

template <int L, int YS, int V, int G> struct Cfg {
  static constexpr int Lh = L / 2;
  static constexpr int YSv = YS;
  static constexpr int NCL = L / YS;              // strips per lattice = CTAs per cluster
  static constexpr bool HALO = NCL > 1;
  static constexpr int TPR = Lh / V;              // threads per row
  static constexpr int TPS = YS * TPR;            // threads per system (strip)
  static constexpr int NT = G * TPS;              // threads per CTA
  static constexpr int CSG = L * Lh;              // one [y][j] array in global memory
  static constexpr int HPG = 3 * CSG;             // spin half-plane (one colour, 3 components) in global memory
  static constexpr int CSS = (YS + (HALO ? 2 : 0)) * Lh;   // shared spin array: halo row below, YS rows, halo row above
  static constexpr int HPS = 3 * CSS;
  static constexpr int CSJ = YS * Lh;             // shared J/H array of a strip
  static constexpr int JA = 11 * CSJ + (HALO ? 2 * Lh : 0);   // ring A slot: 11 arrays, then (strips) the row y0-1 of the two Jy
                                                              // arrays (colour 0, colour 1); ring B slot: colour-0 Jz
  static constexpr int DS = Tune<L>::DS;          // spin planes in flight ahead of the step that uses them
  static constexpr int DJ = Tune<L>::DJ;          // J/H planes in flight
  static constexpr int NC1 = DS + 2;              // ring C1: planes k, k+1 live + DS in flight
  static constexpr int NC0 = DS + 1;              // ring C0: plane k live + DS in flight
  static constexpr int NJA = DJ + 2;              // J/H ring A: planes k-1, k live + DJ in flight
  static constexpr int NJB = DJ + 3;              // J/H ring B: planes k-2, k-1, k live + DJ in flight; also the mbarrier ring
  static constexpr int CS0 = YS * Lh;             // ring C0 holds own columns only: no halo rows
  static constexpr int HP0 = 3 * CS0;
  static constexpr int RW = TPS < 32 ? TPS : 32;  // shuffle width of the per-system reduction
  static constexpr int WPS = TPS / RW;            // partial sums per system after the shuffle stage
  // byte offsets inside dynamic shared memory
  static constexpr uint32_t red_off = 64;         // [G][WPS][4] doubles (after NJB <= 6 J/H mbarriers and 2 halo mbarriers)
  static constexpr uint32_t red2_off = red_off + G * WPS * 32;        // [G][NCL][4] doubles: per-strip sums, used in rank 0
  static constexpr uint32_t ja_off = 128 * ((red2_off + G * NCL * 32 + 127) / 128);
  static constexpr uint32_t jb_off = ja_off + 4u * NJA * JA;
  static constexpr uint32_t sys_off = jb_off + 4u * NJB * CSJ;
  static constexpr uint32_t sys_bytes = 4u * ((NC1 + 2) * HPS + NC0 * HP0);    // per system: C1 ring, X0[2], C0 ring
  static constexpr size_t smem_bytes = sys_off + (size_t)G * sys_bytes;
  static_assert(L % YS == 0 && Lh % V == 0 && V % 2 == 0, "strip height divides L, even vector width divides the row length");
  static_assert((YS * Lh * 4) % 16 == 0 && (Lh * 4) % 16 == 0, "bulk copies move multiples of 16 bytes");
  static_assert(!HALO || V == 4, "halo copies use 16-byte cp.async.cg");
  static_assert(!HALO || YS >= 2, "a thread is on at most one strip edge");
  static_assert(NJB <= 6, "mbarrier area holds NJB J/H barriers and two halo barriers");
  static_assert(!HALO || DJ >= 2, "strip kernels: J/H ring depth 1 faulted at L = 64, G = 1 (round 1) and its cause is not established; only DJ >= 2 is validated");
  static constexpr uint32_t halo_bytes = G * 2u * 3u * Lh * 4u;   // new colour-0 halo rows received per step: both neighbours, G systems
  static_assert(smem_bytes <= 232448, "exceeds the 227 KB of shared memory per CTA");
};

// per-thread constants of the march
struct Th {
  int gy, j0;                 // global row, first compact site
  int grow;                   // gy * Lh + j0: element offset of the own column inside a global [y][j] array
  int grow_halo;              // HALO edge threads: element offset of the halo row they fetch (row gy-1 or gy+1, periodic)
  int edge;                   // HALO: -1 = lowest row of the strip, +1 = highest row, 0 = interior
  uint32_t row, rowp, rowm;   // byte offsets inside a shared [y][j] array: own row, row y+1, row y-1 at j0
  uint32_t row0;              // own row at j0 inside an array without halo rows (ring C0, J/H arrays)
  uint32_t jym0, jym1;        // J/H arrays: offset of row y-1 at j0 relative to the OTHER colour's Jy array, for the colour-0 /
                              // colour-1 update (strips: the lowest row reads the halo rows at the end of the ring slot)
  int lane_prev, lane_next;   // lanes of the threads that own the sites left / right of this thread's V sites in the same row
                              // (periodic; a row is TPR consecutive lanes of one warp): the x neighbour outside the thread's
                              // own sites is one of THEIR registers and travels by shuffle
  uint32_t lanes;             // shuffle mask: the lanes of this warp that exist
  uint32_t halo;              // HALO edge threads: byte offset of the halo row they fill (== rowm or rowp)
  uint32_t push;              // HALO edge threads: cluster address of X0[0], component 0, halo row at j0 in the neighbour CTA
  uint32_t push_bar;          // HALO edge threads: cluster address of the neighbour CTA's halo mbarrier of X0[0]
};

struct HbPar { float beta; uint32_t sysid, c1, c3; PhiloxKey key; };

// fp64 partial sums of one thread in the final sweep of a call:
// e = sum_{i in colour 1} s_i.h_i + sum_{i in colour 0} s_i.H_i  (= -E, site terms in fp32: DESIGN.md §3.6), m = sum_i s_i
struct EAcc { double e, mx, my, mz; };

// shared-memory addresses of the coupling / field arrays one colour update reads
struct JAddr {
  uint32_t own_xy;   // own colour, this plane: Jx at +0, Jy at +CJB  (bonds to +x, +y)
  uint32_t own_z;    // own colour, this plane: Jz                    (bond to +z)
  uint32_t own_h;    // own colour, this plane: Hx, Hy, Hz at +0, +CJB, +2CJB
  uint32_t oth_xy;   // other colour, this plane: Jx, Jy              (bonds from -x, -y)
  uint32_t oth_z;    // other colour, plane below: Jz                 (bond from -z)
  uint32_t ym;       // offset of row y-1 at j0 from the other colour's Jy array (th.jym0 / th.jym1)
};

// Local field of V sites of one colour in plane zp, accumulated in the order H, x+, x-, y+, y-, z+, z-
// (DESIGN.md §3.1), then the move; two sites per packed operation (hsg_math.cuh).  `q` = the thread's own column of the
// other colour in this plane, `xs` = shared-memory half-plane of the other colour in this plane (rows y+-1),
// `zlo`/`zhi` = own column of the other colour in planes zp-1 / zp+1.  The x neighbours of compact site j are the other
// colour's sites j-1+off and j+off of the same row: inside the thread's own V sites they are its registers `q`, the one
// outside is a register of the neighbouring lane (shuffle).  CSB / CJB = byte strides between the component arrays of a
// shared spin half-plane / between the arrays of a shared J/H plane.
// EN = 0: move only; 1: also accumulate s_i.H_i and s_i of the NEW spin (colour 0 in the final sweep);
// 2: s_i.h_i instead, the whole local field (colour 1 in the final sweep, when all its neighbours already hold their
// final values: every bond of the lattice once).
// FM: the heat-bath draw is the fast-math variant hb_draw_fast (HSG_FLAG_FAST_MATH), otherwise the reference arithmetic.
template <uint32_t CSB, uint32_t CJB, int V, bool HB, int EN, bool FM>
__device__ __forceinline__ void update_sites(F2 (&out)[3][V / 2], const F2 (&own)[3][V / 2], const F2 (&q)[3][V / 2],
                                             const F2 (&zlo)[3][V / 2], const F2 (&zhi)[3][V / 2], uint32_t xs,
                                             const JAddr& ja, const Th& th, int off, const HbPar& hp, uint32_t site0, EAcc& ea) {
  constexpr int NP = V / 2;
  const bool up = off != 0;
  const int src = up ? th.lane_next : th.lane_prev;        // the lane that owns the x neighbour outside this thread's sites
  // pair p of an array shifted by one site: towards higher j (x+ neighbours when off = 1), towards lower j (x- when off = 0)
  auto shifted = [&](const F2 (&v)[NP], float outside, int p) {
    const float lo = up ? f2_hi(v[p]) : (p > 0 ? f2_hi(v[p > 0 ? p - 1 : 0]) : outside);
    const float hi = up ? (p + 1 < NP ? f2_lo(v[p + 1 < NP ? p + 1 : 0]) : outside) : f2_lo(v[p]);
    return make_f2(lo, hi);
  };
  F2 Jxp[NP], Jxm[NP], Jyp[NP], Jym[NP], Jzp[NP], Jzm[NP];
  lds<V>(Jxp, ja.own_xy + th.row0);
  lds<V>(Jyp, ja.own_xy + CJB + th.row0);
  lds<V>(Jzp, ja.own_z + th.row0);
  {
    F2 t[NP];
    lds<V>(t, ja.oth_xy + th.row0);
    // the bond from x-1 is the +x coupling stored at the other colour's site j-1+off: the thread's own t[] when off = 1
    const float te = shfl_idx(th.lanes, f2_hi(t[NP - 1]), th.lane_prev);
#pragma unroll
    for (int p = 0; p < NP; ++p) Jxm[p] = up ? t[p] : shifted(t, te, p);
  }
  lds<V>(Jym, ja.oth_xy + CJB + ja.ym);
  lds<V>(Jzm, ja.oth_z + th.row0);
  F2 h[3][NP], Hs[3][NP];
  const uint32_t xs_p = xs + th.rowp, xs_m = xs + th.rowm;
#pragma unroll
  for (int mu = 0; mu < 3; ++mu) {
    F2 Hm[NP], yp[NP], ym[NP];
    lds<V>(Hm, ja.own_h + mu * CJB + th.row0);
    lds<V>(yp, xs_p + mu * CSB);
    lds<V>(ym, xs_m + mu * CSB);
    const float se = shfl_idx(th.lanes, up ? f2_lo(q[mu][0]) : f2_hi(q[mu][NP - 1]), src);
#pragma unroll
    for (int p = 0; p < NP; ++p) {
      const F2 sh = shifted(q[mu], se, p);
      const F2 sxp = up ? sh : q[mu][p];
      const F2 sxm = up ? q[mu][p] : sh;
      F2 acc = Hm[p];
      acc = fma_rn(Jxp[p], sxp, acc);
      acc = fma_rn(Jxm[p], sxm, acc);
      acc = fma_rn(Jyp[p], yp[p], acc);
      acc = fma_rn(Jym[p], ym[p], acc);
      acc = fma_rn(Jzp[p], zhi[mu][p], acc);
      acc = fma_rn(Jzm[p], zlo[mu][p], acc);
      h[mu][p] = acc;
      if (EN == 1) Hs[mu][p] = Hm[p];
    }
  }
#pragma unroll
  for (int p = 0; p < NP; ++p) {
    const V3<F2> hv = {h[0][p], h[1][p], h[2][p]};
    V3<F2> s;
    if (HB) {
      // heat bath: one Philox call per pair of sites (e, e+1), e even: counter word 0 = the site with even compact index
      // (j0 is a multiple of V), which takes output words 0, 1; its partner takes words 2, 3
      uint32_t w0, w1, w2, w3;
      philox4x32_10(site0 + 4u * (uint32_t)p, hp.c1, hp.sysid, hp.c3, hp.key.k0, hp.key.k1, w0, w1, w2, w3);
      if constexpr (FM) s = hb_draw_fast(hv, hp.beta, make_f2(u01(w0), u01(w2)), make_f2(u01(w1), u01(w3)));
      else s = hb_draw(hv, hp.beta, make_f2(u01(w0), u01(w2)), make_f2(u01(w1), u01(w3)));
    } else {
      const V3<F2> sv = {own[0][p], own[1][p], own[2][p]};
      s = or_reflect(sv, hv);
    }
    out[0][p] = s.x; out[1][p] = s.y; out[2][p] = s.z;
    if (EN >= 1) {
      const V3<F2> f = {EN == 2 ? h[0][p] : Hs[0][p], EN == 2 ? h[1][p] : Hs[1][p], EN == 2 ? h[2][p] : Hs[2][p]};
      const F2 sf = dot3(s, f);
      ea.e += (double)f2_lo(sf); ea.e += (double)f2_hi(sf);
      ea.mx += (double)f2_lo(s.x); ea.mx += (double)f2_hi(s.x);
      ea.my += (double)f2_lo(s.y); ea.my += (double)f2_hi(s.y);
      ea.mz += (double)f2_lo(s.z); ea.mz += (double)f2_hi(s.z);
    }
  }
}

// Shared state of one CTA during the march (32-bit shared-window addresses)
struct Smem {
  uint32_t full;       // [NJB] mbarriers of the J/H stream
  uint32_t hfull;      // [2] mbarriers: halo rows of X0[0], X0[1] have arrived from the neighbour strips
  uint32_t ja, jb;     // J/H rings A ([NJA][11 CSJ]) and B ([NJB][CSJ])
  uint32_t c1, c0;     // this thread's system: rings of old colour-1 / colour-0 half-planes
  uint32_t x0;         // this thread's system: [2][HPS] new colour-0 spins of planes k-1, k
  int y0;              // first row of this CTA's strip
};

struct Stream {        // J/H plane stream: index q -> plane (q-1) mod L
  int issued, waited, total;
};

// J/H stream: warp 0 keeps DJ planes in flight beyond the newest index `nd` this step reads; everyone waits for nd.
// Slot reuse is safe because the barrier that ended the previous step separates the last reads of index
// nd-2 (ring A) and nd-3 (ring B) from the copies issued here.  Whole-plane CTAs move a plane with two bulk copies;
// strip CTAs move the YS rows of each of the twelve arrays plus the halo row of the two Jy arrays (14 copies, one per lane).
template <class C, int L, class SmemT>
__device__ __forceinline__ void ring_advance(const SmemT& sm, const float* __restrict__ jh_d, Stream& st, int nd, uint64_t pol) {
  constexpr uint32_t JAB = 4u * C::JA, JBB = 4u * C::CSJ;
  // issuing a bulk copy costs its warp tens of cycles, and the CTA waits for its slowest warp at the step barrier: the
  // copies of a plane are issued by the first lanes of different warps (two for a whole plane, four for a strip)
  constexpr bool TWO = !C::HALO && C::NT > 32;
  constexpr bool FOUR = C::HALO && C::NT >= 128;
  if (FOUR ? ((tid_x() & 31u) == 0 && tid_x() < 128) : (tid_x() < 32 || (TWO && tid_x() == 32))) {
    const int upto = imin(nd + C::DJ, st.total - 1);
    while (st.issued < upto) {
      ++st.issued;
      const int plane = (st.issued + L - 1) % L;
      const uint32_t bar = sm.full + 8u * ((uint32_t)st.issued % C::NJB);
      const uint32_t dA = sm.ja + ((uint32_t)st.issued % C::NJA) * JAB, dB = sm.jb + ((uint32_t)st.issued % C::NJB) * JBB;
      const float* src = jh_d + (size_t)plane * 12 * C::CSG;
      if (!C::HALO) {
        if (tid_x() == 0) {
          mbar_expect_tx(bar, JAB + JBB);
          bulk_g2s(dA, src, JAB, bar, pol);
        }
        if (tid_x() == (TWO ? 32 : 0))     // (its complete_tx may land before the expect_tx: the phase still needs that arrive)
          bulk_g2s(dB, src + 11 * C::CSG, JBB, bar, pol);
      } else {
        // strip-major J/H layout (hsg_layout.cuh): the twelve arrays of this strip of the plane are contiguous; the row
        // y0-1 of the two Jy arrays comes from the last row of the strip below.  Four copies, one per lane.
        constexpr uint32_t ROWB = 4u * C::Lh, STRIPB = 4u * C::YSv * C::Lh;
        const int lane = FOUR ? (int)(tid_x() >> 5) : (int)tid_x();      // which of the four copies
        if (lane == 0)       // (a complete_tx that lands before this expect_tx is fine: the phase still needs the arrive)
          mbar_expect_tx(bar, 12u * STRIPB + 2u * ROWB);
        if (!FOUR) warp_sync();
        if (lane < 4) {
          const int strip = sm.y0 / C::YSv, below = (strip + C::NCL - 1) % C::NCL;
          const float* blk = src + (size_t)strip * 12 * C::CSJ;
          const float* blo = src + (size_t)below * 12 * C::CSJ + (size_t)(C::YSv - 1) * C::Lh;
          const uint32_t dst = lane == 0 ? dA : lane == 1 ? dB : dA + 11u * JBB + (uint32_t)(lane - 2) * ROWB;
          const float* from = lane == 0 ? blk : lane == 1 ? blk + 11 * C::CSJ : blo + (lane == 2 ? 1 : 6) * C::CSJ;
          const uint32_t bytes = lane == 0 ? 11u * STRIPB : lane == 1 ? STRIPB : ROWB;
          bulk_g2s(dst, from, bytes, bar, pol);
        }
      }
    }
  }
  while (st.waited < nd) {
    ++st.waited;
    const uint32_t bar = sm.full + 8u * ((uint32_t)st.waited % C::NJB);
    const uint32_t parity = ((uint32_t)st.waited / C::NJB) & 1u;
    mbar_wait(bar, parity);
  }
}

// The barrier that ends a step.  Inside the CTA it is a __syncthreads.  Between the strips of a cluster it is split:
// every thread ARRIVES at the end of step j and WAITS in step j+1 just before it publishes its new colour-0 spins, so a
// CTA runs up to half a step ahead of its neighbours.  What the cluster phase orders:
//   * my colour-1 reads of the halo X0[(j-1)&1] in step j (before my arrive) -> the neighbour's push into the same
//     buffer in step j+1 (after its wait);
//   * my fetch of an old colour-1 halo row (waited for at the top of step z-1) -> the owner's store of the new row in step z+1.
// Both are read-before-overwrite orders, so the per-step arrive is RELAXED (a releasing arrive would stall every step
// until the step's global stores are acknowledged).  The pushed halo rows themselves are ordered by their mbarrier
// (st.async complete_tx).  Only the last arrive of a sweep RELEASES, pairing with the acquiring wait of the next
// prologue: it makes the new colour-1 rows in global memory visible to the neighbour that fetches them as halo rows.
template <class C, bool RELEASE = false> __device__ __forceinline__ void step_end() {
  cta_sync();
  if (C::HALO) { if (RELEASE) cluster_arrive(); else cluster_arrive_relaxed(); }
}
template <class C> __device__ __forceinline__ void step_wait() {
  if (C::HALO) cluster_wait();
}

// One full sweep (both colours, all planes) of the G systems of this CTA.
template <int L, int YS, int V, int G, bool HB, bool EN, bool FM>
__device__ __forceinline__ void march_sweep(const Smem& sm, float* __restrict__ S, const float* __restrict__ jh_d,
                                            const Th& th, const HbPar& hp, int qbase, Stream& st, EAcc& ea,
                                            uint64_t pol_spin, uint64_t pol_jh, uint32_t& hph) {
  using C = Cfg<L, YS, V, G>;
  constexpr int CS = C::CSG, HP = C::HPG, PS = 2 * C::HPG;
  constexpr uint32_t CSB = 4u * C::CSS, HPB = 4u * C::HPS, CJB = 4u * C::CSJ, JAB = 4u * C::JA, JBB = 4u * C::CSJ;
  constexpr uint32_t CS0B = 4u * C::CS0, HP0B = 4u * C::HP0;
  constexpr bool HALO = C::HALO;
  constexpr int NP = V / 2;
  F2 A[3][NP], B[3][NP], Cc[3][NP], O[3][NP], P[3][NP], Q[3][NP], R[3][NP], On[3][NP];
  float* Sr = S + th.grow;                             // own column, plane 0, colour 0, component 0
  const float* Sh = S + th.grow_halo;                  // HALO edge threads: the halo row they fetch

  // old colour 1 of plane zc -> ring C1 slot `slot`: own column, plus the halo row of the strip's edge threads
  auto fetch_c1 = [&](int zc, int slot) {
    const uint32_t d1 = sm.c1 + (uint32_t)slot * HPB;
#pragma unroll
    for (int mu = 0; mu < 3; ++mu) {
      cp_async<V>(d1 + mu * CSB + th.row, Sr + zc * PS + HP + mu * CS, pol_spin);
      if (HALO && th.edge != 0) cp_async<V>(d1 + mu * CSB + th.halo, Sh + zc * PS + HP + mu * CS, pol_spin);
    }
  };
  // stage t = the planes step t consumes for the first time: old colour 1 of plane t+1 (ring C1, slot (t+1) % C::NC1)
  // and, for over-relaxation, old colour 0 of plane t (ring C0, slot t % C::NC0); own column only.
  auto issue_stage = [&](int t) {
    if (t < L) {
      fetch_c1((t + 1 == L) ? 0 : t + 1, (t + 1) % C::NC1);
      if (!HB) {
        const uint32_t d0 = sm.c0 + (uint32_t)(t % C::NC0) * HP0B + th.row0;
#pragma unroll
        for (int mu = 0; mu < 3; ++mu) cp_async<V>(d0 + mu * CS0B, Sr + t * PS + mu * CS, pol_spin);
      }
    }
    cp_async_commit();                                  // an empty group keeps the group count uniform
  };
  // new colour-0 spins of a plane -> X0[par] of this CTA and, from the strip's edge rows, the neighbour CTA's halo row
  auto publish_x0 = [&](uint32_t par, const F2 (&v)[3][NP]) {
#pragma unroll
    for (int mu = 0; mu < 3; ++mu) {
      sts<V>(sm.x0 + par * HPB + mu * CSB + th.row, v[mu]);
      if (HALO && th.edge != 0) st_async<V>(th.push + par * HPB + mu * CSB, v[mu], th.push_bar + 8u * par);
    }
  };
  // halo rows of X0[par]: thread 0 arms the mbarrier before the neighbours may push (they wait for this CTA's arrive of
  // the previous step), every thread waits for the bytes before the colour-1 update that reads them; bit `par` of hph
  // is the parity of the phase in flight
  auto arm_halo = [&](uint32_t par) {
    if (HALO && tid_x() == 0) mbar_expect_tx(sm.hfull + 8u * par, C::halo_bytes);
  };
  auto wait_halo = [&](uint32_t par) {
    if (HALO) { mbar_wait(sm.hfull + 8u * par, (hph >> par) & 1u); hph ^= 1u << par; }
  };

  // prologue: B = c1old(0) through ring slot 0 (the whole plane is needed there), A = c1old(L-1), stages 0..DS-1
  step_wait<C>();                                       // strips: the neighbours' stores of the previous sweep are visible
  fetch_c1(0, 0);
  cp_async_commit();
#pragma unroll
  for (int t = 0; t < C::DS; ++t) issue_stage(t);
#pragma unroll
  for (int mu = 0; mu < 3; ++mu) {
    ldg<V>(A[mu], Sr + (L - 1) * PS + HP + mu * CS);
#pragma unroll
    for (int e = 0; e < NP; ++e) { P[mu][e] = make_f2(0.0f, 0.0f); Q[mu][e] = P[mu][e]; O[mu][e] = P[mu][e]; On[mu][e] = P[mu][e]; }
  }
  cp_async_wait<C::DS>();
#pragma unroll
  for (int mu = 0; mu < 3; ++mu) lds<V>(B[mu], sm.c1 + mu * CSB + th.row);
  step_end<C>();
  // main steps: colour 0 of plane k, then colour 1 of plane k-1
#pragma unroll (EN ? 1 : (HB ? kUnrollHB : kUnroll))
  for (int k = 0; k < L; ++k) {
    const int nd = qbase + k + 1;                       // newest J/H stream index this step reads (plane k)
    ring_advance<C, L>(sm, jh_d, st, nd, pol_jh);
    arm_halo((uint32_t)(k & 1));
    cp_async_wait<C::DS - 1>();                           // stage k has landed (own column)
#pragma unroll
    for (int mu = 0; mu < 3; ++mu) {
      lds<V>(Cc[mu], sm.c1 + (uint32_t)((k + 1) % C::NC1) * HPB + mu * CSB + th.row);
      if (!HB) lds<V>(O[mu], sm.c0 + (uint32_t)(k % C::NC0) * HP0B + mu * CS0B + th.row0);
    }
    issue_stage(k + C::DS);
    if (k + 1 == L) {                                   // the new colour 0 of plane 0, needed by step L
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) ldg<V>(On[mu], Sr + mu * CS);
    }
    const int off = (th.gy + k) & 1;
    const uint32_t ak = sm.ja + ((uint32_t)nd % C::NJA) * JAB;                     // plane k
    const uint32_t ak1 = sm.ja + ((uint32_t)(nd + C::NJA - 1) % C::NJA) * JAB;       // plane k-1
    const uint32_t bk = sm.jb + ((uint32_t)nd % C::NJB) * JBB;                     // colour-0 Jz of plane k
    const uint32_t bk2 = sm.jb + ((uint32_t)(nd + C::NJB - 2) % C::NJB) * JBB;       // colour-0 Jz of plane k-2
    const uint32_t par = (uint32_t)(k & 1);
    {
      const uint32_t site0 = (uint32_t)(2 * th.j0 + off + L * (th.gy + L * k));
      const JAddr ja = {ak, bk, ak + 2 * CJB, ak + 5 * CJB, ak1 + 7 * CJB, th.jym0};
      update_sites<CSB, CJB, V, HB, EN ? 1 : 0, FM>(R, O, B, A, Cc, sm.c1 + (uint32_t)(k % C::NC1) * HPB, ja, th, off, hp, site0, ea);
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) stg<V>(Sr + k * PS + mu * CS, R[mu]);
      step_wait<C>();
      publish_x0(par, R);
    }
    if (k >= 1) wait_halo(par ^ 1u);                   // (step 0's rows are pushed again in the tail: consumed unread)
    if (k >= 2) {     // colour 1 of plane k-1
      const uint32_t site0 = (uint32_t)(2 * th.j0 + off + L * (th.gy + L * (k - 1)));
      const JAddr ja = {ak1 + 5 * CJB, ak1 + 7 * CJB, ak1 + 8 * CJB, ak1, bk2, th.jym1};
      F2 N1[3][NP];
      update_sites<CSB, CJB, V, HB, EN ? 2 : 0, FM>(N1, A, Q, P, R, sm.x0 + (par ^ 1u) * HPB, ja, th, off, hp, site0, ea);
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) stg<V>(Sr + (k - 1) * PS + HP + mu * CS, N1[mu]);
    }
    step_end<C>();
#pragma unroll
    for (int mu = 0; mu < 3; ++mu)
#pragma unroll
      for (int e = 0; e < NP; ++e) { A[mu][e] = B[mu][e]; B[mu][e] = Cc[mu][e]; P[mu][e] = Q[mu][e]; Q[mu][e] = R[mu][e]; }
  }
  cp_async_wait<0>();                                   // only empty groups are left
  // tail: colour 1 of plane L-1 (step L) and of plane 0 (step L+1); their z+ neighbours are the new colour-0
  // spins of planes 0 and 1, read back from the thread's own column
#pragma unroll 1
  for (int kk = 0; kk < 2; ++kk) {
    const int k = L + kk;
    const int nd = qbase + k;                            // plane k-1 (mod L)
    ring_advance<C, L>(sm, jh_d, st, nd, pol_jh);
#pragma unroll
    for (int mu = 0; mu < 3; ++mu)
#pragma unroll
      for (int e = 0; e < NP; ++e) R[mu][e] = On[mu][e];
    if (kk == 0) arm_halo(0u);
    step_wait<C>();
    if (kk == 0) {
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) ldg<V>(On[mu], Sr + PS + mu * CS);   // new colour 0 of plane 1, needed by step L+1
      publish_x0(0u, R);                                 // L is even: X0[L & 1] = X0[0] <- new colour 0 of plane 0
    }
    wait_halo((uint32_t)((k - 1) & 1));
    const int off = (th.gy + k) & 1;
    const uint32_t a1 = sm.ja + ((uint32_t)nd % C::NJA) * JAB;                     // plane k-1
    const uint32_t b2 = sm.jb + ((uint32_t)(nd + C::NJB - 1) % C::NJB) * JBB;        // colour-0 Jz of plane k-2
    const int z1 = kk == 0 ? L - 1 : 0;
    const uint32_t site0 = (uint32_t)(2 * th.j0 + off + L * (th.gy + L * z1));
    const JAddr ja = {a1 + 5 * CJB, a1 + 7 * CJB, a1 + 8 * CJB, a1, b2, th.jym1};
    F2 N1[3][NP];
    update_sites<CSB, CJB, V, HB, EN ? 2 : 0, FM>(N1, A, Q, P, R, sm.x0 + (uint32_t)((k - 1) & 1) * HPB, ja, th, off, hp, site0, ea);
#pragma unroll
    for (int mu = 0; mu < 3; ++mu) stg<V>(Sr + z1 * PS + HP + mu * CS, N1[mu]);
    if (kk == 1) step_end<C, true>();
    else step_end<C>();
#pragma unroll
    for (int mu = 0; mu < 3; ++mu)
#pragma unroll
      for (int e = 0; e < NP; ++e) { A[mu][e] = B[mu][e]; P[mu][e] = Q[mu][e]; Q[mu][e] = R[mu][e]; }
  }
}

template <int L, int YS, int V, int G, bool FM>
__global__ void __launch_bounds__(Cfg<L, YS, V, G>::NT, 1) zmarch_kernel(ZmarchArgs a) {
  using C = Cfg<L, YS, V, G>;
  HSG_DYN_SMEM(smem_raw);
  const uint32_t base = smem_u32(smem_raw);
  const int gs = tid_x() / C::TPS, tl = tid_x() % C::TPS;
  const int rank = C::HALO ? (int)cluster_ctarank() : 0;   // strip index
  const int group = C::HALO ? (int)(ctaid_x() / C::NCL) : (int)ctaid_x();
  Smem sm;
  sm.full = base;
  sm.hfull = base + 48;
  sm.ja = base + C::ja_off;
  sm.jb = base + C::jb_off;
  sm.c1 = base + C::sys_off + (uint32_t)gs * C::sys_bytes;
  sm.x0 = sm.c1 + 4u * C::NC1 * C::HPS;
  sm.c0 = sm.x0 + 4u * 2 * C::HPS;
  sm.y0 = rank * YS;
  if (tid_x() == 0) {
#pragma unroll
    for (int i = 0; i < C::NJB; ++i) mbar_init(reinterpret_cast<uint64_t*>(smem_raw) + i, 1);
    mbar_init(reinterpret_cast<uint64_t*>(smem_raw) + 6, 1);
    mbar_init(reinterpret_cast<uint64_t*>(smem_raw) + 7, 1);
    fence_mbarrier_init();
  }
  step_end<C, true>();                                   // strips: the first wait (in the prologue) sees every CTA of the cluster running

  constexpr int HR = C::HALO ? 1 : 0;                    // shared arrays keep local row r at row r + HR
  Th th;
  const int ly = tl / C::TPR;
  th.j0 = (tl % C::TPR) * V;
  th.gy = sm.y0 + ly;
  th.grow = th.gy * C::Lh + th.j0;
  th.row = 4u * (uint32_t)((ly + HR) * C::Lh + th.j0);
  th.row0 = 4u * (uint32_t)(ly * C::Lh + th.j0);
  if (C::HALO) {
    th.rowp = th.row + 4u * C::Lh;
    th.rowm = th.row - 4u * C::Lh;
    th.edge = (ly == 0) ? -1 : (ly == YS - 1 ? 1 : 0);
    const int hy = (th.gy + L + th.edge) % L;
    th.grow_halo = hy * C::Lh + th.j0;
    th.halo = th.edge < 0 ? th.rowm : th.rowp;
    // the new colour-0 spins of an edge row are the neighbour strip's halo row on its far side
    const uint32_t nb = (uint32_t)((rank + C::NCL + th.edge) % C::NCL);
    const uint32_t nb_row = 4u * (uint32_t)((th.edge < 0 ? YS + 1 : 0) * C::Lh + th.j0);
    th.push = th.edge != 0 ? mapa_u32(sm.x0 + nb_row, nb) : 0u;
    th.push_bar = th.edge != 0 ? mapa_u32(sm.hfull, nb) : 0u;
  } else {
    th.rowp = 4u * (uint32_t)(((ly + 1 == L) ? 0 : ly + 1) * C::Lh + th.j0);
    th.rowm = 4u * (uint32_t)(((ly == 0) ? L - 1 : ly - 1) * C::Lh + th.j0);
    th.edge = 0; th.grow_halo = 0; th.halo = 0; th.push = 0; th.push_bar = 0;
  }
  if (C::HALO && ly == 0) {       // row y0-1 of the other colour's Jy: halo rows behind the 11 arrays of the ring-A slot
    th.jym0 = 4u * (uint32_t)((11 - 6) * C::CSJ + C::Lh + th.j0);    // colour-0 update reads colour-1 Jy (array 6), halo row 1
    th.jym1 = 4u * (uint32_t)((11 - 1) * C::CSJ + th.j0);            // colour-1 update reads colour-0 Jy (array 1), halo row 0
  } else {
    th.jym0 = th.jym1 = 4u * (uint32_t)(((ly == 0) ? L - 1 : ly - 1) * C::Lh + th.j0);
  }
  {
    // the TPR threads of a row are consecutive lanes of one warp (TPR divides 32)
    static_assert(32 % C::TPR == 0 || C::TPR % 32 == 0, "a row occupies whole warps or a power-of-two part of one");
    static_assert(C::TPR <= 32, "a row must fit one warp: its x neighbours travel by shuffle");
    const int lane = (int)(tid_x() & 31u), first = lane & ~(C::TPR - 1);
    th.lane_prev = first | ((lane - 1) & (C::TPR - 1));
    th.lane_next = first | ((lane + 1) & (C::TPR - 1));
    th.lanes = C::NT >= 32 ? 0xffffffffu : ((1u << (C::NT & 31)) - 1u);
  }

  const Geom& g = a.g;
  const int slot = group * G + gs;                      // G consecutive slots of one sample
  const int d = slot / (g.O * g.T);
  const int grp = slot / g.T;
  const int t = a.temp_of_slot[slot];
  HbPar hp;
  hp.beta = a.beta[t];
  hp.sysid = (uint32_t)((g.sample_offset * g.O * g.T) + (unsigned long long)grp * g.T + t);
  hp.key = a.key;
  float* S = a.spins + (size_t)slot * 3 * g.N;
  const float* jh_d = a.jh + (size_t)d * 6 * g.N;
  const uint64_t pol_spin = policy_evict_first();       // spins stream through L2 once per sweep
  const uint64_t pol_jh = policy_evict_last();          // J/H of a sample are re-read by the CTAs of its O*T/G groups

  const int n_sweeps = a.n_or + a.n_hb;
  Stream st;
  st.issued = -1; st.waited = -1;
  st.total = n_sweeps * L + 2;                          // planes L-1, 0, 1, ..., L-1, 0, 1, ... (index q -> plane (q-1) mod L)
  EAcc ea = {0.0, 0.0, 0.0, 0.0};
  uint32_t hph = 0;                                     // phase parities of the two halo mbarriers
  const bool want_e = a.e_slot != nullptr;
  for (int s = 0; s < n_sweeps; ++s) {
    const bool fin = want_e && s + 1 == n_sweeps;       // the final sweep also reduces E and m
    if (s < a.n_or) {
      hp.c1 = 0; hp.c3 = 0;
      if (fin) march_sweep<L, YS, V, G, false, true, false>(sm, S, jh_d, th, hp, s * L, st, ea, pol_spin, pol_jh, hph);
      else march_sweep<L, YS, V, G, false, false, false>(sm, S, jh_d, th, hp, s * L, st, ea, pol_spin, pol_jh, hph);
    } else {
      const unsigned long long khb = a.k_hb + (unsigned long long)(s - a.n_or);
      hp.c1 = (uint32_t)(khb & 0xFFFFFFFFull); hp.c3 = counter_hi(khb, DOMAIN_HB);
      if (fin) march_sweep<L, YS, V, G, true, true, FM>(sm, S, jh_d, th, hp, s * L, st, ea, pol_spin, pol_jh, hph);
      else march_sweep<L, YS, V, G, true, false, FM>(sm, S, jh_d, th, hp, s * L, st, ea, pol_spin, pol_jh, hph);
    }
  }
  step_wait<C>();                                        // strips: nobody pushes into this CTA any more
  if (want_e) {
    // fixed-order reduction per system: lanes by shuffle, warps by one thread, strips by rank 0 (deterministic)
    constexpr int WPS = C::WPS, RW = C::RW;
    double v[4] = {ea.e, ea.mx, ea.my, ea.mz};
    double* red = reinterpret_cast<double*>(smem_raw + C::red_off);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
#pragma unroll
      for (int o = RW / 2; o > 0; o >>= 1) v[i] += shfl_down(th.lanes, v[i], o, RW);   // (th.lanes: a 16-thread CTA has half a warp)
    }
    if (tl % RW == 0) {
#pragma unroll
      for (int i = 0; i < 4; ++i) red[(gs * WPS + tl / RW) * 4 + i] = v[i];
    }
    cta_sync();
    double x = 0.0;
    if (tl < 4)
      for (int w = 0; w < WPS; ++w) x += red[(gs * WPS + w) * 4 + tl];
    if (C::HALO) {
      if (tl < 4) st_cluster_f64(mapa_u32(base + C::red2_off + 8u * (uint32_t)((gs * C::NCL + rank) * 4 + tl), 0u), x);
      cluster_arrive();
      cluster_wait();
      if (rank == 0 && tl < 4) {
        const double* red2 = reinterpret_cast<const double*>(smem_raw + C::red2_off);
        x = 0.0;
        for (int r = 0; r < C::NCL; ++r) x += red2[(gs * C::NCL + r) * 4 + tl];
      }
    }
    if (rank == 0 && tl < 4) {
      if (tl == 0) a.e_slot[slot] = -x;
      else a.m_slot[slot * 3 + (tl - 1)] = x / (double)g.N;
    }
  }
}

}  // namespace zm

}  // namespace hsg
