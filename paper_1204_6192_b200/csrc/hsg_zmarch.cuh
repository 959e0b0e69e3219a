// hsg_zmarch.cuh — the fused z-marching sweep kernel.
//
// One launch runs a whole hsg_sweep(n_or, n_hb) call.  A CTA owns G configuration slots of ONE disorder
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
//     shared with younger loads) lets a step wait for the oldest stage while DS-1 younger ones stay in
//     flight: the bytes in flight per SM, not the issue rate, bound this kernel (Little's law).
//   * In-plane neighbours (rows y-1, y+1 and the one x neighbour outside the thread's V sites) are read
//     from shared memory: ring C1 holds the old colour-1 spins of plane k, X0 (double-buffered) the new
//     colour-0 spins of plane k-1; one __syncthreads per step.
//   * Couplings and fields of the sample stream through shared-memory rings filled by bulk async copies
//     (cp.async.bulk, mbarrier completion) issued DJ steps ahead by thread 0, and are shared by the G
//     systems of the CTA (PAPER.md:161's R_TO idea).  Eleven of the twelve arrays of a plane live for two
//     steps (ring A); the +z couplings of colour 0 live for three (ring B).
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
};

namespace zm {

#ifndef HSG_ZM_UNROLL
#define HSG_ZM_UNROLL 2
#endif
#ifndef HSG_ZM_L32_V
#define HSG_ZM_L32_V 4
#endif
#ifndef HSG_ZM_L32_G
#define HSG_ZM_L32_G 2
#endif
#ifndef HSG_ZM_L16_V
#define HSG_ZM_L16_V 4
#endif
#ifndef HSG_ZM_DS
#define HSG_ZM_DS 2              // spin planes in flight ahead of the step that uses them
#endif
#ifndef HSG_ZM_DJ
#define HSG_ZM_DJ 2              // J/H planes in flight ahead of the step that uses them
#endif
#ifndef HSG_ZM_UNROLL_HB
#define HSG_ZM_UNROLL_HB 2
#endif
constexpr int kUnroll = HSG_ZM_UNROLL;   // unroll factor of the main march loop
constexpr int kUnrollHB = HSG_ZM_UNROLL_HB;
constexpr int kDS = HSG_ZM_DS, kDJ = HSG_ZM_DJ;
constexpr int kNC1 = kDS + 2;            // ring C1: planes k, k+1 live + DS in flight
constexpr int kNC0 = kDS + 1;            // ring C0: plane k live + DS in flight
constexpr int kNJA = kDJ + 2;            // J/H ring A: planes k-1, k live + DJ in flight
constexpr int kNJB = kDJ + 3;            // J/H ring B: planes k-2, k-1, k live + DJ in flight; also the mbarrier ring

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

// ---------------------------------------------------------------- V-wide vector access (V = 2 or 4 floats)
template <int V> struct VT;
template <> struct VT<2> { using type = float2; };
template <> struct VT<4> { using type = float4; };

// shared memory by 32-bit shared-window byte address (keeps all address arithmetic 32-bit)
template <int V> __device__ __forceinline__ void lds(float (&r)[V], uint32_t a);
template <> __device__ __forceinline__ void lds<2>(float (&r)[2], uint32_t a) {
  asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(r[0]), "=f"(r[1]) : "r"(a) : "memory");
}
template <> __device__ __forceinline__ void lds<4>(float (&r)[4], uint32_t a) {
  asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3]) : "r"(a) : "memory");
}
__device__ __forceinline__ float lds1(uint32_t a) {
  float r;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(r) : "r"(a) : "memory");
  return r;
}
template <int V> __device__ __forceinline__ void sts(uint32_t a, const float (&r)[V]);
template <> __device__ __forceinline__ void sts<2>(uint32_t a, const float (&r)[2]) {
  asm volatile("st.shared.v2.f32 [%0], {%1,%2};" ::"r"(a), "f"(r[0]), "f"(r[1]) : "memory");
}
template <> __device__ __forceinline__ void sts<4>(uint32_t a, const float (&r)[4]) {
  asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(a), "f"(r[0]), "f"(r[1]), "f"(r[2]), "f"(r[3]) : "memory");
}
// streaming global access for the spins: each value is touched once per sweep
template <int V> __device__ __forceinline__ void ldg(float (&r)[V], const float* p) {
  const typename VT<V>::type t = __ldcs(reinterpret_cast<const typename VT<V>::type*>(p));
  const float* f = reinterpret_cast<const float*>(&t);
#pragma unroll
  for (int e = 0; e < V; ++e) r[e] = f[e];
}
template <int V> __device__ __forceinline__ void stg(float* p, const float (&r)[V]) {
  typename VT<V>::type t;
  float* f = reinterpret_cast<float*>(&t);
#pragma unroll
  for (int e = 0; e < V; ++e) f[e] = r[e];
  __stcs(reinterpret_cast<typename VT<V>::type*>(p), t);
}

template <int L, int V, int G> struct Cfg {
  static constexpr int Lh = L / 2;
  static constexpr int TPR = Lh / V;              // threads per row
  static constexpr int TPS = L * TPR;             // threads per system
  static constexpr int NT = G * TPS;              // threads per CTA
  static constexpr int CS = L * Lh;               // one [y][j] array
  static constexpr int HP = 3 * CS;               // spin half-plane (one colour, 3 components)
  static constexpr int JP = 12 * CS;              // J/H plane: 11 arrays for ring A + colour-0 Jz for ring B
  static constexpr int JA = 11 * CS;
  static constexpr int RW = TPS < 32 ? TPS : 32;  // shuffle width of the per-system reduction
  static constexpr int WPS = TPS / RW;            // partial sums per system after the shuffle stage
  // byte offsets inside dynamic shared memory
  static constexpr uint32_t red_off = 64;         // [G][WPS][4] doubles (after kNJB <= 8 mbarriers)
  static constexpr uint32_t ja_off = 64 + 128 * ((G * WPS * 32 + 127) / 128);
  static constexpr uint32_t jb_off = ja_off + 4u * kNJA * JA;
  static constexpr uint32_t sys_off = jb_off + 4u * kNJB * CS;
  static constexpr uint32_t sys_bytes = 4u * (kNC1 + kNC0 + 2) * HP;     // per system: C1 ring, C0 ring, X0[2]
  static constexpr size_t smem_bytes = sys_off + (size_t)G * sys_bytes;
  static_assert(Lh % V == 0, "row length must be a multiple of the vector width");
  static_assert((CS * 4) % 16 == 0, "bulk copies move multiples of 16 bytes");
  static_assert(kNJB <= 8, "mbarrier area holds 8 barriers");
};

// per-thread constants of the march (byte offsets inside a [y][j] array)
struct Th {
  int y, j0;
  uint32_t row, rowp, rowm;   // own row, row y+1, row y-1 (periodic) at j0
  uint32_t edge0, edge1;      // own row at j0-1 and j0+V (periodic): the x neighbour outside the thread's V sites
};

struct HbPar { float beta; uint32_t sysid, c1, c3; PhiloxKey key; };

// fp64 partial sums of one thread in the final sweep of a call:
// e = sum_{i in colour 1} s_i.(sum_6 J_ij s_j) + sum_i H_i.s_i  (= -E), m = sum_i s_i; exact fp32 x fp32 products
struct EAcc { double e, mx, my, mz; };

// shared-memory addresses of the coupling / field arrays one colour update reads
struct JAddr {
  uint32_t own_xy;   // own colour, this plane: Jx at +0, Jy at +CSB  (bonds to +x, +y)
  uint32_t own_z;    // own colour, this plane: Jz                    (bond to +z)
  uint32_t own_h;    // own colour, this plane: Hx, Hy, Hz at +0, +CSB, +2CSB
  uint32_t oth_xy;   // other colour, this plane: Jx, Jy              (bonds from -x, -y)
  uint32_t oth_z;    // other colour, plane below: Jz                 (bond from -z)
};

// Local field of V sites of one colour in plane zp, accumulated in the order H, x+, x-, y+, y-, z+, z-
// (DESIGN.md §3.1), then the move.  `q` = the thread's own column of the other colour in this plane,
// `xs` = shared-memory half-plane of the other colour in this plane (rows y+-1 and the x edge),
// `zlo`/`zhi` = own column of the other colour in planes zp-1 / zp+1.
// EN = 0: move only; 1: also accumulate H_i.s_i and s_i of the NEW spin (colour 0 in the final sweep);
// 2: additionally s_i.(sum_6 J_ij s_j) with every bond of the site (colour 1 in the final sweep, when all its
// neighbours already hold their final values).
template <int L, int V, bool HB, int EN>
__device__ __forceinline__ void update_sites(float (&out)[3][V], const float (&own)[3][V], const float (&q)[3][V],
                                             const float (&zlo)[3][V], const float (&zhi)[3][V], uint32_t xs,
                                             const JAddr& ja, const Th& th, int off, const HbPar& hp, uint32_t site0, EAcc& ea) {
  constexpr uint32_t CSB = 4u * L * (L / 2);
  const uint32_t edge = off ? th.edge1 : th.edge0;
  float Jxp[V], Jxm[V], Jyp[V], Jym[V], Jzp[V], Jzm[V];
  lds<V>(Jxp, ja.own_xy + th.row);
  lds<V>(Jyp, ja.own_xy + CSB + th.row);
  lds<V>(Jzp, ja.own_z + th.row);
  {
    float t[V];
    lds<V>(t, ja.oth_xy + th.row);
    const float te = lds1(ja.oth_xy + th.edge0);
#pragma unroll
    for (int e = 0; e < V; ++e) Jxm[e] = off ? t[e] : (e > 0 ? t[e > 0 ? e - 1 : 0] : te);
  }
  lds<V>(Jym, ja.oth_xy + CSB + th.rowm);
  lds<V>(Jzm, ja.oth_z + th.row);
  float h[3][V];
  float Hs[3][V];
  double hd[3][V];
  const uint32_t xs_p = xs + th.rowp, xs_m = xs + th.rowm, xs_e = xs + edge;
#pragma unroll
  for (int mu = 0; mu < 3; ++mu) {
    float Hm[V], yp[V], ym[V];
    lds<V>(Hm, ja.own_h + mu * CSB + th.row);
    lds<V>(yp, xs_p + mu * CSB);
    lds<V>(ym, xs_m + mu * CSB);
    const float se = lds1(xs_e + mu * CSB);
#pragma unroll
    for (int e = 0; e < V; ++e) {
      const float sxp = off ? (e + 1 < V ? q[mu][e + 1 < V ? e + 1 : 0] : se) : q[mu][e];
      const float sxm = off ? q[mu][e] : (e > 0 ? q[mu][e > 0 ? e - 1 : 0] : se);
      float acc = Hm[e];
      acc = __fmaf_rn(Jxp[e], sxp, acc);
      acc = __fmaf_rn(Jxm[e], sxm, acc);
      acc = __fmaf_rn(Jyp[e], yp[e], acc);
      acc = __fmaf_rn(Jym[e], ym[e], acc);
      acc = __fmaf_rn(Jzp[e], zhi[mu][e], acc);
      acc = __fmaf_rn(Jzm[e], zlo[mu][e], acc);
      h[mu][e] = acc;
      if (EN >= 1) Hs[mu][e] = Hm[e];
      if (EN == 2) {
        double d = (double)Jxp[e] * (double)sxp;
        d = fma((double)Jxm[e], (double)sxm, d);
        d = fma((double)Jyp[e], (double)yp[e], d);
        d = fma((double)Jym[e], (double)ym[e], d);
        d = fma((double)Jzp[e], (double)zhi[mu][e], d);
        d = fma((double)Jzm[e], (double)zlo[mu][e], d);
        hd[mu][e] = d;
      }
    }
  }
#pragma unroll
  for (int e = 0; e < V; ++e) {
    const Vec3 hv = {h[0][e], h[1][e], h[2][e]};
    Vec3 s;
    if (HB) {
      uint32_t w0, w1, w2, w3;
      philox4x32_10(site0 + 2u * (uint32_t)e, hp.c1, hp.sysid, hp.c3, hp.key.k0, hp.key.k1, w0, w1, w2, w3);
      s = hb_draw(hv, hp.beta, u01(w0), u01(w1));
    } else {
      const Vec3 sv = {own[0][e], own[1][e], own[2][e]};
      s = or_reflect(sv, hv);
    }
    out[0][e] = s.x; out[1][e] = s.y; out[2][e] = s.z;
    if (EN >= 1) {
      const double sx = (double)s.x, sy = (double)s.y, sz = (double)s.z;
      double d = (double)Hs[0][e] * sx;
      d = fma((double)Hs[1][e], sy, d);
      d = fma((double)Hs[2][e], sz, d);
      if (EN == 2) {
        d = fma(hd[0][e], sx, d);
        d = fma(hd[1][e], sy, d);
        d = fma(hd[2][e], sz, d);
      }
      ea.e += d; ea.mx += sx; ea.my += sy; ea.mz += sz;
    }
  }
}

// Shared state of one CTA during the march (32-bit shared-window addresses)
struct Smem {
  uint32_t full;       // [kNJB] mbarriers
  uint32_t ja, jb;     // J/H rings A ([kNJA][11 CS]) and B ([kNJB][CS])
  uint32_t c1, c0;     // this thread's system: rings of old colour-1 / colour-0 half-planes
  uint32_t x0;         // this thread's system: [2][HP] new colour-0 spins of planes k-1, k
};

struct Stream {        // J/H plane stream: index q -> plane (q-1) mod L
  int issued, waited, total;
};

// J/H stream: thread 0 keeps kDJ planes in flight beyond the newest index `nd` this step reads; everyone waits for nd.
// Slot reuse is safe because the __syncthreads that ended the previous step separates the last reads of index
// nd-2 (ring A) and nd-3 (ring B) from the copies issued here.
template <int L, int CS>
__device__ __forceinline__ void ring_advance(const Smem& sm, const float* __restrict__ jh_d, Stream& st, int nd, uint64_t pol) {
  constexpr uint32_t JAB = 44u * CS, JBB = 4u * CS;
  if (threadIdx.x == 0) {
    const int upto = min(nd + kDJ, st.total - 1);
    while (st.issued < upto) {
      ++st.issued;
      const int plane = (st.issued + L - 1) % L;
      const uint32_t bar = sm.full + 8u * ((uint32_t)st.issued % kNJB);
      const float* src = jh_d + (size_t)plane * 12 * CS;
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(JAB + JBB) : "memory");
      asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                   ::"r"(sm.ja + ((uint32_t)st.issued % kNJA) * JAB), "l"(src), "r"(JAB), "r"(bar), "l"(pol) : "memory");
      asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                   ::"r"(sm.jb + ((uint32_t)st.issued % kNJB) * JBB), "l"(src + 11 * CS), "r"(JBB), "r"(bar), "l"(pol) : "memory");
    }
  }
  while (st.waited < nd) {
    ++st.waited;
    const uint32_t bar = sm.full + 8u * ((uint32_t)st.waited % kNJB);
    const uint32_t parity = ((uint32_t)st.waited / kNJB) & 1u;
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
}

// One full sweep (both colours, all planes) of the G systems of this CTA.
template <int L, int V, int G, bool HB, bool EN>
__device__ __forceinline__ void march_sweep(const Smem& sm, float* __restrict__ S, const float* __restrict__ jh_d,
                                            const Th& th, const HbPar& hp, int qbase, Stream& st, EAcc& ea,
                                            uint64_t pol_spin, uint64_t pol_jh) {
  using C = Cfg<L, V, G>;
  constexpr int CS = C::CS, HP = C::HP, PS = 2 * C::HP;
  constexpr uint32_t CSB = 4u * CS, HPB = 4u * HP, JAB = 44u * CS, JBB = 4u * CS;
  float A[3][V], B[3][V], Cc[3][V], O[3][V], P[3][V], Q[3][V], R[3][V], On[3][V];
  float* Sr = S + (th.row >> 2);                       // own column, plane 0, colour 0, component 0

  // stage t = the planes step t consumes for the first time: old colour 1 of plane t+1 (ring C1, slot (t+1) % kNC1)
  // and, for over-relaxation, old colour 0 of plane t (ring C0, slot t % kNC0); own column only.
  auto issue_stage = [&](int t) {
    if (t < L) {
      const int zc = (t + 1 == L) ? 0 : t + 1;
      const uint32_t d1 = sm.c1 + (uint32_t)((t + 1) % kNC1) * HPB + th.row;
      const uint32_t d0 = sm.c0 + (uint32_t)(t % kNC0) * HPB + th.row;
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) {
        cp_async<V>(d1 + mu * CSB, Sr + zc * PS + HP + mu * CS, pol_spin);
        if (!HB) cp_async<V>(d0 + mu * CSB, Sr + t * PS + mu * CS, pol_spin);
      }
    }
    cp_async_commit();                                  // an empty group keeps the group count uniform
  };

  // prologue: B = c1old(0) through ring slot 0 (the whole plane is needed there), A = c1old(L-1), stages 0..DS-1
#pragma unroll
  for (int mu = 0; mu < 3; ++mu) cp_async<V>(sm.c1 + mu * CSB + th.row, Sr + HP + mu * CS, pol_spin);
  cp_async_commit();
#pragma unroll
  for (int t = 0; t < kDS; ++t) issue_stage(t);
#pragma unroll
  for (int mu = 0; mu < 3; ++mu) {
    ldg<V>(A[mu], Sr + (L - 1) * PS + HP + mu * CS);
#pragma unroll
    for (int e = 0; e < V; ++e) { P[mu][e] = 0.0f; Q[mu][e] = 0.0f; O[mu][e] = 0.0f; On[mu][e] = 0.0f; }
  }
  cp_async_wait<kDS>();
#pragma unroll
  for (int mu = 0; mu < 3; ++mu) lds<V>(B[mu], sm.c1 + mu * CSB + th.row);
  __syncthreads();
  // main steps: colour 0 of plane k, then colour 1 of plane k-1
#pragma unroll (EN ? 1 : (HB ? kUnrollHB : kUnroll))
  for (int k = 0; k < L; ++k) {
    const int nd = qbase + k + 1;                       // newest J/H stream index this step reads (plane k)
    ring_advance<L, CS>(sm, jh_d, st, nd, pol_jh);
    cp_async_wait<kDS - 1>();                           // stage k has landed (own column)
#pragma unroll
    for (int mu = 0; mu < 3; ++mu) {
      lds<V>(Cc[mu], sm.c1 + (uint32_t)((k + 1) % kNC1) * HPB + mu * CSB + th.row);
      if (!HB) lds<V>(O[mu], sm.c0 + (uint32_t)(k % kNC0) * HPB + mu * CSB + th.row);
    }
    issue_stage(k + kDS);
    if (k + 1 == L) {                                   // the new colour 0 of plane 0, needed by step L
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) ldg<V>(On[mu], Sr + mu * CS);
    }
    const int off = (th.y + k) & 1;
    const uint32_t ak = sm.ja + ((uint32_t)nd % kNJA) * JAB;                     // plane k
    const uint32_t ak1 = sm.ja + ((uint32_t)(nd + kNJA - 1) % kNJA) * JAB;       // plane k-1
    const uint32_t bk = sm.jb + ((uint32_t)nd % kNJB) * JBB;                     // colour-0 Jz of plane k
    const uint32_t bk2 = sm.jb + ((uint32_t)(nd + kNJB - 2) % kNJB) * JBB;       // colour-0 Jz of plane k-2
    const uint32_t par = (uint32_t)(k & 1);
    {
      const uint32_t site0 = (uint32_t)(2 * th.j0 + off + L * (th.y + L * k));
      const JAddr ja = {ak, bk, ak + 2 * CSB, ak + 5 * CSB, ak1 + 7 * CSB};
      update_sites<L, V, HB, EN ? 1 : 0>(R, O, B, A, Cc, sm.c1 + (uint32_t)(k % kNC1) * HPB, ja, th, off, hp, site0, ea);
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) {
        stg<V>(Sr + k * PS + mu * CS, R[mu]);
        sts<V>(sm.x0 + par * HPB + mu * CSB + th.row, R[mu]);
      }
    }
    if (k >= 2) {     // colour 1 of plane k-1
      const uint32_t site0 = (uint32_t)(2 * th.j0 + off + L * (th.y + L * (k - 1)));
      const JAddr ja = {ak1 + 5 * CSB, ak1 + 7 * CSB, ak1 + 8 * CSB, ak1, bk2};
      float N1[3][V];
      update_sites<L, V, HB, EN ? 2 : 0>(N1, A, Q, P, R, sm.x0 + (par ^ 1u) * HPB, ja, th, off, hp, site0, ea);
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) stg<V>(Sr + (k - 1) * PS + HP + mu * CS, N1[mu]);
    }
    __syncthreads();
#pragma unroll
    for (int mu = 0; mu < 3; ++mu)
#pragma unroll
      for (int e = 0; e < V; ++e) { A[mu][e] = B[mu][e]; B[mu][e] = Cc[mu][e]; P[mu][e] = Q[mu][e]; Q[mu][e] = R[mu][e]; }
  }
  cp_async_wait<0>();                                   // only empty groups are left
  // tail: colour 1 of plane L-1 (step L) and of plane 0 (step L+1); their z+ neighbours are the new colour-0
  // spins of planes 0 and 1, read back from the thread's own column
#pragma unroll 1
  for (int kk = 0; kk < 2; ++kk) {
    const int k = L + kk;
    const int nd = qbase + k;                            // plane k-1 (mod L)
    ring_advance<L, CS>(sm, jh_d, st, nd, pol_jh);
#pragma unroll
    for (int mu = 0; mu < 3; ++mu)
#pragma unroll
      for (int e = 0; e < V; ++e) R[mu][e] = On[mu][e];
    if (kk == 0) {
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) {
        ldg<V>(On[mu], Sr + PS + mu * CS);               // new colour 0 of plane 1, needed by step L+1
        sts<V>(sm.x0 + mu * CSB + th.row, R[mu]);         // L is even: X0[L & 1] = X0[0] <- new colour 0 of plane 0
      }
    }
    const int off = (th.y + k) & 1;
    const uint32_t a1 = sm.ja + ((uint32_t)nd % kNJA) * JAB;                     // plane k-1
    const uint32_t b2 = sm.jb + ((uint32_t)(nd + kNJB - 1) % kNJB) * JBB;        // colour-0 Jz of plane k-2
    const int z1 = kk == 0 ? L - 1 : 0;
    const uint32_t site0 = (uint32_t)(2 * th.j0 + off + L * (th.y + L * z1));
    const JAddr ja = {a1 + 5 * CSB, a1 + 7 * CSB, a1 + 8 * CSB, a1, b2};
    float N1[3][V];
    update_sites<L, V, HB, EN ? 2 : 0>(N1, A, Q, P, R, sm.x0 + (uint32_t)((k - 1) & 1) * HPB, ja, th, off, hp, site0, ea);
#pragma unroll
    for (int mu = 0; mu < 3; ++mu) stg<V>(Sr + z1 * PS + HP + mu * CS, N1[mu]);
    __syncthreads();
#pragma unroll
    for (int mu = 0; mu < 3; ++mu)
#pragma unroll
      for (int e = 0; e < V; ++e) { A[mu][e] = B[mu][e]; P[mu][e] = Q[mu][e]; Q[mu][e] = R[mu][e]; }
  }
}

template <int L, int V, int G>
__global__ void __launch_bounds__(Cfg<L, V, G>::NT, 1) zmarch_kernel(ZmarchArgs a) {
  using C = Cfg<L, V, G>;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const uint32_t base = smem_u32(smem_raw);
  const int gs = threadIdx.x / C::TPS, tl = threadIdx.x % C::TPS;
  Smem sm;
  sm.full = base;
  sm.ja = base + C::ja_off;
  sm.jb = base + C::jb_off;
  sm.c1 = base + C::sys_off + (uint32_t)gs * C::sys_bytes;
  sm.c0 = sm.c1 + 4u * kNC1 * C::HP;
  sm.x0 = sm.c0 + 4u * kNC0 * C::HP;
  if (threadIdx.x == 0) {
#pragma unroll
    for (int i = 0; i < kNJB; ++i) mbar_init(reinterpret_cast<uint64_t*>(smem_raw) + i, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  Th th;
  th.y = tl / C::TPR; th.j0 = (tl % C::TPR) * V;
  th.row = 4u * (uint32_t)(th.y * C::Lh + th.j0);
  th.rowp = 4u * (uint32_t)(((th.y + 1 == L) ? 0 : th.y + 1) * C::Lh + th.j0);
  th.rowm = 4u * (uint32_t)(((th.y == 0) ? L - 1 : th.y - 1) * C::Lh + th.j0);
  th.edge0 = 4u * (uint32_t)(th.y * C::Lh + ((th.j0 == 0) ? C::Lh - 1 : th.j0 - 1));
  th.edge1 = 4u * (uint32_t)(th.y * C::Lh + ((th.j0 + V == C::Lh) ? 0 : th.j0 + V));

  const Geom& g = a.g;
  const int slot = blockIdx.x * G + gs;                 // G consecutive slots of one sample
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
  const bool want_e = a.e_slot != nullptr;
  for (int s = 0; s < n_sweeps; ++s) {
    const bool fin = want_e && s + 1 == n_sweeps;       // the final sweep also reduces E and m
    if (s < a.n_or) {
      hp.c1 = 0; hp.c3 = 0;
      if (fin) march_sweep<L, V, G, false, true>(sm, S, jh_d, th, hp, s * L, st, ea, pol_spin, pol_jh);
      else march_sweep<L, V, G, false, false>(sm, S, jh_d, th, hp, s * L, st, ea, pol_spin, pol_jh);
    } else {
      const unsigned long long khb = a.k_hb + (unsigned long long)(s - a.n_or);
      hp.c1 = (uint32_t)(khb & 0xFFFFFFFFull); hp.c3 = counter_hi(khb, DOMAIN_HB);
      if (fin) march_sweep<L, V, G, true, true>(sm, S, jh_d, th, hp, s * L, st, ea, pol_spin, pol_jh);
      else march_sweep<L, V, G, true, false>(sm, S, jh_d, th, hp, s * L, st, ea, pol_spin, pol_jh);
    }
  }
  if (want_e) {
    // fixed-order reduction per system: lanes by shuffle, warps by one thread (deterministic)
    constexpr int WPS = C::WPS, RW = C::RW;
    double v[4] = {ea.e, ea.mx, ea.my, ea.mz};
    double* red = reinterpret_cast<double*>(smem_raw + C::red_off);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
#pragma unroll
      for (int o = RW / 2; o > 0; o >>= 1) v[i] += __shfl_down_sync(0xffffffffu, v[i], o, RW);
    }
    if (tl % RW == 0) {
#pragma unroll
      for (int i = 0; i < 4; ++i) red[(gs * WPS + tl / RW) * 4 + i] = v[i];
    }
    __syncthreads();
    if (tl < 4) {
      double x = 0.0;
      for (int w = 0; w < WPS; ++w) x += red[(gs * WPS + w) * 4 + tl];
      if (tl == 0) a.e_slot[slot] = -x;
      else a.m_slot[slot * 3 + (tl - 1)] = x / (double)g.N;
    }
  }
}

}  // namespace zm

// ------------------------------------------------------------------------------------------------ host side
template <int L, int V, int G>
inline cudaError_t zmarch_launch_t(const ZmarchArgs& a, cudaStream_t stream) {
  using C = zm::Cfg<L, V, G>;
  static bool configured = false;
  if (!configured) {
    const cudaError_t e = cudaFuncSetAttribute(zm::zmarch_kernel<L, V, G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::smem_bytes);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  zm::zmarch_kernel<L, V, G><<<a.g.R / G, C::NT, C::smem_bytes, stream>>>(a);
  return cudaGetLastError();
}

// largest group size the geometry allows: the G slots of a CTA must belong to one sample
inline int zmarch_pick_g(const Geom& g, int gmax) {
  int G = gmax;
  while (G > 1 && (g.O * g.T) % G != 0) G >>= 1;
  return G;
}

inline bool zmarch_supported(const Geom& g) { return g.L == 8 || g.L == 16 || g.L == 32; }

#define HSG_ZM_CASE(L_, V_, G_) if (a.g.L == L_ && G == G_) return zmarch_launch_t<L_, V_, G_>(a, stream);
inline cudaError_t zmarch_launch(const ZmarchArgs& a, cudaStream_t stream, int* n_launch) {
  *n_launch = 1;
  if (a.g.L == 32) {
    const int G = zmarch_pick_g(a.g, HSG_ZM_L32_G);
    HSG_ZM_CASE(32, HSG_ZM_L32_V, HSG_ZM_L32_G)
#if HSG_ZM_L32_G > 2
    HSG_ZM_CASE(32, HSG_ZM_L32_V, 2)
#endif
#if HSG_ZM_L32_G > 1
    HSG_ZM_CASE(32, HSG_ZM_L32_V, 1)
#endif
  }
#ifndef HSG_ZM_ONLY_L32     // (variant builds for experiments instantiate L = 32 only)
  else if (a.g.L == 16) {
    const int G = zmarch_pick_g(a.g, 8);
    HSG_ZM_CASE(16, HSG_ZM_L16_V, 8) HSG_ZM_CASE(16, HSG_ZM_L16_V, 4) HSG_ZM_CASE(16, HSG_ZM_L16_V, 2) HSG_ZM_CASE(16, HSG_ZM_L16_V, 1)
  } else if (a.g.L == 8) {
    const int G = zmarch_pick_g(a.g, 8);
    HSG_ZM_CASE(8, 2, 8) HSG_ZM_CASE(8, 2, 4) HSG_ZM_CASE(8, 2, 2) HSG_ZM_CASE(8, 2, 1)
  }
#endif
  *n_launch = 0;
  return cudaErrorNotSupported;
}
#undef HSG_ZM_CASE

}  // namespace hsg
