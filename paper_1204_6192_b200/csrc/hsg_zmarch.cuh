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
//     colours and in every plane.  All its global loads and stores go to its own column (128-bit,
//     coalesced over the warp), so no inter-thread ordering of global memory is ever needed; the z
//     neighbours of a site are the thread's own registers from the neighbouring steps.
//   * In-plane neighbours (rows y-1, y+1 and the one x neighbour outside the thread's V sites) are
//     exchanged through shared memory: X1 holds the old colour-1 spins of plane k, X0 the new colour-0
//     spins of plane k-1, both double-buffered, one __syncthreads per step.
//   * Couplings and fields of the sample stream through a 4-slot shared-memory ring filled by bulk
//     async copies (cp.async.bulk, one 12*L*L/2-float plane per copy, mbarrier completion) issued one
//     step ahead by thread 0, and are shared by the G systems of the CTA (PAPER.md:161's R_TO idea).
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
#define HSG_ZM_L32_V 2
#endif
#ifndef HSG_ZM_L32_G
#define HSG_ZM_L32_G 2
#endif
#ifndef HSG_ZM_L16_V
#define HSG_ZM_L16_V 2
#endif
constexpr int kRing = 4;
constexpr int kUnroll = HSG_ZM_UNROLL;   // unroll factor of the main march loop   // J/H ring slots: planes k-2, k-1, k live + plane k+1 in flight

// ---------------------------------------------------------------- PTX wrappers: mbarrier + bulk async copy
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}

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
  static constexpr int JP = 12 * CS;              // J/H plane (2 colours x 6 arrays)
  static constexpr int RW = TPS < 32 ? TPS : 32;  // shuffle width of the per-system reduction
  static constexpr int WPS = TPS / RW;            // partial sums per system after the shuffle stage
  static constexpr uint32_t red_off = 64;         // byte offsets inside dynamic shared memory: [G][WPS][4] doubles
  static constexpr uint32_t ring_off = 64 + 128 * ((G * WPS * 32 + 127) / 128);
  static constexpr uint32_t x_off = ring_off + 4u * kRing * JP;
  static constexpr size_t smem_bytes = x_off + sizeof(float) * ((size_t)G * 4 * HP);
  static_assert(Lh % V == 0, "row length must be a multiple of the vector width");
  static_assert((JP * 4) % 16 == 0, "bulk copies move multiples of 16 bytes");
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

// Local field of V sites of colour `cu` in plane zp, accumulated in the order H, x+, x-, y+, y-, z+, z-
// (DESIGN.md §3.1), then the move.  `q` = the thread's own column of the other colour in this plane,
// `xs` = shared-memory half-plane of the other colour in this plane (rows y+-1 and the x edge),
// `zlo`/`zhi` = own column of the other colour in planes zp-1 / zp+1,
// `jo` = J/H arrays of colour cu in plane zp, `jx` = arrays of the other colour in plane zp,
// `jzlo` = Jz array of the other colour in plane zp-1 (shared-memory ring; all 32-bit shared addresses).
// EN = 0: move only; 1: also accumulate H_i.s_i and s_i of the NEW spin (colour 0 in the final sweep);
// 2: additionally s_i.(sum_6 J_ij s_j) with every bond of the site (colour 1 in the final sweep, when all its
// neighbours already hold their final values).
template <int L, int V, bool HB, int EN>
__device__ __forceinline__ void update_sites(float (&out)[3][V], const float (&own)[3][V], const float (&q)[3][V],
                                             const float (&zlo)[3][V], const float (&zhi)[3][V], uint32_t xs,
                                             uint32_t jo, uint32_t jx, uint32_t jzlo,
                                             const Th& th, int off, const HbPar& hp, uint32_t site0, EAcc& ea) {
  constexpr uint32_t CSB = 4u * L * (L / 2);
  const uint32_t edge = off ? th.edge1 : th.edge0;
  float Jxp[V], Jxm[V], Jyp[V], Jym[V], Jzp[V], Jzm[V];
  const uint32_t jo_row = jo + th.row;
  lds<V>(Jxp, jo_row);
  lds<V>(Jyp, jo_row + CSB);
  lds<V>(Jzp, jo_row + 2 * CSB);
  {
    float t[V];
    lds<V>(t, jx + th.row);
    const float te = lds1(jx + th.edge0);
#pragma unroll
    for (int e = 0; e < V; ++e) Jxm[e] = off ? t[e] : (e > 0 ? t[e > 0 ? e - 1 : 0] : te);
  }
  lds<V>(Jym, jx + CSB + th.rowm);
  lds<V>(Jzm, jzlo + th.row);
  float h[3][V];
  float Hs[3][V];
  double hd[3][V];
  const uint32_t xs_p = xs + th.rowp, xs_m = xs + th.rowm, xs_e = xs + edge;
#pragma unroll
  for (int mu = 0; mu < 3; ++mu) {
    float Hm[V], yp[V], ym[V];
    lds<V>(Hm, jo_row + (3 + mu) * CSB);
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
  uint32_t full;       // [kRing] mbarriers
  uint32_t ring;       // [kRing][JP] floats
  uint32_t x0;         // this thread's system: [2][HP] new colour-0 spins of planes k-1, k
  uint32_t x1;         // this thread's system: [2][HP] old colour-1 spins of planes k, k+1
};

struct Stream {        // J/H plane stream: index q -> plane (q-1) mod L
  int issued, waited, total;
};

template <int L, int JP>
__device__ __forceinline__ void ring_advance(const Smem& sm, const float* __restrict__ jh_d, Stream& st, int nd) {
  if (threadIdx.x == 0) {                               // producer: keep one plane in flight
    const int upto = min(nd + 1, st.total - 1);
    while (st.issued < upto) {
      ++st.issued;
      const int plane = (st.issued + L - 1) % L;
      const uint32_t slot = (uint32_t)st.issued % kRing;
      const uint32_t bar = sm.full + 8u * slot;
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"((uint32_t)JP * 4u) : "memory");
      asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                   ::"r"(sm.ring + slot * (uint32_t)JP * 4u), "l"(jh_d + (size_t)plane * JP), "r"((uint32_t)JP * 4u), "r"(bar) : "memory");
    }
  }
  while (st.waited < nd) {
    ++st.waited;
    const uint32_t bar = sm.full + 8u * ((uint32_t)st.waited % kRing);
    const uint32_t parity = ((uint32_t)st.waited / kRing) & 1u;
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
                                            const Th& th, const HbPar& hp, int qbase, Stream& st, EAcc& ea) {
  using C = Cfg<L, V, G>;
  constexpr int CS = C::CS, HP = C::HP, JP = C::JP, PS = 2 * C::HP;
  constexpr uint32_t CSB = 4u * CS, HPB = 4u * HP, JPB = 4u * JP;
  float A[3][V], B[3][V], Cc[3][V], O[3][V], P[3][V], Q[3][V], R[3][V], Cn[3][V], On[3][V];
  float* Sr = S + (th.row >> 2);                       // own column, plane 0, colour 0, component 0
  // prologue: A = c1old(L-1), B = c1old(0) (published in X1[0]), prefetch c1old(1) and c0old(0)
#pragma unroll
  for (int mu = 0; mu < 3; ++mu) {
    ldg<V>(A[mu], Sr + (L - 1) * PS + HP + mu * CS);
    ldg<V>(B[mu], Sr + HP + mu * CS);
    ldg<V>(Cn[mu], Sr + 1 * PS + HP + mu * CS);
    if (!HB) ldg<V>(On[mu], Sr + mu * CS);
#pragma unroll
    for (int e = 0; e < V; ++e) { P[mu][e] = 0.0f; Q[mu][e] = 0.0f; if (HB) On[mu][e] = 0.0f; }
    sts<V>(sm.x1 + mu * CSB + th.row, B[mu]);
  }
  __syncthreads();
  // main steps: colour 0 of plane k, then colour 1 of plane k-1
#pragma unroll (EN ? 1 : kUnroll)
  for (int k = 0; k < L; ++k) {
    const int nd = qbase + k + 1;                       // newest J/H stream index this step reads (plane k)
    ring_advance<L, JP>(sm, jh_d, st, nd);
#pragma unroll
    for (int mu = 0; mu < 3; ++mu)
#pragma unroll
      for (int e = 0; e < V; ++e) { Cc[mu][e] = Cn[mu][e]; O[mu][e] = On[mu][e]; }
    if (k + 1 < L) {                                    // prefetch the next step's planes
      const int zc = (k + 2 == L) ? 0 : k + 2;
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) {
        ldg<V>(Cn[mu], Sr + zc * PS + HP + mu * CS);
        if (!HB) ldg<V>(On[mu], Sr + (k + 1) * PS + mu * CS);
      }
    } else {                                            // k = L-1: the new colour 0 of plane 0, needed by step L
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) ldg<V>(On[mu], Sr + mu * CS);
    }
    const int off = (th.y + k) & 1;
    const uint32_t jk = sm.ring + ((uint32_t)nd % kRing) * JPB;                  // plane k
    const uint32_t jk1 = sm.ring + ((uint32_t)(nd + kRing - 1) % kRing) * JPB;   // plane k-1
    const uint32_t jk2 = sm.ring + ((uint32_t)(nd + kRing - 2) % kRing) * JPB;   // plane k-2
    const uint32_t par = (uint32_t)(k & 1);
    {
      const uint32_t site0 = (uint32_t)(2 * th.j0 + off + L * (th.y + L * k));
      update_sites<L, V, HB, EN ? 1 : 0>(R, O, B, A, Cc, sm.x1 + par * HPB, jk, jk + 6 * CSB, jk1 + 8 * CSB, th, off, hp, site0, ea);
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) {
        stg<V>(Sr + k * PS + mu * CS, R[mu]);
        sts<V>(sm.x0 + par * HPB + mu * CSB + th.row, R[mu]);
      }
    }
    if (k >= 2) {     // colour 1 of plane k-1
      const uint32_t site0 = (uint32_t)(2 * th.j0 + off + L * (th.y + L * (k - 1)));
      float N1[3][V];
      update_sites<L, V, HB, EN ? 2 : 0>(N1, A, Q, P, R, sm.x0 + (par ^ 1u) * HPB, jk1 + 6 * CSB, jk1, jk2 + 2 * CSB, th, off, hp, site0, ea);
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) stg<V>(Sr + (k - 1) * PS + HP + mu * CS, N1[mu]);
    }
    if (k + 1 < L) {
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) sts<V>(sm.x1 + (par ^ 1u) * HPB + mu * CSB + th.row, Cc[mu]);
    }
    __syncthreads();
#pragma unroll
    for (int mu = 0; mu < 3; ++mu)
#pragma unroll
      for (int e = 0; e < V; ++e) { A[mu][e] = B[mu][e]; B[mu][e] = Cc[mu][e]; P[mu][e] = Q[mu][e]; Q[mu][e] = R[mu][e]; }
  }
  // tail: colour 1 of plane L-1 (step L) and of plane 0 (step L+1); their z+ neighbours are the new colour-0
  // spins of planes 0 and 1, read back from the thread's own column
#pragma unroll 1
  for (int kk = 0; kk < 2; ++kk) {
    const int k = L + kk;
    const int nd = qbase + k;                            // plane k-1 (mod L)
    ring_advance<L, JP>(sm, jh_d, st, nd);
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
    const uint32_t j1 = sm.ring + ((uint32_t)nd % kRing) * JPB;                  // plane k-1
    const uint32_t j2 = sm.ring + ((uint32_t)(nd + kRing - 1) % kRing) * JPB;    // plane k-2
    const int z1 = kk == 0 ? L - 1 : 0;
    const uint32_t site0 = (uint32_t)(2 * th.j0 + off + L * (th.y + L * z1));
    float N1[3][V];
    update_sites<L, V, HB, EN ? 2 : 0>(N1, A, Q, P, R, sm.x0 + (uint32_t)((k - 1) & 1) * HPB, j1 + 6 * CSB, j1, j2 + 2 * CSB, th, off, hp, site0, ea);
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
  sm.ring = base + C::ring_off;
  sm.x0 = base + C::x_off + 4u * (uint32_t)(gs * 4) * C::HP;
  sm.x1 = sm.x0 + 4u * 2 * C::HP;
  if (threadIdx.x == 0) {
#pragma unroll
    for (int i = 0; i < kRing; ++i) mbar_init(reinterpret_cast<uint64_t*>(smem_raw) + i, 1);
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
      if (fin) march_sweep<L, V, G, false, true>(sm, S, jh_d, th, hp, s * L, st, ea);
      else march_sweep<L, V, G, false, false>(sm, S, jh_d, th, hp, s * L, st, ea);
    } else {
      const unsigned long long khb = a.k_hb + (unsigned long long)(s - a.n_or);
      hp.c1 = (uint32_t)(khb & 0xFFFFFFFFull); hp.c3 = counter_hi(khb, DOMAIN_HB);
      if (fin) march_sweep<L, V, G, true, true>(sm, S, jh_d, th, hp, s * L, st, ea);
      else march_sweep<L, V, G, true, false>(sm, S, jh_d, th, hp, s * L, st, ea);
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
struct ZmarchVariant { int L, V, G; };

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
  } else if (a.g.L == 16) {
    const int G = zmarch_pick_g(a.g, 8);
    HSG_ZM_CASE(16, HSG_ZM_L16_V, 8) HSG_ZM_CASE(16, HSG_ZM_L16_V, 4) HSG_ZM_CASE(16, HSG_ZM_L16_V, 2) HSG_ZM_CASE(16, HSG_ZM_L16_V, 1)
  } else if (a.g.L == 8) {
    const int G = zmarch_pick_g(a.g, 8);
    HSG_ZM_CASE(8, 2, 8) HSG_ZM_CASE(8, 2, 4) HSG_ZM_CASE(8, 2, 2) HSG_ZM_CASE(8, 2, 1)
  }
  *n_launch = 0;
  return cudaErrorNotSupported;
}
#undef HSG_ZM_CASE

}  // namespace hsg
