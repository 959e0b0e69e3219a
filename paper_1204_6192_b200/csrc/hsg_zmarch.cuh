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
};

namespace zm {

constexpr int kRing = 4;   // J/H ring slots: planes k-2, k-1, k live + plane k+1 in flight

// ---------------------------------------------------------------- PTX wrappers: mbarrier + bulk async copy
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// ---------------------------------------------------------------- V-wide vector access (V = 2 or 4 floats)
template <int V> struct VT;
template <> struct VT<2> { using type = float2; };
template <> struct VT<4> { using type = float4; };

template <int V> __device__ __forceinline__ void ld(float (&r)[V], const float* p) {
  const typename VT<V>::type t = *reinterpret_cast<const typename VT<V>::type*>(p);
  const float* f = reinterpret_cast<const float*>(&t);
#pragma unroll
  for (int e = 0; e < V; ++e) r[e] = f[e];
}
template <int V> __device__ __forceinline__ void st(float* p, const float (&r)[V]) {
  typename VT<V>::type t;
  float* f = reinterpret_cast<float*>(&t);
#pragma unroll
  for (int e = 0; e < V; ++e) f[e] = r[e];
  *reinterpret_cast<typename VT<V>::type*>(p) = t;
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
  static constexpr size_t smem_bytes = 64 + sizeof(float) * ((size_t)kRing * JP + (size_t)G * 4 * HP);
  static_assert(Lh % V == 0, "row length must be a multiple of the vector width");
  static_assert((JP * 4) % 16 == 0, "bulk copies move multiples of 16 bytes");
};

// per-thread constants of the march
struct Th {
  int y, j0;
  int row, rowp, rowm;     // float offsets inside a [y][j] array: own row, row y+1, row y-1 (periodic) at j0
  int edge0, edge1;        // own row at j0-1 and j0+V (periodic): the x neighbour outside the thread's V sites
};

// Local field of V sites of colour `cu` in plane zp, accumulated in the order H, x+, x-, y+, y-, z+, z-
// (DESIGN.md §3.1), then the move.  `q` = the thread's own column of the other colour in this plane,
// `xs` = shared-memory half-plane of the other colour in this plane (rows y+-1 and the x edge),
// `zlo`/`zhi` = own column of the other colour in planes zp-1 / zp+1,
// `jo` = J/H arrays of colour cu in plane zp, `jx` = arrays of the other colour in plane zp,
// `jzlo` = Jz array of the other colour in plane zp-1 (all in the shared-memory ring).
template <int L, int V, bool HB>
__device__ __forceinline__ void update_sites(float (&out)[3][V], const float (&own)[3][V], const float (&q)[3][V],
                                             const float (&zlo)[3][V], const float (&zhi)[3][V], const float* __restrict__ xs,
                                             const float* __restrict__ jo, const float* __restrict__ jx, const float* __restrict__ jzlo,
                                             const Th& th, int off, float beta, uint32_t sysid, uint32_t c1, uint32_t c3,
                                             PhiloxKey key, uint32_t site0) {
  constexpr int CS = L * (L / 2);
  const int edge = off ? th.edge1 : th.edge0;
  float Jxp[V], Jxm[V], Jyp[V], Jym[V], Jzp[V], Jzm[V];
  ld<V>(Jxp, jo + 0 * CS + th.row);
  ld<V>(Jyp, jo + 1 * CS + th.row);
  ld<V>(Jzp, jo + 2 * CS + th.row);
  {
    float t[V];
    ld<V>(t, jx + 0 * CS + th.row);
    const float te = jx[0 * CS + th.edge0];
#pragma unroll
    for (int e = 0; e < V; ++e) Jxm[e] = off ? t[e] : (e > 0 ? t[e > 0 ? e - 1 : 0] : te);
  }
  ld<V>(Jym, jx + 1 * CS + th.rowm);
  ld<V>(Jzm, jzlo + th.row);
  float h[3][V];
#pragma unroll
  for (int mu = 0; mu < 3; ++mu) {
    float Hm[V], yp[V], ym[V];
    ld<V>(Hm, jo + (3 + mu) * CS + th.row);
    ld<V>(yp, xs + mu * CS + th.rowp);
    ld<V>(ym, xs + mu * CS + th.rowm);
    const float se = xs[mu * CS + edge];
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
    }
  }
#pragma unroll
  for (int e = 0; e < V; ++e) {
    const Vec3 hv = {h[0][e], h[1][e], h[2][e]};
    Vec3 s;
    if (HB) {
      uint32_t w0, w1, w2, w3;
      philox4x32_10(site0 + 2u * (uint32_t)e, c1, sysid, c3, key.k0, key.k1, w0, w1, w2, w3);
      s = hb_draw(hv, beta, u01(w0), u01(w1));
    } else {
      const Vec3 sv = {own[0][e], own[1][e], own[2][e]};
      s = or_reflect(sv, hv);
    }
    out[0][e] = s.x; out[1][e] = s.y; out[2][e] = s.z;
  }
}

// Shared state of one CTA during the march
template <int L, int V, int G> struct Smem {
  using C = Cfg<L, V, G>;
  uint64_t* full;      // [kRing] mbarriers
  float* ring;         // [kRing][JP]
  float* x0;           // this thread's system: [2][HP] new colour-0 spins of planes k-1, k
  float* x1;           // this thread's system: [2][HP] old colour-1 spins of planes k, k+1
};

// One full sweep (both colours, all planes) of the G systems of this CTA.
template <int L, int V, int G, bool HB>
__device__ __forceinline__ void march_sweep(const Smem<L, V, G>& sm, float* __restrict__ S, const float* __restrict__ jh_d,
                                            const Th& th, float beta, uint32_t sysid, unsigned long long khb, PhiloxKey key,
                                            int qbase, int total, int& issued, int& waited) {
  using C = Cfg<L, V, G>;
  constexpr int CS = C::CS, HP = C::HP, JP = C::JP, PS = 2 * C::HP;
  const uint32_t c1 = (uint32_t)(khb & 0xFFFFFFFFull), c3 = counter_hi(khb, DOMAIN_HB);
  float A[3][V], B[3][V], Cc[3][V], O[3][V], P[3][V], Q[3][V], R[3][V], Cn[3][V], On[3][V];
  // prologue: A = c1old(L-1), B = c1old(0) (published in X1[0]), prefetch c1old(1) and c0old(0)
#pragma unroll
  for (int mu = 0; mu < 3; ++mu) {
    ldg<V>(A[mu], S + (L - 1) * PS + HP + mu * CS + th.row);
    ldg<V>(B[mu], S + HP + mu * CS + th.row);
    ldg<V>(Cn[mu], S + 1 * PS + HP + mu * CS + th.row);
    if (!HB) ldg<V>(On[mu], S + mu * CS + th.row);
#pragma unroll
    for (int e = 0; e < V; ++e) { P[mu][e] = 0.0f; Q[mu][e] = 0.0f; if (HB) On[mu][e] = 0.0f; }
    st<V>(sm.x1 + mu * CS + th.row, B[mu]);
  }
  __syncthreads();
#pragma unroll 1
  for (int k = 0; k < L + 2; ++k) {
    const int nd = qbase + (k < L ? k + 1 : k);           // newest J/H stream index this step reads
    if (threadIdx.x == 0) {                               // producer: keep one plane in flight
      const int upto = min(nd + 1, total - 1);
      while (issued < upto) {
        ++issued;
        const int plane = (issued + L - 1) % L;
        uint64_t* bar = sm.full + (issued % kRing);
        mbar_expect_tx(bar, JP * 4);
        bulk_g2s(sm.ring + (issued % kRing) * JP, jh_d + (size_t)plane * JP, JP * 4, bar);
      }
    }
#pragma unroll
    for (int mu = 0; mu < 3; ++mu)
#pragma unroll
      for (int e = 0; e < V; ++e) { Cc[mu][e] = Cn[mu][e]; O[mu][e] = On[mu][e]; }
    if (k + 1 < L) {
      const int zc = (k + 2 == L) ? 0 : k + 2;
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) {
        ldg<V>(Cn[mu], S + zc * PS + HP + mu * CS + th.row);
        if (!HB) ldg<V>(On[mu], S + (k + 1) * PS + mu * CS + th.row);
      }
    }
    while (waited < nd) { ++waited; mbar_wait(sm.full + (waited % kRing), (uint32_t)(waited / kRing) & 1u); }
    const int off = (th.y + k) & 1;
    const float* jk = sm.ring + (nd % kRing) * JP;                 // k < L: plane k;   k >= L: plane k-1
    const float* jk1 = sm.ring + ((nd - 1) % kRing) * JP;
    const float* jk2 = sm.ring + ((nd - 2 + kRing) % kRing) * JP;
    if (k < L) {
      const uint32_t site0 = (uint32_t)(2 * th.j0 + off + L * (th.y + L * k));
      update_sites<L, V, HB>(R, O, B, A, Cc, sm.x1 + (k & 1) * HP, jk, jk + 6 * CS, jk1 + 8 * CS, th, off, beta, sysid, c1, c3, key, site0);
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) stg<V>(S + k * PS + mu * CS + th.row, R[mu]);
    } else {
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) ldg<V>(R[mu], S + (k - L) * PS + mu * CS + th.row);   // new colour 0 of planes 0, 1
    }
    if (k <= L) {
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) st<V>(sm.x0 + (k & 1) * HP + mu * CS + th.row, R[mu]);
    }
    if (k >= 2) {     // colour 1 of plane k-1 (plane 0 when k = L+1)
      const int z1 = (k - 1 == L) ? 0 : k - 1;
      const float* j1 = (k < L) ? jk1 : jk;          // plane k-1
      const float* j2 = (k < L) ? jk2 : jk1;         // plane k-2
      const uint32_t site0 = (uint32_t)(2 * th.j0 + off + L * (th.y + L * z1));
      float N1[3][V];
      update_sites<L, V, HB>(N1, A, Q, P, R, sm.x0 + ((k - 1) & 1) * HP, j1 + 6 * CS, j1, j2 + 2 * CS, th, off, beta, sysid, c1, c3, key, site0);
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) stg<V>(S + z1 * PS + HP + mu * CS + th.row, N1[mu]);
    }
    if (k + 1 < L) {
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) st<V>(sm.x1 + ((k + 1) & 1) * HP + mu * CS + th.row, Cc[mu]);
    }
    __syncthreads();
#pragma unroll
    for (int mu = 0; mu < 3; ++mu)
#pragma unroll
      for (int e = 0; e < V; ++e) { A[mu][e] = B[mu][e]; B[mu][e] = Cc[mu][e]; P[mu][e] = Q[mu][e]; Q[mu][e] = R[mu][e]; }
  }
}

template <int L, int V, int G>
__global__ void __launch_bounds__(Cfg<L, V, G>::NT, 1) zmarch_kernel(ZmarchArgs a) {
  using C = Cfg<L, V, G>;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Smem<L, V, G> sm;
  sm.full = reinterpret_cast<uint64_t*>(smem_raw);
  sm.ring = reinterpret_cast<float*>(smem_raw + 64);
  float* xbase = sm.ring + kRing * C::JP;
  const int gs = threadIdx.x / C::TPS, tl = threadIdx.x % C::TPS;
  sm.x0 = xbase + (gs * 4) * C::HP;
  sm.x1 = xbase + (gs * 4 + 2) * C::HP;
  if (threadIdx.x == 0) {
#pragma unroll
    for (int i = 0; i < kRing; ++i) mbar_init(sm.full + i, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  Th th;
  th.y = tl / C::TPR; th.j0 = (tl % C::TPR) * V;
  th.row = th.y * C::Lh + th.j0;
  th.rowp = ((th.y + 1 == L) ? 0 : th.y + 1) * C::Lh + th.j0;
  th.rowm = ((th.y == 0) ? L - 1 : th.y - 1) * C::Lh + th.j0;
  th.edge0 = th.y * C::Lh + ((th.j0 == 0) ? C::Lh - 1 : th.j0 - 1);
  th.edge1 = th.y * C::Lh + ((th.j0 + V == C::Lh) ? 0 : th.j0 + V);

  const Geom& g = a.g;
  const int slot = blockIdx.x * G + gs;                 // G consecutive slots of one sample
  const int d = slot / (g.O * g.T);
  const int grp = slot / g.T;
  const int t = a.temp_of_slot[slot];
  const float beta = a.beta[t];
  const uint32_t sysid = (uint32_t)((g.sample_offset * g.O * g.T) + (unsigned long long)grp * g.T + t);
  float* S = a.spins + (size_t)slot * 3 * g.N;
  const float* jh_d = a.jh + (size_t)d * 6 * g.N;

  const int n_sweeps = a.n_or + a.n_hb;
  const int total = n_sweeps * L + 2;                   // J/H stream: planes L-1, 0, 1, ..., repeated; index q -> plane (q-1) mod L
  int issued = -1, waited = -1;
  for (int s = 0; s < n_sweeps; ++s) {
    if (s < a.n_or) march_sweep<L, V, G, false>(sm, S, jh_d, th, beta, sysid, 0ull, a.key, s * L, total, issued, waited);
    else march_sweep<L, V, G, true>(sm, S, jh_d, th, beta, sysid, a.k_hb + (unsigned long long)(s - a.n_or), a.key, s * L, total, issued, waited);
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
    const int G = zmarch_pick_g(a.g, 4);
    HSG_ZM_CASE(32, 4, 4) HSG_ZM_CASE(32, 4, 2) HSG_ZM_CASE(32, 4, 1)
  } else if (a.g.L == 16) {
    const int G = zmarch_pick_g(a.g, 8);
    HSG_ZM_CASE(16, 4, 8) HSG_ZM_CASE(16, 4, 4) HSG_ZM_CASE(16, 4, 2) HSG_ZM_CASE(16, 4, 1)
  } else if (a.g.L == 8) {
    const int G = zmarch_pick_g(a.g, 8);
    HSG_ZM_CASE(8, 2, 8) HSG_ZM_CASE(8, 2, 4) HSG_ZM_CASE(8, 2, 2) HSG_ZM_CASE(8, 2, 1)
  }
  *n_launch = 0;
  return cudaErrorNotSupported;
}
#undef HSG_ZM_CASE

}  // namespace hsg
