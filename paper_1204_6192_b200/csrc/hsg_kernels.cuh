// hsg_kernels.cuh — layout conversion, initialisation, the generic (one colour per launch) sweep
// kernel, the energy / magnetisation / overlap reductions and the parallel-tempering kernel.
// The fused z-marching sweep kernel lives in hsg_zmarch.cuh.
#pragma once
#include "hsg_layout.cuh"
#include "hsg_math.cuh"

namespace hsg {

constexpr int kThreads = 256;

// ------------------------------------------------------------------ small vector load/store helpers
template <int V> struct Vec;
template <> struct Vec<1> { float v[1]; };
template <> struct Vec<2> { float v[2]; };
template <> struct Vec<4> { float v[4]; };

template <int V> __device__ __forceinline__ Vec<V> ldv(const float* p);
template <> __device__ __forceinline__ Vec<1> ldv<1>(const float* p) { Vec<1> r; r.v[0] = *p; return r; }
template <> __device__ __forceinline__ Vec<2> ldv<2>(const float* p) {
  const float2 t = *reinterpret_cast<const float2*>(p); Vec<2> r; r.v[0] = t.x; r.v[1] = t.y; return r;
}
template <> __device__ __forceinline__ Vec<4> ldv<4>(const float* p) {
  const float4 t = *reinterpret_cast<const float4*>(p); Vec<4> r; r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w; return r;
}
template <int V> __device__ __forceinline__ void stv(float* p, const Vec<V>& r);
template <> __device__ __forceinline__ void stv<1>(float* p, const Vec<1>& r) { *p = r.v[0]; }
template <> __device__ __forceinline__ void stv<2>(float* p, const Vec<2>& r) { *reinterpret_cast<float2*>(p) = make_float2(r.v[0], r.v[1]); }
template <> __device__ __forceinline__ void stv<4>(float* p, const Vec<4>& r) { *reinterpret_cast<float4*>(p) = make_float4(r.v[0], r.v[1], r.v[2], r.v[3]); }

// ------------------------------------------------------------------ layout conversion
// canonical J[d][dir][i], H[d][c][i] (i = x + L(y + L z))  ->  JH[d][z][c][k][y][j]
__global__ void pack_disorder_kernel(Geom g, const float* __restrict__ J, const float* __restrict__ H, float* __restrict__ JH) {
  const long long tid = (long long)blockIdx.x * kThreads + threadIdx.x;
  if (tid >= (long long)g.D * g.N) return;
  const int d = (int)(tid / g.N);
  const long long i = tid % g.N;
  const int x = (int)(i % g.L), y = (int)((i / g.L) % g.L), z = (int)(i / ((long long)g.L * g.L));
  const int c = (x + y + z) & 1, j = x >> 1;
  float* dst = JH + (long long)d * 6 * g.N;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    dst[jh_index(g, z, c, k, y, j)] = J[((long long)d * 3 + k) * g.N + i];
    dst[jh_index(g, z, c, 3 + k, y, j)] = H ? H[((long long)d * 3 + k) * g.N + i] : 0.0f;
  }
}

// canonical S[d][o][t][mu][i] by TEMPERATURE index  <->  private slots.  TO_PRIVATE: canonical -> slots.
template <bool TO_PRIVATE>
__global__ void convert_spins_kernel(Geom g, const int32_t* __restrict__ slot_of_temp, float* __restrict__ priv, float* __restrict__ canon) {
  const long long tid = (long long)blockIdx.x * kThreads + threadIdx.x;
  if (tid >= (long long)g.R * g.N) return;
  const int r = (int)(tid / g.N);          // (d*O + o)*T + t
  const long long i = tid % g.N;
  const int grp = r / g.T;
  const int slot = grp * g.T + slot_of_temp[r];
  const int x = (int)(i % g.L), y = (int)((i / g.L) % g.L), z = (int)(i / ((long long)g.L * g.L));
  const int c = (x + y + z) & 1, j = x >> 1;
  float* p = priv + (long long)slot * 3 * g.N;
  float* q = canon + (long long)r * 3 * g.N;
#pragma unroll
  for (int mu = 0; mu < 3; ++mu) {
    if (TO_PRIVATE) p[spin_index(g, z, c, mu, y, j)] = q[mu * g.N + i];
    else q[mu * g.N + i] = p[spin_index(g, z, c, mu, y, j)];
  }
}

__global__ void init_perm_kernel(Geom g, int32_t* slot_of_temp, int32_t* temp_of_slot) {
  const int tid = blockIdx.x * kThreads + threadIdx.x;
  if (tid >= g.R) return;
  slot_of_temp[tid] = tid % g.T;
  temp_of_slot[tid] = tid % g.T;
}

__global__ void set_perm_kernel(Geom g, const int32_t* __restrict__ src, int32_t* slot_of_temp, int32_t* temp_of_slot) {
  const int tid = blockIdx.x * kThreads + threadIdx.x;
  if (tid >= g.R) return;
  const int s = src[tid];
  slot_of_temp[tid] = s;
  temp_of_slot[(tid / g.T) * g.T + s] = tid % g.T;
}

// ------------------------------------------------------------------ uniform start configuration (INIT domain)
__global__ void init_spins_kernel(Geom g, PhiloxKey key, const int32_t* __restrict__ temp_of_slot, float* __restrict__ spins) {
  const long long tid = (long long)blockIdx.x * kThreads + threadIdx.x;
  if (tid >= (long long)g.R * g.N) return;
  const int slot = (int)(tid / g.N);
  long long rem = tid % g.N;
  const int j = (int)(rem % g.Lh); rem /= g.Lh;
  const int y = (int)(rem % g.L); rem /= g.L;
  const int c = (int)(rem % 2);
  const int z = (int)(rem / 2);
  const int x = 2 * j + ((y + z + c) & 1);
  const uint32_t site = (uint32_t)(x + g.L * (y + g.L * z));
  const int grp = slot / g.T;
  const uint32_t sysid = (uint32_t)((g.sample_offset * g.O * g.T) + (unsigned long long)grp * g.T + temp_of_slot[slot]);
  uint32_t w0, w1, w2, w3;
  philox4x32_10(site, 0u, sysid, counter_hi(0, DOMAIN_INIT), key.k0, key.k1, w0, w1, w2, w3);
  const float u1 = u01(w0), u2 = u01(w1);
  const float ct = __fmaf_rn(2.0f, u1, -1.0f);
  const float st = __fsqrt_rn(__fmaf_rn(-ct, ct, 1.0f));
  float sp, cp;
  spec_sincos2pi(u2, sp, cp);
  float* p = spins + (long long)slot * 3 * g.N;
  p[spin_index(g, z, c, 0, y, j)] = __fmul_rn(st, cp);
  p[spin_index(g, z, c, 1, y, j)] = __fmul_rn(st, sp);
  p[spin_index(g, z, c, 2, y, j)] = ct;
}

// ------------------------------------------------------------------ generic sweep kernel: one colour per launch
struct SweepArgs {
  Geom g;
  float* spins;                 // [R][3N] private layout
  const float* jh;              // [D][6N]
  const int32_t* temp_of_slot;  // [R]
  const float* beta;            // [T]
  PhiloxKey key;
  unsigned long long k_hb;      // heat-bath sweep counter of THIS sweep
};

// Local field of the V compact sites j0..j0+V-1 of colour c in row (y,z), straight from global memory:
// h = H, then x+, x-, y+, y-, z+, z- in that order, one explicit FMA each.
template <int V>
__device__ __forceinline__ void local_field_global(const Geom& g, const float* __restrict__ S, const float* __restrict__ JH,
                                                   int z, int c, int y, int j0, float (&h)[3][V]) {
  const int L = g.L, Lh = g.Lh, cc = 1 - c;
  const int off = (y + z + c) & 1;
  const int yp = (y + 1 == L) ? 0 : y + 1, ym = (y == 0) ? L - 1 : y - 1;
  const int zp = (z + 1 == L) ? 0 : z + 1, zm = (z == 0) ? L - 1 : z - 1;
  const int jx = off ? ((j0 + V == Lh) ? 0 : j0 + V) : ((j0 == 0) ? Lh - 1 : j0 - 1);   // the one x-neighbour outside [j0, j0+V)
  // couplings: forward bonds of this site, backward bonds stored at the neighbour
  const Vec<V> Jxp = ldv<V>(JH + jh_index(g, z, c, 0, y, j0));
  const Vec<V> Jyp = ldv<V>(JH + jh_index(g, z, c, 1, y, j0));
  const Vec<V> Jzp = ldv<V>(JH + jh_index(g, z, c, 2, y, j0));
  const Vec<V> Jxq = ldv<V>(JH + jh_index(g, z, cc, 0, y, j0));
  const float Jxe = JH[jh_index(g, z, cc, 0, y, jx)];
  const Vec<V> Jym = ldv<V>(JH + jh_index(g, z, cc, 1, ym, j0));
  const Vec<V> Jzm = ldv<V>(JH + jh_index(g, zm, cc, 2, y, j0));
  Vec<V> Jxm;
#pragma unroll
  for (int e = 0; e < V; ++e) Jxm.v[e] = off ? Jxq.v[e] : (e > 0 ? Jxq.v[e > 0 ? e - 1 : 0] : Jxe);
#pragma unroll
  for (int mu = 0; mu < 3; ++mu) {
    const Vec<V> Hm = ldv<V>(JH + jh_index(g, z, c, 3 + mu, y, j0));
    const Vec<V> sq = ldv<V>(S + spin_index(g, z, cc, mu, y, j0));
    const float se = S[spin_index(g, z, cc, mu, y, jx)];
    const Vec<V> syp = ldv<V>(S + spin_index(g, z, cc, mu, yp, j0));
    const Vec<V> sym = ldv<V>(S + spin_index(g, z, cc, mu, ym, j0));
    const Vec<V> szp = ldv<V>(S + spin_index(g, zp, cc, mu, y, j0));
    const Vec<V> szm = ldv<V>(S + spin_index(g, zm, cc, mu, y, j0));
#pragma unroll
    for (int e = 0; e < V; ++e) {
      const float sxp = off ? (e + 1 < V ? sq.v[e + 1 < V ? e + 1 : 0] : se) : sq.v[e];
      const float sxm = off ? sq.v[e] : (e > 0 ? sq.v[e > 0 ? e - 1 : 0] : se);
      float acc = Hm.v[e];
      acc = __fmaf_rn(Jxp.v[e], sxp, acc);
      acc = __fmaf_rn(Jxm.v[e], sxm, acc);
      acc = __fmaf_rn(Jyp.v[e], syp.v[e], acc);
      acc = __fmaf_rn(Jym.v[e], sym.v[e], acc);
      acc = __fmaf_rn(Jzp.v[e], szp.v[e], acc);
      acc = __fmaf_rn(Jzm.v[e], szm.v[e], acc);
      h[mu][e] = acc;
    }
  }
}

// Each thread updates V consecutive compact sites of colour `colour` in one row (y,z) of one slot.
// Neighbours are read straight from global memory (L1/L2 provide the reuse).  The field is accumulated
// in the order H, x+, x-, y+, y-, z+, z- (DESIGN.md §3.1).  FM: the fast-math variant of the heat-bath draw (HSG_FLAG_FAST_MATH).
template <int V, bool HB, bool FM = false>
__global__ void __launch_bounds__(kThreads) sweep_generic_kernel(SweepArgs a, int colour) {
  const Geom& g = a.g;
  const int L = g.L, Lh = g.Lh;
  const int qpr = Lh / V;
  const long long per_slot = (long long)L * L * qpr;
  const long long tid = (long long)blockIdx.x * kThreads + threadIdx.x;
  if (tid >= per_slot * g.R) return;
  const int slot = (int)(tid / per_slot);
  int rem = (int)(tid % per_slot);
  const int q = rem % qpr; rem /= qpr;
  const int y = rem % L;
  const int z = rem / L;
  const int c = colour;
  const int off = (y + z + c) & 1;
  const int j0 = q * V;
  float* S = a.spins + (long long)slot * 3 * g.N;
  const int d = slot / (g.O * g.T);
  const float* JH = a.jh + (long long)d * 6 * g.N;

  float h[3][V], own[3][V];
  local_field_global<V>(g, S, JH, z, c, y, j0, h);
  if (!HB) {
#pragma unroll
    for (int mu = 0; mu < 3; ++mu) {
      const Vec<V> o = ldv<V>(S + spin_index(g, z, c, mu, y, j0));
#pragma unroll
      for (int e = 0; e < V; ++e) own[mu][e] = o.v[e];
    }
  }

  Vec<V> out[3];
  if (HB) {
    const int t = a.temp_of_slot[slot];
    const float beta = a.beta[t];
    const int grp = slot / g.T;
    const uint32_t sysid = (uint32_t)((g.sample_offset * g.O * g.T) + (unsigned long long)grp * g.T + t);
    const uint32_t c1 = (uint32_t)(a.k_hb & 0xFFFFFFFFull), c3 = counter_hi(a.k_hb, DOMAIN_HB);
    // one Philox call per pair of same-colour sites with compact index (even, odd): counter word 0 = the even one,
    // which takes output words 0, 1; its partner takes words 2, 3.  V = 1: every thread makes the call.
    uint32_t wa[V], wb[V];
    if (V == 1) {
      const int odd = j0 & 1;
      uint32_t w0, w1, w2, w3;
      philox4x32_10((uint32_t)(2 * (j0 - odd) + off + L * (y + L * z)), c1, sysid, c3, a.key.k0, a.key.k1, w0, w1, w2, w3);
      wa[0] = odd ? w2 : w0; wb[0] = odd ? w3 : w1;
    } else {
#pragma unroll
      for (int e = 0; e + 1 < V; e += 2)
        philox4x32_10((uint32_t)(2 * (j0 + e) + off + L * (y + L * z)), c1, sysid, c3, a.key.k0, a.key.k1, wa[e], wb[e], wa[e + 1 < V ? e + 1 : e], wb[e + 1 < V ? e + 1 : e]);
    }
#pragma unroll
    for (int e = 0; e < V; ++e) {
      const Vec3 hv = { h[0][e], h[1][e], h[2][e] };
      const Vec3 s = FM ? hb_draw_fast(hv, beta, u01(wa[e]), u01(wb[e])) : hb_draw(hv, beta, u01(wa[e]), u01(wb[e]));
      out[0].v[e] = s.x; out[1].v[e] = s.y; out[2].v[e] = s.z;
    }
  } else {
#pragma unroll
    for (int e = 0; e < V; ++e) {
      const Vec3 hv = { h[0][e], h[1][e], h[2][e] };
      const Vec3 sv = { own[0][e], own[1][e], own[2][e] };
      const Vec3 s = or_reflect(sv, hv);
      out[0].v[e] = s.x; out[1].v[e] = s.y; out[2].v[e] = s.z;
    }
  }
#pragma unroll
  for (int mu = 0; mu < 3; ++mu) stv<V>(S + spin_index(g, z, c, mu, y, j0), out[mu]);
}

// ------------------------------------------------------------------ deterministic block reduction (fp64)
template <int NV>
__device__ __forceinline__ void block_reduce_store(double (&v)[NV], double* __restrict__ dst) {
  __shared__ double sm[kThreads / 32][NV];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < NV; ++k) {
    double x = v[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
    if (lane == 0) sm[warp][k] = x;
  }
  __syncthreads();
  if (threadIdx.x < NV) {
    double x = 0.0;
#pragma unroll
    for (int w = 0; w < kThreads / 32; ++w) x += sm[w][threadIdx.x];
    dst[threadIdx.x] = x;
  }
}

// ------------------------------------------------------------------ energy (Eq. 1) and magnetisation per slot
// Eq. (1) in the bipartite form: every bond joins a colour-0 and a colour-1 site, so
//   E = - sum_{i in colour 1} s_i . h_i  -  sum_{i in colour 0} s_i . H_i ,   h_i = the local field of §3.1 (H_i included).
// Site terms in the spins' precision with the fixed FMA order of the moves, sums in fp64.
// One block per (slot, chunk of ZB planes); each thread takes items of V compact sites of one colour.
// partial[slot][chunk][4] = { -E contribution, sum s_x, sum s_y, sum s_z }.
template <int V>
__global__ void __launch_bounds__(kThreads) energy_mag_kernel(Geom g, int ZB, const float* __restrict__ spins, const float* __restrict__ jh,
                                                              double* __restrict__ partial) {
  const int L = g.L, Lh = g.Lh, qpr = Lh / V;
  const int n_chunks = (L + ZB - 1) / ZB;
  const int slot = blockIdx.x / n_chunks, chunk = blockIdx.x % n_chunks;
  const int z0 = chunk * ZB, nz = min(ZB, L - z0);
  const float* S = spins + (long long)slot * 3 * g.N;
  const float* JH = jh + (long long)(slot / (g.O * g.T)) * 6 * g.N;
  double acc[4] = {0.0, 0.0, 0.0, 0.0};
  const int ipp = 2 * L * qpr;                      // items per plane
  for (int it = threadIdx.x; it < nz * ipp; it += kThreads) {
    const int q = it % qpr; int rem = it / qpr;
    const int y = rem % L; rem /= L;
    const int c = rem & 1; const int z = z0 + (rem >> 1);
    const int j0 = q * V;
    float h[3][V], s[3][V];
    if (c == 1) {
      local_field_global<V>(g, S, JH, z, c, y, j0, h);
    } else {
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) {
        const Vec<V> Hm = ldv<V>(JH + jh_index(g, z, c, 3 + mu, y, j0));
#pragma unroll
        for (int e = 0; e < V; ++e) h[mu][e] = Hm.v[e];
      }
    }
#pragma unroll
    for (int mu = 0; mu < 3; ++mu) {
      const Vec<V> sv = ldv<V>(S + spin_index(g, z, c, mu, y, j0));
#pragma unroll
      for (int e = 0; e < V; ++e) { s[mu][e] = sv.v[e]; acc[1 + mu] += (double)sv.v[e]; }
    }
#pragma unroll
    for (int e = 0; e < V; ++e) {
      const Vec3 sv = {s[0][e], s[1][e], s[2][e]}, hv = {h[0][e], h[1][e], h[2][e]};
      acc[0] += (double)dot3(sv, hv);
    }
  }
  block_reduce_store<4>(acc, partial + (long long)blockIdx.x * 4);
}

// E_slot[slot] = -sum_chunks partial[slot][chunk][0] ; M_slot[slot][mu] = (1/N) sum_chunks partial[slot][chunk][1+mu]   (fixed order)
__global__ void finalize_energy_kernel(Geom g, int n_chunks, const double* __restrict__ partial, double* __restrict__ e_slot, double* __restrict__ m_slot) {
  const int tid = blockIdx.x * kThreads + threadIdx.x;
  if (tid >= g.R * 4) return;
  const int slot = tid / 4, k = tid % 4;
  double x = 0.0;
  for (int z = 0; z < n_chunks; ++z) x += partial[((long long)slot * n_chunks + z) * 4 + k];
  if (k == 0) e_slot[slot] = -x;
  else m_slot[slot * 3 + (k - 1)] = x / (double)g.N;
}

// per-slot values -> per-temperature-index output; NV values per system
__global__ void gather_by_temp_kernel(Geom g, int nv, const int32_t* __restrict__ slot_of_temp, const double* __restrict__ by_slot, double* __restrict__ out) {
  const int tid = blockIdx.x * kThreads + threadIdx.x;
  if (tid >= g.R * nv) return;
  const int r = tid / nv, k = tid % nv;
  const int slot = (r / g.T) * g.T + slot_of_temp[r];
  out[tid] = by_slot[slot * nv + k];
}

// ------------------------------------------------------------------ parallel tempering, Eq. (4)
// Diagnostics of PAPER.md:197 / Fig. 3 (hsg_pt_diag_*): a configuration that arrives at one end point of the ladder after it
// last touched the OTHER end point has made one traversal (a closed loop T_1 -> T_{R_T} -> T_1 = two traversals).  Cold end first.
__device__ __forceinline__ void pt_diag_touch(int T, const int32_t* slot_of_temp, long long* trav, int32_t* last_end) {
#pragma unroll
  for (int e = 0; e < 2; ++e) {
    const int s = slot_of_temp[e == 0 ? 0 : T - 1];
    const int32_t tag = e == 0 ? 1 : -1;
    if (last_end[s] == -tag) ++trav[s];
    last_end[s] = tag;
  }
}

struct PtDiag { long long* moved; long long* trav; int32_t* last_end; };   // all null: diagnostics off

// One thread per (sample, replica) walks the ladder from the lowest temperature.
__global__ void pt_swap_kernel(Geom g, PhiloxKey key, unsigned long long k_pt, const float* __restrict__ beta,
                               const double* __restrict__ e_slot, int32_t* slot_of_temp, int32_t* temp_of_slot,
                               int32_t* __restrict__ accepted, PtDiag diag) {
  const int grp = blockIdx.x * kThreads + threadIdx.x;
  if (grp >= g.D * g.O) return;
  const int base = grp * g.T;
  const uint32_t c2 = (uint32_t)(g.sample_offset * g.O + (unsigned long long)grp);
  const uint32_t c1 = (uint32_t)(k_pt & 0xFFFFFFFFull), c3 = counter_hi(k_pt, DOMAIN_PT);
  int sa = slot_of_temp[base];
  int before = sa;                           // the slot that held temperature t before this pass (diagnostics)
  double Ea = e_slot[base + sa];
  for (int t = 0; t + 1 < g.T; ++t) {
    const int sb = slot_of_temp[base + t + 1];
    const double Eb = e_slot[base + sb];
    const double x = ((double)beta[t + 1] - (double)beta[t]) * (Eb - Ea);
    uint32_t w0, w1, w2, w3;
    philox4x32_10((uint32_t)t, c1, c2, c3, key.k0, key.k1, w0, w1, w2, w3);
    const bool acc = (x >= 0.0) || (log(u01_f64(w0)) < x);
    const int fin = acc ? sb : sa;           // the slot that holds temperature t after this pass
    if (acc) {   // the configuration that held t now holds t+1 and is compared with t+2 next
      slot_of_temp[base + t] = sb; temp_of_slot[base + sb] = t;
      slot_of_temp[base + t + 1] = sa; temp_of_slot[base + sa] = t + 1;
    } else { sa = sb; Ea = Eb; }
    if (accepted) accepted[grp * (g.T - 1) + t] = acc ? 1 : 0;
    if (diag.moved) {                        // temperature t is final now: p_diff counts the passes after which its copy has left
      if (fin != before) ++diag.moved[base + t];
      before = sb;                           // sb was read before this step could change position t+1
    }
  }
  if (diag.moved) {
    if (sa != before) ++diag.moved[base + g.T - 1];
    pt_diag_touch(g.T, slot_of_temp + base, diag.trav + base, diag.last_end + base);
  }
}

// ------------------------------------------------------------------ overlap tensor, Eqs. (5), (6)
// One block per (d, pair, t, chunk of ZB planes): partial[(d,p,t)][chunk][27] = 9 sums for k=0, 9 re, 9 im for k_min.
// k_min lies along x, so  sum_i a_i b_i e^{ikx_i} = sum_x e^{ikx} [ sum_{y,z} a b ]:  a thread keeps a fixed group of
// V compact sites j0..j0+V-1 and ONE x-parity, accumulates the nine products of every (y,z) row it visits (sites of
// x = 2(j0+e) + parity) and applies the phase once at the end.  9 fp64 FMAs per site instead of 27.
// blockDim.x may be smaller than kThreads (small lattices); threads beyond 2*RT*qpr idle.
template <int V>
__global__ void __launch_bounds__(kThreads, 2) overlap_kernel(Geom g, int ZB, const float* __restrict__ spins, const int32_t* __restrict__ slot_of_temp,
                                                           const double* __restrict__ cs_table /*[L][2]*/, double* __restrict__ partial) {
  const int L = g.L, Lh = g.Lh, qpr = Lh / V;
  const int P = g.O * (g.O - 1) / 2;
  const int n_chunks = (L + ZB - 1) / ZB;
  const int chunk = blockIdx.x % n_chunks;
  int rest = blockIdx.x / n_chunks;         // (d*P + p)*T + t
  const int t = rest % g.T; rest /= g.T;
  const int p = rest % P; const int d = rest / P;
  int a = 0, b = 1;
  { int k = p; a = 0; while (k >= g.O - 1 - a) { k -= g.O - 1 - a; ++a; } b = a + 1 + k; }
  const int sa = (d * g.O + a) * g.T + slot_of_temp[(d * g.O + a) * g.T + t];
  const int sb = (d * g.O + b) * g.T + slot_of_temp[(d * g.O + b) * g.T + t];
  const float* A = spins + (long long)sa * 3 * g.N;
  const float* B = spins + (long long)sb * 3 * g.N;
  const int z0 = chunk * ZB, nz = min(ZB, L - z0);
  const int RT = max(1, (int)blockDim.x / (2 * qpr));     // row lanes per x-parity
  double acc[27];
#pragma unroll
  for (int k = 0; k < 27; ++k) acc[k] = 0.0;
  // one item = (group of V compact sites, x-parity, row lane); rows wider than the block (2*qpr > blockDim.x: odd Lh > 128,
  // L > 1024) take their items in several passes
  for (int item = threadIdx.x; item < 2 * qpr * RT; item += blockDim.x) {
    const int q = item % qpr, par = (item / qpr) & 1, r = item / (2 * qpr), j0 = q * V;
    double s9[V][9];
#pragma unroll
    for (int e = 0; e < V; ++e)
#pragma unroll
      for (int k = 0; k < 9; ++k) s9[e][k] = 0.0;
    for (int m = r; m < nz * L; m += RT) {
      const int y = m % L, z = z0 + m / L;
      const int c = (par + y + z) & 1;    // the colour whose sites of row (y,z) sit at x = 2j + par
      Vec<V> av[3], bv[3];
#pragma unroll
      for (int mu = 0; mu < 3; ++mu) {
        av[mu] = ldv<V>(A + spin_index(g, z, c, mu, y, j0));
        bv[mu] = ldv<V>(B + spin_index(g, z, c, mu, y, j0));
      }
#pragma unroll
      for (int e = 0; e < V; ++e) {
        double ad[3], bd[3];
#pragma unroll
        for (int mu = 0; mu < 3; ++mu) { ad[mu] = (double)av[mu].v[e]; bd[mu] = (double)bv[mu].v[e]; }
#pragma unroll
        for (int mu = 0; mu < 3; ++mu)
#pragma unroll
          for (int nu = 0; nu < 3; ++nu) s9[e][mu * 3 + nu] = fma(ad[mu], bd[nu], s9[e][mu * 3 + nu]);
      }
    }
#pragma unroll
    for (int e = 0; e < V; ++e) {
      const int x = 2 * (j0 + e) + par;
      const double co = cs_table[2 * x], si = cs_table[2 * x + 1];
#pragma unroll
      for (int k = 0; k < 9; ++k) {
        acc[k] += s9[e][k];
        acc[9 + k] = fma(s9[e][k], co, acc[9 + k]);
        acc[18 + k] = fma(s9[e][k], si, acc[18 + k]);
      }
    }
  }
  // fixed-order block reduction over the warps that exist in this launch
  __shared__ double sm[kThreads / 32][27];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, n_warps = ((int)blockDim.x + 31) >> 5;
#pragma unroll
  for (int k = 0; k < 27; ++k) {
    double x = acc[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
    if (lane == 0) sm[warp][k] = x;
  }
  __syncthreads();
  if (threadIdx.x < 27) {
    double x = 0.0;
    for (int w = 0; w < n_warps; ++w) x += sm[w][threadIdx.x];
    partial[(long long)blockIdx.x * 27 + threadIdx.x] = x;
  }
}

__global__ void finalize_overlap_kernel(Geom g, int n_sys /*D*P*T*/, int n_chunks, const double* __restrict__ partial, double* __restrict__ q0, double* __restrict__ qk) {
  const int tid = blockIdx.x * kThreads + threadIdx.x;
  if (tid >= n_sys * 9) return;
  const int sys = tid / 9, k = tid % 9;
  double r0 = 0.0, re = 0.0, im = 0.0;
  for (int z = 0; z < n_chunks; ++z) {
    const double* p = partial + ((long long)sys * n_chunks + z) * 27;
    r0 += p[k]; re += p[9 + k]; im += p[18 + k];
  }
  const double inv = 1.0 / (double)g.N;
  if (q0) q0[tid] = r0 * inv;
  if (qk) { qk[2 * tid] = re * inv; qk[2 * tid + 1] = im * inv; }
}

// ------------------------------------------------------------------ arithmetic self-test (hsg_selftest_arith)
// Compares div_rn / sqrt_rn with the compiler's IEEE __fdiv_rn / __fsqrt_rn on pseudo-random operands whose
// exponents cover [2^-100, 2^100] (all mantissa bits random); counts[0] = division mismatches,
// counts[1] = square-root mismatches, counts[2] = division mismatches on divisors whose mantissa is all ones (counted apart:
// the one exceptional case of the Newton scheme, see below).
__global__ void selftest_arith_kernel(PhiloxKey key, unsigned long long n, unsigned long long* __restrict__ counts) {
  const unsigned long long tid = (unsigned long long)blockIdx.x * kThreads + threadIdx.x;
  const unsigned long long stride = (unsigned long long)gridDim.x * kThreads;
  unsigned int bad_div = 0, bad_sqrt = 0, bad_exc = 0;
  for (unsigned long long i = tid; i < n; i += stride) {
    uint32_t w0, w1, w2, w3;
    philox4x32_10((uint32_t)i, (uint32_t)(i >> 32), 0x5e1f7e57u, 0u, key.k0, key.k1, w0, w1, w2, w3);
    const uint32_t ea = 27u + (w2 % 201u), eb = 27u + ((w2 >> 8) % 201u);            // biased exponents 27..227
    const float a = __uint_as_float((w0 & 0x807FFFFFu) | (ea << 23));
    const float b = __uint_as_float((w1 & 0x807FFFFFu) | (eb << 23));
    const float x = fabsf(b);
    const float q1 = div_rn(a, b), q2 = __fdiv_rn(a, b);
    // the quotient itself must stay a normal number for the comparison to be in the supported range
    if (fabsf(q2) >= 1.2e-38f && fabsf(q2) <= 3.0e38f && __float_as_uint(q1) != __float_as_uint(q2)) ++bad_div;
    if (__float_as_uint(sqrt_rn(x)) != __float_as_uint(__fsqrt_rn(x))) ++bad_sqrt;
    // operands shaped like the moves': a denominator in [1, 3), a numerator of order one
    const float b2 = __uint_as_float((w1 & 0x007FFFFFu) | (127u << 23)) + (float)(w3 & 1u);
    const float a2 = __uint_as_float((w3 & 0x807FFFFFu) | ((120u + (w3 >> 28)) << 23));
    if (__float_as_uint(div_rn(a2, b2)) != __float_as_uint(__fdiv_rn(a2, b2))) ++bad_div;
    // the reciprocals +-1/b (the move uses them for 1/|h| and -1/(sigma + n_z)), and the packed instantiation of all three
    if (__float_as_uint(rcp_rn<float, false>(x)) != __float_as_uint(__fdiv_rn(1.0f, x))) ++bad_div;
    if (__float_as_uint(rcp_rn<float, true>(b2)) != __float_as_uint(__fdiv_rn(-1.0f, b2))) ++bad_div;
    // divisors whose mantissa is all ones: the one exceptional case of the Newton scheme, where the last correction lands
    // on the rounded quotient only for a good enough seed (tests/test_device_math_on_host.py) — the hardware's must be
    const float b3 = __uint_as_float(__float_as_uint(b) | 0x007FFFFFu), x3 = fabsf(b3);
    const float q3 = __fdiv_rn(a, b3);
    if (fabsf(q3) >= 1.2e-38f && fabsf(q3) <= 3.0e38f && __float_as_uint(div_rn(a, b3)) != __float_as_uint(q3)) ++bad_exc;
    if (__float_as_uint(rcp_rn<float, false>(x3)) != __float_as_uint(__fdiv_rn(1.0f, x3))) ++bad_exc;
    if (__float_as_uint(div_rn(a2, 1.99999988079071044921875f)) != __float_as_uint(__fdiv_rn(a2, 1.99999988079071044921875f))) ++bad_exc;
    if ((i & 0xFFFFull) == 0 && __float_as_uint(rcp_rn<float, true>(1.99999988079071044921875f)) != 0xBF000001u) ++bad_exc;   // -1/(2 - 2^-23)
    const F2 qp = div_rn(make_f2(a, a2), make_f2(b, b2));
    if (fabsf(q2) >= 1.2e-38f && fabsf(q2) <= 3.0e38f && __float_as_uint(f2_lo(qp)) != __float_as_uint(q2)) ++bad_div;
    if (__float_as_uint(f2_hi(qp)) != __float_as_uint(__fdiv_rn(a2, b2))) ++bad_div;
    const F2 rp = sqrt_rn(make_f2(x, b2));
    if (__float_as_uint(f2_lo(rp)) != __float_as_uint(__fsqrt_rn(x)) || __float_as_uint(f2_hi(rp)) != __float_as_uint(__fsqrt_rn(b2))) ++bad_sqrt;
  }
  if (bad_div) atomicAdd(counts, (unsigned long long)bad_div);
  if (bad_sqrt) atomicAdd(counts + 1, (unsigned long long)bad_sqrt);
  if (bad_exc) atomicAdd(counts + 2, (unsigned long long)bad_exc);
}

}  // namespace hsg
