// hsg_observables.cuh — reductions beyond E / m / q^{mu nu}(k): the four-replica susceptibility summands of the field
// case (Eqs. 9-11), the chiral overlaps (Eqs. 12-13) and the parallel-tempering
// diagnostics of PAPER.md:197 / Fig. 3 (the tracker itself runs inside pt_swap_kernel, hsg_kernels.cuh).
#pragma once
#include "hsg_kernels.cuh"

namespace hsg {

// fixed-order block reduction of NV doubles per thread over the warps present in this launch -> dst[NV]
template <int NV>
__device__ __forceinline__ void block_reduce_store_n(const double (&v)[NV], double* __restrict__ dst) {
  __shared__ double sm[kThreads / 32][NV];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, n_warps = ((int)blockDim.x + 31) >> 5;
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
    for (int w = 0; w < n_warps; ++w) x += sm[w][threadIdx.x];
    dst[threadIdx.x] = x;
  }
}

// ------------------------------------------------------------------ field case, Eq. (10)
// In Eq. (10) site i carries the component index mu in both of its spin factors and site j the index nu, so with
//   A_ab(k) = sum_i (s_i^(a) . s_i^(b)) e^{ik x_i}          (a, b = replicas 1..4 = 0..3 of the sample, same temperature)
// chi_1 = |A_12|^2, chi_2 = A_13 conj(A_14), chi_3 = A_13 conj(A_24).  One block per (d, t, chunk of ZB planes) reads
// the four replicas once: partial[(d,t)][chunk][12] = for the pairs (12),(13),(14),(24): sum at k=0, re, im at k_min.
// Dot products from exact fp32 x fp32 products in fp64; k_min along x, so the phase is applied once per
// x column as in overlap_kernel.
template <int V>
__global__ void __launch_bounds__(kThreads, 2) field_trace_kernel(Geom g, int ZB, const float* __restrict__ spins, const int32_t* __restrict__ slot_of_temp,
                                                               const double* __restrict__ cs_table, double* __restrict__ partial) {
  const int L = g.L, Lh = g.Lh, qpr = Lh / V;
  const int n_chunks = (L + ZB - 1) / ZB;
  const int chunk = blockIdx.x % n_chunks;
  const int dt = blockIdx.x / n_chunks;         // d*T + t
  const int t = dt % g.T, d = dt / g.T;
  const float* S[4];
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    const int grp = d * g.O + r;
    S[r] = spins + (long long)(grp * g.T + slot_of_temp[grp * g.T + t]) * 3 * g.N;
  }
  const int z0 = chunk * ZB, nz = min(ZB, L - z0);
  const int RT = max(1, (int)blockDim.x / (2 * qpr));     // row lanes per x-parity
  double acc[12];
#pragma unroll
  for (int k = 0; k < 12; ++k) acc[k] = 0.0;
  // a thread keeps one x-parity and a group of V compact sites per pass; groups beyond blockDim are taken in further passes
  for (int item = threadIdx.x; item < 2 * qpr * RT; item += blockDim.x) {
    const int q = item % qpr, par = (item / qpr) & 1, r = item / (2 * qpr), j0 = q * V;
    double s4[V][4];
#pragma unroll
    for (int e = 0; e < V; ++e)
#pragma unroll
      for (int k = 0; k < 4; ++k) s4[e][k] = 0.0;
    for (int m = r; m < nz * L; m += RT) {
      const int y = m % L, z = z0 + m / L;
      const int c = (par + y + z) & 1;
      Vec<V> v[4][3];
#pragma unroll
      for (int rr = 0; rr < 4; ++rr)
#pragma unroll
        for (int mu = 0; mu < 3; ++mu) v[rr][mu] = ldv<V>(S[rr] + spin_index(g, z, c, mu, y, j0));
#pragma unroll
      for (int e = 0; e < V; ++e) {
        double x[4][3];
#pragma unroll
        for (int rr = 0; rr < 4; ++rr)
#pragma unroll
          for (int mu = 0; mu < 3; ++mu) x[rr][mu] = (double)v[rr][mu].v[e];
        // (the products are exact, so the fma chain equals three rounded additions in the order mu = x, y, z)
        s4[e][0] += fma(x[0][2], x[1][2], fma(x[0][1], x[1][1], x[0][0] * x[1][0]));   // (1).(2)
        s4[e][1] += fma(x[0][2], x[2][2], fma(x[0][1], x[2][1], x[0][0] * x[2][0]));   // (1).(3)
        s4[e][2] += fma(x[0][2], x[3][2], fma(x[0][1], x[3][1], x[0][0] * x[3][0]));   // (1).(4)
        s4[e][3] += fma(x[1][2], x[3][2], fma(x[1][1], x[3][1], x[1][0] * x[3][0]));   // (2).(4)
      }
    }
#pragma unroll
    for (int e = 0; e < V; ++e) {
      const int x = 2 * (j0 + e) + par;
      const double co = cs_table[2 * x], si = cs_table[2 * x + 1];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        acc[3 * k] += s4[e][k];
        acc[3 * k + 1] = fma(s4[e][k], co, acc[3 * k + 1]);
        acc[3 * k + 2] = fma(s4[e][k], si, acc[3 * k + 2]);
      }
    }
  }
  block_reduce_store_n<12>(acc, partial + (long long)blockIdx.x * 12);
}

// chi[(d,t)][2 (k = 0, k_min)][3 (chi_1, chi_2, chi_3)][2 (re, im)] from the chunk partials (fixed order)
__global__ void finalize_field_kernel(int n_dt, int n_chunks, const double* __restrict__ partial, double* __restrict__ chi) {
  const int dt = blockIdx.x * kThreads + threadIdx.x;
  if (dt >= n_dt) return;
  double A[12];
#pragma unroll
  for (int k = 0; k < 12; ++k) A[k] = 0.0;
  for (int c = 0; c < n_chunks; ++c) {
    const double* p = partial + ((long long)dt * n_chunks + c) * 12;
#pragma unroll
    for (int k = 0; k < 12; ++k) A[k] += p[k];
  }
  double* o = chi + (long long)dt * 12;
  // k = 0: A real
  o[0] = A[0] * A[0]; o[1] = 0.0;
  o[2] = A[3] * A[6]; o[3] = 0.0;
  o[4] = A[3] * A[9]; o[5] = 0.0;
  // k_min: A_p = (re, im) = (A[3p+1], A[3p+2])
  const double r12 = A[1], i12 = A[2], r13 = A[4], i13 = A[5], r14 = A[7], i14 = A[8], r24 = A[10], i24 = A[11];
  o[6] = r12 * r12 + i12 * i12; o[7] = 0.0;                          // |A_12|^2
  o[8] = r13 * r14 + i13 * i14; o[9] = i13 * r14 - r13 * i14;        // A_13 conj(A_14)
  o[10] = r13 * r24 + i13 * i24; o[11] = i13 * r24 - r13 * i24;      // A_13 conj(A_24)
}

// ------------------------------------------------------------------ chirality, Eqs. (12), (13)
// kappa_i^alpha = s_{i+alpha} . (s_i x s_{i-alpha}) in the spins' precision with the operation order of DESIGN.md §3.8:
//   c = b x m: c_x = fma(b_y, m_z, -(b_z m_y)), c_y = fma(b_z, m_x, -(b_x m_z)), c_z = fma(b_x, m_y, -(b_y m_x));
//   kappa = fma(p_z, c_z, fma(p_y, c_y, p_x c_x)),  p = s_{i+alpha}, b = s_i, m = s_{i-alpha}
__device__ __forceinline__ float chirality(const Vec3& p, const Vec3& b, const Vec3& m) {
  const float cx = __fmaf_rn(b.y, m.z, -__fmul_rn(b.z, m.y));
  const float cy = __fmaf_rn(b.z, m.x, -__fmul_rn(b.x, m.z));
  const float cz = __fmaf_rn(b.x, m.y, -__fmul_rn(b.y, m.x));
  return __fmaf_rn(p.z, cz, __fmaf_rn(p.y, cy, __fmul_rn(p.x, cx)));
}

// the three chiralities of the V sites x = 2(j0+e)+par of row (y,z) of one configuration (colour c = (par+y+z)&1)
template <int V>
__device__ __forceinline__ void chirality_row(const Geom& g, const float* __restrict__ S, int z, int y, int c, int par, int j0, float (&kap)[3][V]) {
  const int L = g.L, Lh = g.Lh, cc = 1 - c;
  const int yp = (y + 1 == L) ? 0 : y + 1, ym = (y == 0) ? L - 1 : y - 1;
  const int zp = (z + 1 == L) ? 0 : z + 1, zm = (z == 0) ? L - 1 : z - 1;
  // x neighbours are the other colour's sites of this row: par = 0: x-1 -> j-1, x+1 -> j;  par = 1: x-1 -> j, x+1 -> j+1
  const int jx = par ? ((j0 + V == Lh) ? 0 : j0 + V) : ((j0 == 0) ? Lh - 1 : j0 - 1);
  Vec<V> own[3], xq[3], syp[3], sym[3], szp[3], szm[3];
  float xe[3];
#pragma unroll
  for (int mu = 0; mu < 3; ++mu) {
    own[mu] = ldv<V>(S + spin_index(g, z, c, mu, y, j0));
    xq[mu] = ldv<V>(S + spin_index(g, z, cc, mu, y, j0));
    xe[mu] = S[spin_index(g, z, cc, mu, y, jx)];
    syp[mu] = ldv<V>(S + spin_index(g, z, cc, mu, yp, j0));
    sym[mu] = ldv<V>(S + spin_index(g, z, cc, mu, ym, j0));
    szp[mu] = ldv<V>(S + spin_index(g, zp, cc, mu, y, j0));
    szm[mu] = ldv<V>(S + spin_index(g, zm, cc, mu, y, j0));
  }
#pragma unroll
  for (int e = 0; e < V; ++e) {
    const Vec3 b = {own[0].v[e], own[1].v[e], own[2].v[e]};
    Vec3 xp, xm;
    float* fp = &xp.x; float* fm = &xm.x;
#pragma unroll
    for (int mu = 0; mu < 3; ++mu) {
      fp[mu] = par ? (e + 1 < V ? xq[mu].v[e + 1 < V ? e + 1 : 0] : xe[mu]) : xq[mu].v[e];
      fm[mu] = par ? xq[mu].v[e] : (e > 0 ? xq[mu].v[e > 0 ? e - 1 : 0] : xe[mu]);
    }
    kap[0][e] = chirality(xp, b, xm);
    kap[1][e] = chirality(Vec3{syp[0].v[e], syp[1].v[e], syp[2].v[e]}, b, Vec3{sym[0].v[e], sym[1].v[e], sym[2].v[e]});
    kap[2][e] = chirality(Vec3{szp[0].v[e], szp[1].v[e], szp[2].v[e]}, b, Vec3{szm[0].v[e], szm[1].v[e], szm[2].v[e]});
  }
}

// One block per (d, pair, t, chunk of ZB planes): partial[...][9] = for alpha = x, y, z: sum at k = 0, re, im at k_min of
// kappa^{alpha(a)} kappa^{alpha(b)} (product and sums in fp64).  Neighbours straight from global memory (L1/L2 reuse).
template <int V>
__global__ void __launch_bounds__(kThreads, 2) chiral_kernel(Geom g, int ZB, const float* __restrict__ spins, const int32_t* __restrict__ slot_of_temp,
                                                          const double* __restrict__ cs_table, double* __restrict__ partial) {
  const int L = g.L, Lh = g.Lh, qpr = Lh / V;
  const int P = g.O * (g.O - 1) / 2;
  const int n_chunks = (L + ZB - 1) / ZB;
  const int chunk = blockIdx.x % n_chunks;
  int rest = blockIdx.x / n_chunks;         // (d*P + p)*T + t
  const int t = rest % g.T; rest /= g.T;
  const int p = rest % P; const int d = rest / P;
  int a = 0, b = 1;
  { int k = p; a = 0; while (k >= g.O - 1 - a) { k -= g.O - 1 - a; ++a; } b = a + 1 + k; }
  const float* A = spins + (long long)((d * g.O + a) * g.T + slot_of_temp[(d * g.O + a) * g.T + t]) * 3 * g.N;
  const float* B = spins + (long long)((d * g.O + b) * g.T + slot_of_temp[(d * g.O + b) * g.T + t]) * 3 * g.N;
  const int z0 = chunk * ZB, nz = min(ZB, L - z0);
  const int RT = max(1, (int)blockDim.x / (2 * qpr));
  double acc[9];
#pragma unroll
  for (int k = 0; k < 9; ++k) acc[k] = 0.0;
  for (int item = threadIdx.x; item < 2 * qpr * RT; item += blockDim.x) {
    const int q = item % qpr, par = (item / qpr) & 1, r = item / (2 * qpr), j0 = q * V;
    double s3[V][3];
#pragma unroll
    for (int e = 0; e < V; ++e) { s3[e][0] = 0.0; s3[e][1] = 0.0; s3[e][2] = 0.0; }
    for (int m = r; m < nz * L; m += RT) {
      const int y = m % L, z = z0 + m / L;
      const int c = (par + y + z) & 1;
      float ka[3][V], kb[3][V];
      chirality_row<V>(g, A, z, y, c, par, j0, ka);
      chirality_row<V>(g, B, z, y, c, par, j0, kb);
#pragma unroll
      for (int e = 0; e < V; ++e)
#pragma unroll
        for (int al = 0; al < 3; ++al) s3[e][al] = fma((double)ka[al][e], (double)kb[al][e], s3[e][al]);
    }
#pragma unroll
    for (int e = 0; e < V; ++e) {
      const int x = 2 * (j0 + e) + par;
      const double co = cs_table[2 * x], si = cs_table[2 * x + 1];
#pragma unroll
      for (int al = 0; al < 3; ++al) {
        acc[3 * al] += s3[e][al];
        acc[3 * al + 1] = fma(s3[e][al], co, acc[3 * al + 1]);
        acc[3 * al + 2] = fma(s3[e][al], si, acc[3 * al + 2]);
      }
    }
  }
  block_reduce_store_n<9>(acc, partial + (long long)blockIdx.x * 9);
}

__global__ void finalize_chiral_kernel(Geom g, int n_sys /*D*P*T*/, int n_chunks, const double* __restrict__ partial, double* __restrict__ qc0, double* __restrict__ qck) {
  const int tid = blockIdx.x * kThreads + threadIdx.x;
  if (tid >= n_sys * 3) return;
  const int sys = tid / 3, al = tid % 3;
  double r0 = 0.0, re = 0.0, im = 0.0;
  for (int c = 0; c < n_chunks; ++c) {
    const double* p = partial + ((long long)sys * n_chunks + c) * 9 + 3 * al;
    r0 += p[0]; re += p[1]; im += p[2];
  }
  const double inv = 1.0 / (double)g.N;
  if (qc0) qc0[tid] = r0 * inv;
  if (qck) { qck[2 * tid] = re * inv; qck[2 * tid + 1] = im * inv; }
}

// ------------------------------------------------------------------ parallel-tempering diagnostics (Fig. 3)
// state per (d,o): moved[T] by temperature index, trav[T] and last_end[T] by configuration slot (pt_swap_kernel updates them)
__global__ void pt_diag_reset_kernel(Geom g, const int32_t* __restrict__ slot_of_temp, long long* moved, long long* trav, int32_t* last_end) {
  const int grp = blockIdx.x * kThreads + threadIdx.x;
  if (grp >= g.D * g.O) return;
  const int base = grp * g.T;
  for (int t = 0; t < g.T; ++t) { moved[base + t] = 0; trav[base + t] = 0; last_end[base + t] = 0; }
  pt_diag_touch(g.T, slot_of_temp + base, trav + base, last_end + base);
}

// p_diff[t] = sum_{d,o} moved[d][o][t] / (D O n_pass), fixed order
__global__ void pt_diag_pdiff_kernel(Geom g, unsigned long long n_pass, const long long* __restrict__ moved, double* __restrict__ p_diff) {
  const int t = blockIdx.x * kThreads + threadIdx.x;
  if (t >= g.T) return;
  double acc = 0.0;
  for (int grp = 0; grp < g.D * g.O; ++grp) acc += (double)moved[grp * g.T + t];
  p_diff[t] = n_pass ? acc / ((double)g.D * (double)g.O * (double)n_pass) : 0.0;
}

}  // namespace hsg
