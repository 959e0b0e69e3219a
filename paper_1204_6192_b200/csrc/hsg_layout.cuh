// hsg_layout.cuh — private HBM layout of the engine.
//
// Checkerboard-compacted, plane-major SoA.  A site (x,y,z) has colour c = (x+y+z)&1 and compact
// x-index j = x>>1, i.e. x = 2j + ((y+z+c)&1); Lh = L/2.
//   spins of one configuration slot : S[z][c][mu][y][j]    fp32, 3N floats   (mu = spin component)
//   disorder of one sample          : JH[z][strip][a][y][j] fp32, 6N floats  a = jh_slot(c, k), k=0,1,2: J of
//                                     the bond from this site to +x,+y,+z ; k=3,4,5: H_x,H_y,H_z
// so that (i) all sites a colour update touches are unit-stride in j (128-bit vector loads, one
// colour never interleaved with the other), (ii) the four y/z neighbours of compact site j sit at the
// SAME j in the other colour's rows, the x neighbours at j and j-1 (or j+1), and (iii) one z-plane of
// one colour is a single contiguous block (3*L*Lh floats) that a bulk async copy can move.
#pragma once
#include <cstdint>

namespace hsg {

struct Geom {
  int L, Lh;          // lattice edge, L/2
  int ys;             // rows per strip of the J/H layout: L, or the strip height of the z-marching kernel (16 at L = 64)
  int D, O, T;        // samples, replicas, temperatures
  int R;              // D*O*T systems
  long long N;        // L^3
  unsigned long long sample_offset;
};

__host__ __device__ __forceinline__ long long row_elems(const Geom& g) { return g.Lh; }
__host__ __device__ __forceinline__ long long comp_elems(const Geom& g) { return (long long)g.L * g.Lh; }   // one [y][j] array
__host__ __device__ __forceinline__ long long spin_halfplane(const Geom& g) { return 3 * comp_elems(g); }
__host__ __device__ __forceinline__ long long spin_plane(const Geom& g) { return 6 * comp_elems(g); }
__host__ __device__ __forceinline__ long long jh_halfplane(const Geom& g) { return 6 * comp_elems(g); }
__host__ __device__ __forceinline__ long long jh_plane(const Geom& g) { return 12 * comp_elems(g); }

__host__ __device__ __forceinline__ long long spin_index(const Geom& g, int z, int c, int mu, int y, int j) {
  return (((long long)(z * 2 + c) * 3 + mu) * g.L + y) * g.Lh + j;
}
// Order of the twelve [y][j] arrays inside one J/H plane: everything a z-marching step needs for two steps
// first (11 arrays, one bulk copy), the +z couplings of colour 0 last (needed for three steps, ring of its own):
//   0,1: colour-0 Jx,Jy   2,3,4: colour-0 Hx,Hy,Hz   5,6,7: colour-1 Jx,Jy,Jz   8,9,10: colour-1 Hx,Hy,Hz   11: colour-0 Jz
__host__ __device__ __forceinline__ int jh_slot(int c, int k) {
  return c ? 5 + k : (k < 2 ? k : (k == 2 ? 11 : k - 1));
}
// Strip-major inside a plane: JH[z][y / ys][a][y % ys][j], so that the twelve arrays of one strip of one plane are one
// contiguous block (two bulk copies per step for a strip CTA of the z-marching kernel); ys = L: JH[z][a][y][j].
__host__ __device__ __forceinline__ long long jh_index(const Geom& g, int z, int c, int k, int y, int j) {
  const int strip = y / g.ys, r = y % g.ys;
  return ((((long long)z * (g.L / g.ys) + strip) * 12 + jh_slot(c, k)) * g.ys + r) * g.Lh + j;
}

}  // namespace hsg
