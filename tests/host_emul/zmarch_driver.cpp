// zmarch_driver.cpp — runs paper_1204_6192_b200/csrc/hsg_zmarch.cuh (the sweep kernel, unmodified) on the host execution model of
// emu.h: packs canonical J, H and spins into the kernel's private layout (hsg_layout.cuh), launches the kernel cluster by
// cluster the way hsg_zmarch_dispatch.cuh does (over-relaxation launch with V sites per thread, heat-bath launch with VHB),
// and unpacks.  One translation unit per lattice size: compile with -DEMU_L=8|16|32|64.  Test infrastructure.
#include <vector>
#include "hsg_zmarch.cuh"

using namespace hsg;

namespace {

template <int L, int YS, int V, int G, bool FM = false>
void launch(const ZmarchArgs& a) {
  using C = zm::Cfg<L, YS, V, G>;
  std::vector<uint32_t> mbars;
  for (uint32_t i = 0; i < 8; ++i) mbars.push_back(8u * i);          // NJB J/H barriers and two halo barriers (Cfg)
  const int n_groups = a.g.R / G;
  for (int grp = 0; grp < n_groups; ++grp) {                          // one cluster (or CTA) after the other
    emu::Launch ln(C::NCL, C::NT, C::smem_bytes, (unsigned)(grp * C::NCL), mbars);
    ln.run([&a] { zm::zmarch_kernel<L, YS, V, G, FM>(a); });
  }
}

// hsg_sweep(n_or, n_hb) as zmarch_launch_g makes it
template <int L, int G>
void sweep(const ZmarchArgs& a) {
  using T = zm::Tune<L>;
  if (T::VHB != T::V && a.n_hb > 0) {
    if (a.n_or > 0) { ZmarchArgs o = a; o.n_hb = 0; o.e_slot = nullptr; launch<L, T::YS, T::V, G>(o); }
    ZmarchArgs h = a; h.n_or = 0;
    if (a.fast_math) launch<L, T::YS, T::VHB, G, true>(h); else launch<L, T::YS, T::VHB, G>(h);
    return;
  }
  if constexpr (T::VHB == T::V) {
    if (a.fast_math && a.n_hb > 0) { launch<L, T::YS, T::V, G, true>(a); return; }
  }
  launch<L, T::YS, T::V, G>(a);
}

template <int L>
int dispatch(int G, const ZmarchArgs& a) {
  switch (G) {
    case 1: sweep<L, 1>(a); return 0;
    case 2: sweep<L, 2>(a); return 0;
#if EMU_L == 8 || EMU_L == 16
    case 4: sweep<L, 4>(a); return 0;
    case 8: sweep<L, 8>(a); return 0;
#endif
    default: return -1;
  }
}

}  // namespace

#define EMU_CAT2(a, b) a##b
#define EMU_CAT(a, b) EMU_CAT2(a, b)

// S: canonical spins [D][O][T][3][N] (configuration t of a chain holds temperature t), updated in place;
// E [R], M [R][3]: the fused reductions of the final sweep.  fast_math: HSG_FLAG_FAST_MATH.  mode: 0 = asynchronous copies land when issued, 1 = when waited for.
extern "C" int EMU_CAT(emu_zmarch_l, EMU_L)(int G, int mode, int D, int O, int T, const float* temps, unsigned long long seed,
                                             unsigned long long sample_offset, unsigned long long k_hb, int n_or, int n_hb,
                                             const float* J, const float* H, float* S, double* E, double* M, int fast_math) {
  constexpr int L = EMU_L;
  Geom g{};
  g.L = L; g.Lh = L / 2; g.ys = L == 64 ? 16 : L; g.D = D; g.O = O; g.T = T; g.R = D * O * T; g.N = (long long)L * L * L;
  g.sample_offset = sample_offset;
  if ((O * T) % G != 0) return -2;
  const long long N = g.N;
  std::vector<float> jh((size_t)6 * N * D), priv((size_t)3 * N * g.R), beta(T);
  std::vector<int32_t> temp_of_slot(g.R);
  for (int t = 0; t < T; ++t) beta[t] = (float)(1.0 / (double)temps[t]);
  for (int r = 0; r < g.R; ++r) temp_of_slot[r] = r % T;
  for (int d = 0; d < D; ++d)
    for (long long i = 0; i < N; ++i) {
      const int x = (int)(i % L), y = (int)((i / L) % L), z = (int)(i / ((long long)L * L));
      const int c = (x + y + z) & 1, j = x >> 1;
      for (int k = 0; k < 3; ++k) {
        jh[(size_t)d * 6 * N + jh_index(g, z, c, k, y, j)] = J[((size_t)d * 3 + k) * N + i];
        jh[(size_t)d * 6 * N + jh_index(g, z, c, 3 + k, y, j)] = H ? H[((size_t)d * 3 + k) * N + i] : 0.0f;
      }
    }
  auto convert = [&](bool to_private) {
    for (int r = 0; r < g.R; ++r)
      for (long long i = 0; i < N; ++i) {
        const int x = (int)(i % L), y = (int)((i / L) % L), z = (int)(i / ((long long)L * L));
        const int c = (x + y + z) & 1, j = x >> 1;
        for (int mu = 0; mu < 3; ++mu) {
          float& p = priv[(size_t)r * 3 * N + spin_index(g, z, c, mu, y, j)];
          float& q = S[(size_t)r * 3 * N + (size_t)mu * N + i];
          if (to_private) p = q; else q = p;
        }
      }
  };
  convert(true);
  std::vector<double> e_slot(g.R, 0.0), m_slot((size_t)3 * g.R, 0.0);
  ZmarchArgs a{g, priv.data(), jh.data(), temp_of_slot.data(), beta.data(), PhiloxKey{(uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32)},
               k_hb, n_or, n_hb, E ? e_slot.data() : nullptr, m_slot.data(), fast_math};
  emu::mode = mode;
  hsg::seed_jitter = 0;      // exact reciprocal seeds (the variable is shared with any other host build loaded in this process)
  const int rc = dispatch<L>(G, a);
  if (rc != 0) return rc;
  convert(false);
  if (E) for (int r = 0; r < g.R; ++r) E[r] = e_slot[r];
  if (M) for (size_t k = 0; k < m_slot.size(); ++k) M[k] = m_slot[k];
  return 0;
}
