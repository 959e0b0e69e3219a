// kernels_driver.cpp — runs the plain kernels of paper_1204_6192_b200/csrc/hsg_kernels.cuh and hsg_observables.cuh (unmodified)
// on the host execution model, with the launch shapes of csrc/hsg_shapes.h and the launch sequences of csrc/hsg_api.cu
// restated: layout conversion, start spins, the generic sweep kernel, energy / magnetisation / overlap reductions,
// parallel tempering with its diagnostics, field-case and chiral reductions.  Test infrastructure
// (tests/test_kernels_on_host.py); everything is host memory.
#include <cmath>
#include <vector>
#include "cuda_builtins.h"
#include "hsg_kernels.cuh"
#include "hsg_observables.cuh"
#include "hsg_shapes.h"

using namespace hsg;

namespace {

// kernels without barriers or shuffles: the threads of the grid one after the other in this OS thread
template <class F> void serial_grid(unsigned grid, unsigned block, F kernel) {
  gridDim.x = grid; blockDim.x = block;
  for (unsigned b = 0; b < grid; ++b)
    for (unsigned t = 0; t < block; ++t) { blockIdx.x = b; threadIdx.x = t; kernel(); }
}

struct Ctx {
  Geom g; PhiloxKey key; bool fast;
  std::vector<float> spins, jh, beta;
  std::vector<int32_t> slot_of_temp, temp_of_slot, diag_last;
  std::vector<double> cs, e_slot, m_slot, e_partial, q_partial;
  std::vector<long long> diag_moved, diag_trav;
  bool diag_on = false; unsigned long long diag_passes = 0, k_hb = 0, k_pt = 0;
  bool energy_valid = false;
};

void energy_mag(Ctx& c) {
  if (c.energy_valid) return;
  const Geom& g = c.g;
  const int V = vec_width(g), ZB = reduce_zb(g, V), n_chunks = (g.L + ZB - 1) / ZB;
  const unsigned nb = (unsigned)((long long)g.R * n_chunks);
  auto k = [&] {
    if (V == 4) energy_mag_kernel<4>(g, ZB, c.spins.data(), c.jh.data(), c.e_partial.data());
    else if (V == 2) energy_mag_kernel<2>(g, ZB, c.spins.data(), c.jh.data(), c.e_partial.data());
    else energy_mag_kernel<1>(g, ZB, c.spins.data(), c.jh.data(), c.e_partial.data());
  };
  emu::launch_grid(nb, kThreads, k);
  serial_grid(blocks_for((long long)g.R * 4), kThreads, [&] { finalize_energy_kernel(g, n_chunks, c.e_partial.data(), c.e_slot.data(), c.m_slot.data()); });
  c.energy_valid = true;
}

}  // namespace

extern "C" {

void* emuk_create(int L, int D, int O, int T, const float* temps, unsigned long long seed, unsigned long long sample_offset, int fast) {
  hsg::seed_jitter = 0;      // exact reciprocal seeds (the variable is shared with any other host build loaded in this process)
  Ctx* c = new Ctx();
  Geom& g = c->g;
  g.L = L; g.Lh = L / 2; g.ys = L == 64 ? 16 : L; g.D = D; g.O = O; g.T = T; g.R = D * O * T; g.N = (long long)L * L * L;
  g.sample_offset = sample_offset;
  c->key = PhiloxKey{(uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32)};
  c->fast = fast != 0;
  const size_t P = (size_t)O * (O - 1) / 2;
  c->spins.assign((size_t)3 * g.N * g.R, 0.0f); c->jh.assign((size_t)6 * g.N * D, 0.0f);
  c->beta.resize(T); c->cs.resize(2 * (size_t)L);
  for (int t = 0; t < T; ++t) c->beta[t] = (float)(1.0 / (double)temps[t]);
  for (int x = 0; x < L; ++x) { const double ph = 6.283185307179586476925286766559 * x / L; c->cs[2 * x] = std::cos(ph); c->cs[2 * x + 1] = std::sin(ph); }
  c->slot_of_temp.resize(g.R); c->temp_of_slot.resize(g.R); c->diag_last.assign(g.R, 0);
  c->e_slot.assign(g.R, 0.0); c->m_slot.assign((size_t)3 * g.R, 0.0);
  c->e_partial.assign((size_t)4 * g.R * L, 0.0); c->q_partial.assign((size_t)27 * D * (P ? P : 1) * T * L, 0.0);
  c->diag_moved.assign(g.R, 0); c->diag_trav.assign(g.R, 0);
  serial_grid(blocks_for(g.R), kThreads, [&] { init_perm_kernel(g, c->slot_of_temp.data(), c->temp_of_slot.data()); });
  return c;
}
void emuk_destroy(void* h) { delete (Ctx*)h; }

void emuk_set_disorder(void* h, const float* J, const float* H) {
  Ctx& c = *(Ctx*)h;
  serial_grid(blocks_for((long long)c.g.D * c.g.N), kThreads, [&] { pack_disorder_kernel(c.g, J, H, c.jh.data()); });
  c.energy_valid = false;
}
void emuk_init_spins(void* h) {
  Ctx& c = *(Ctx*)h;
  serial_grid(blocks_for((long long)c.g.R * c.g.N), kThreads, [&] { init_spins_kernel(c.g, c.key, c.temp_of_slot.data(), c.spins.data()); });
  c.energy_valid = false;
}
void emuk_set_spins(void* h, const float* S) {
  Ctx& c = *(Ctx*)h;
  serial_grid(blocks_for((long long)c.g.R * c.g.N), kThreads, [&] { convert_spins_kernel<true>(c.g, c.slot_of_temp.data(), c.spins.data(), const_cast<float*>(S)); });
  c.energy_valid = false;
}
void emuk_get_spins(void* h, float* S) {
  Ctx& c = *(Ctx*)h;
  serial_grid(blocks_for((long long)c.g.R * c.g.N), kThreads, [&] { convert_spins_kernel<false>(c.g, c.slot_of_temp.data(), c.spins.data(), S); });
}
void emuk_set_perm(void* h, const int32_t* perm) {
  Ctx& c = *(Ctx*)h;
  serial_grid(blocks_for(c.g.R), kThreads, [&] { set_perm_kernel(c.g, perm, c.slot_of_temp.data(), c.temp_of_slot.data()); });
}
void emuk_get_perm(void* h, int32_t* perm) { Ctx& c = *(Ctx*)h; for (int r = 0; r < c.g.R; ++r) perm[r] = c.slot_of_temp[r]; }

// hsg_sweep through the generic kernel: one launch per colour (launch_generic_sweep of hsg_api.cu)
void emuk_sweep_generic(void* h, int n_or, int n_hb) {
  Ctx& c = *(Ctx*)h; const Geom& g = c.g;
  const int V = vec_width(g);
  const long long n = (long long)g.R * g.L * g.L * (g.Lh / V);
  for (int s = 0; s < n_or + n_hb; ++s) {
    const bool hb = s >= n_or, fm = hb && c.fast;
    SweepArgs a{g, c.spins.data(), c.jh.data(), c.temp_of_slot.data(), c.beta.data(), c.key, c.k_hb};
    for (int colour = 0; colour < 2; ++colour) {
      auto k = [&] {
        if (V == 4) { if (fm) sweep_generic_kernel<4, true, true>(a, colour); else if (hb) sweep_generic_kernel<4, true>(a, colour); else sweep_generic_kernel<4, false>(a, colour); }
        else if (V == 2) { if (fm) sweep_generic_kernel<2, true, true>(a, colour); else if (hb) sweep_generic_kernel<2, true>(a, colour); else sweep_generic_kernel<2, false>(a, colour); }
        else { if (fm) sweep_generic_kernel<1, true, true>(a, colour); else if (hb) sweep_generic_kernel<1, true>(a, colour); else sweep_generic_kernel<1, false>(a, colour); }
      };
      serial_grid(blocks_for(n), kThreads, k);
    }
    if (hb) ++c.k_hb;
  }
  c.energy_valid = false;
}

void emuk_pt_swap(void* h, int32_t* accepted) {
  Ctx& c = *(Ctx*)h; const Geom& g = c.g;
  energy_mag(c);
  PtDiag diag = c.diag_on ? PtDiag{c.diag_moved.data(), c.diag_trav.data(), c.diag_last.data()} : PtDiag{nullptr, nullptr, nullptr};
  serial_grid(blocks_for((long long)g.D * g.O), kThreads, [&] {
    pt_swap_kernel(g, c.key, c.k_pt, c.beta.data(), c.e_slot.data(), c.slot_of_temp.data(), c.temp_of_slot.data(), accepted, diag);
  });
  ++c.k_pt;
  if (c.diag_on) ++c.diag_passes;
}

void emuk_measure(void* h, double* E, double* M, double* q0, double* qk) {
  Ctx& c = *(Ctx*)h; const Geom& g = c.g;
  if (E || M) {
    energy_mag(c);
    if (E) serial_grid(blocks_for(g.R), kThreads, [&] { gather_by_temp_kernel(g, 1, c.slot_of_temp.data(), c.e_slot.data(), E); });
    if (M) serial_grid(blocks_for((long long)g.R * 3), kThreads, [&] { gather_by_temp_kernel(g, 3, c.slot_of_temp.data(), c.m_slot.data(), M); });
  }
  const int P = g.O * (g.O - 1) / 2;
  if ((q0 || qk) && P > 0) {
    const long long n_sys = (long long)g.D * P * g.T;
    const int V = vec_width(g);
    int ZB, n_chunks, nt;
    reduction_shape(g, V, &ZB, &n_chunks, &nt);
    auto k = [&] {
      if (V == 4) overlap_kernel<4>(g, ZB, c.spins.data(), c.slot_of_temp.data(), c.cs.data(), c.q_partial.data());
      else if (V == 2) overlap_kernel<2>(g, ZB, c.spins.data(), c.slot_of_temp.data(), c.cs.data(), c.q_partial.data());
      else overlap_kernel<1>(g, ZB, c.spins.data(), c.slot_of_temp.data(), c.cs.data(), c.q_partial.data());
    };
    emu::launch_grid((unsigned)(n_sys * n_chunks), (unsigned)nt, k);
    serial_grid(blocks_for(n_sys * 9), kThreads, [&] { finalize_overlap_kernel(g, (int)n_sys, n_chunks, c.q_partial.data(), q0, qk); });
  }
}

int emuk_measure_field(void* h, double* chi) {
  Ctx& c = *(Ctx*)h; const Geom& g = c.g;
  if (g.O < 4) return -3;
  const int V = vec_width(g);
  int ZB, n_chunks, nt;
  reduction_shape(g, V, &ZB, &n_chunks, &nt);
  const int n_dt = g.D * g.T;
  auto k = [&] {
    if (V == 4) field_trace_kernel<4>(g, ZB, c.spins.data(), c.slot_of_temp.data(), c.cs.data(), c.q_partial.data());
    else if (V == 2) field_trace_kernel<2>(g, ZB, c.spins.data(), c.slot_of_temp.data(), c.cs.data(), c.q_partial.data());
    else field_trace_kernel<1>(g, ZB, c.spins.data(), c.slot_of_temp.data(), c.cs.data(), c.q_partial.data());
  };
  emu::launch_grid((unsigned)((long long)n_dt * n_chunks), (unsigned)nt, k);
  serial_grid(blocks_for(n_dt), kThreads, [&] { finalize_field_kernel(n_dt, n_chunks, c.q_partial.data(), chi); });
  return 0;
}

void emuk_measure_chiral(void* h, double* qc0, double* qck) {
  Ctx& c = *(Ctx*)h; const Geom& g = c.g;
  const int P = g.O * (g.O - 1) / 2;
  if (P == 0) return;
  const int V = vec_width(g);
  int ZB, n_chunks, nt;
  reduction_shape(g, V, &ZB, &n_chunks, &nt);
  const long long n_sys = (long long)g.D * P * g.T;
  auto k = [&] {
    if (V == 4) chiral_kernel<4>(g, ZB, c.spins.data(), c.slot_of_temp.data(), c.cs.data(), c.q_partial.data());
    else if (V == 2) chiral_kernel<2>(g, ZB, c.spins.data(), c.slot_of_temp.data(), c.cs.data(), c.q_partial.data());
    else chiral_kernel<1>(g, ZB, c.spins.data(), c.slot_of_temp.data(), c.cs.data(), c.q_partial.data());
  };
  emu::launch_grid((unsigned)(n_sys * n_chunks), (unsigned)nt, k);
  serial_grid(blocks_for(n_sys * 3), kThreads, [&] { finalize_chiral_kernel(g, (int)n_sys, n_chunks, c.q_partial.data(), qc0, qck); });
}

void emuk_diag_reset(void* h) {
  Ctx& c = *(Ctx*)h;
  serial_grid(blocks_for((long long)c.g.D * c.g.O), kThreads, [&] { pt_diag_reset_kernel(c.g, c.slot_of_temp.data(), c.diag_moved.data(), c.diag_trav.data(), c.diag_last.data()); });
  c.diag_on = true; c.diag_passes = 0;
}
unsigned long long emuk_diag_get(void* h, long long* moved, long long* trav, double* p_diff) {
  Ctx& c = *(Ctx*)h;
  for (int r = 0; r < c.g.R; ++r) { moved[r] = c.diag_moved[r]; trav[r] = c.diag_trav[r]; }
  serial_grid(blocks_for(c.g.T), kThreads, [&] { pt_diag_pdiff_kernel(c.g, c.diag_passes, c.diag_moved.data(), p_diff); });
  return c.diag_passes;
}

// hsg_selftest_arith on the host (IEEE division / square root of the host as the reference)
void emuk_selftest(unsigned long long seed, unsigned long long n, unsigned long long* counts) {
  counts[0] = counts[1] = counts[2] = 0;
  hsg::seed_jitter = 0;
  PhiloxKey key{(uint32_t)seed, (uint32_t)(seed >> 32)};
  serial_grid(4, kThreads, [&] { selftest_arith_kernel(key, n, counts); });
}

}  // extern "C"
