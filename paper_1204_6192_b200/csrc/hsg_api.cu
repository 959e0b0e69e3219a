// hsg_api.cu — the C ABI of include/hsg.h: context bookkeeping and kernel launches.
// All device work is enqueued on the stream given at hsg_create(); nothing here synchronises.
#include "../../include/hsg.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "hsg_kernels.cuh"
#include "hsg_observables.cuh"
#include "hsg_shapes.h"
#include "hsg_zmarch_launch.h"

using namespace hsg;

namespace {

constexpr size_t kAlign = 256;
inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

// carve-up of the caller's two buffers (offsets in bytes)
struct StateLayout {
  size_t spins, jh, slot_of_temp, temp_of_slot, beta, cs_table, e_slot, m_slot, diag_moved, diag_trav, diag_last, total;
};
struct ScratchLayout {
  size_t e_partial, q_partial, total;
};

StateLayout state_layout(const Geom& g) {
  StateLayout s{};
  size_t o = 0;
  s.spins = o;        o = align_up(o + sizeof(float) * 3 * (size_t)g.N * g.R);
  s.jh = o;           o = align_up(o + sizeof(float) * 6 * (size_t)g.N * g.D);
  s.slot_of_temp = o; o = align_up(o + sizeof(int32_t) * g.R);
  s.temp_of_slot = o; o = align_up(o + sizeof(int32_t) * g.R);
  s.beta = o;         o = align_up(o + sizeof(float) * g.T);
  s.cs_table = o;     o = align_up(o + sizeof(double) * 2 * g.L);
  s.e_slot = o;       o = align_up(o + sizeof(double) * g.R);
  s.m_slot = o;       o = align_up(o + sizeof(double) * 3 * g.R);
  s.diag_moved = o;   o = align_up(o + sizeof(long long) * g.R);
  s.diag_trav = o;    o = align_up(o + sizeof(long long) * g.R);
  s.diag_last = o;    o = align_up(o + sizeof(int32_t) * g.R);
  s.total = o;
  return s;
}
ScratchLayout scratch_layout(const Geom& g) {
  ScratchLayout s{};
  const size_t P = (size_t)g.O * (g.O - 1) / 2;
  size_t o = 0;
  s.e_partial = o; o = align_up(o + sizeof(double) * 4 * (size_t)g.R * g.L);
  // 27 doubles per (d, pair, t, chunk) for the overlaps; also used for the chiral (9) and field-case (12 per (d, t, chunk)) partials
  s.q_partial = o; o = align_up(o + sizeof(double) * 27 * (size_t)g.D * (P > 0 ? P : 1) * g.T * g.L);
  s.total = o;
  return s;
}

int check_desc(const hsg_desc* d) {
  if (!d || !d->temps_host) return HSG_EINVAL;
  if (d->L < 2 || (d->L & 1) || d->n_samples < 1 || d->n_replicas < 1 || d->n_temps < 1) return HSG_EINVAL;
  if (d->flags & ~(uint32_t)HSG_FLAG_FAST_MATH) return HSG_EINVAL;
  for (int t = 0; t < d->n_temps; ++t) {
    if (!(d->temps_host[t] > 0.0f) || !std::isfinite(d->temps_host[t])) return HSG_EINVAL;
    if (t > 0 && !(d->temps_host[t] > d->temps_host[t - 1])) return HSG_EINVAL;
  }
  const double n = (double)d->L * d->L * d->L;
  if (n > 2147483647.0) return HSG_EINVAL;                                   // site index is the 32-bit Philox word c0
  if ((double)d->n_samples * d->n_replicas * d->n_temps > 1.0e9) return HSG_EINVAL;
  // the global system id ((sample_offset + d) * O + o) * T + t is a 32-bit word of the random-stream counter
  if (((double)d->sample_offset + (double)d->n_samples) * d->n_replicas * d->n_temps >= 4294967296.0) return HSG_EINVAL;
  return HSG_OK;
}

Geom make_geom(const hsg_desc* d) {
  Geom g{};
  g.L = d->L; g.Lh = d->L / 2;
  g.ys = d->L == 64 ? 16 : d->L;           // strips of the J/H layout (hsg_layout.cuh) = strips of zmarch_kernel<64,16,..>
  g.D = d->n_samples; g.O = d->n_replicas; g.T = d->n_temps;
  g.R = g.D * g.O * g.T;
  g.N = (long long)d->L * d->L * d->L;
  g.sample_offset = d->sample_offset;
  return g;
}


}  // namespace

struct hsg_ctx {
  Geom g;
  PhiloxKey key;
  cudaStream_t stream;
  // device pointers into the caller's buffers
  float* spins; float* jh; int32_t* slot_of_temp; int32_t* temp_of_slot; float* beta; double* cs_table;
  double* e_slot; double* m_slot; double* e_partial; double* q_partial;
  long long* diag_moved; long long* diag_trav; int32_t* diag_last;     // parallel-tempering diagnostics (hsg_pt_diag_*)
  bool diag_on; unsigned long long diag_passes;
  unsigned long long k_hb, k_pt;
  bool have_disorder, have_spins;
  bool energy_valid;            // e_slot / m_slot hold the reduction of the current spins
  int device;                   // CUDA device the context was created on (current at every call: hsg.h)
  int sm_count;                 // its number of SMs (grid sizing of the sweep kernels)
  int sweep_kernel_opt;
  bool fuse_energy;             // zmarch: reduce E and m in the final sweep of every hsg_sweep call
  bool fast_math;               // HSG_FLAG_FAST_MATH: heat-bath sweeps draw with the special-function unit
  const char* last_kernel;
  unsigned long long launches;
  std::string err;
};

// every call on a context: non-null, and the device it was created on is current (hsg.h)
#define HSG_ENTER(ctx) do { if (!(ctx)) return HSG_EINVAL; int dev_ = -1; \
  if (cudaGetDevice(&dev_) != cudaSuccess || dev_ != (ctx)->device) { \
    (ctx)->err = "the CUDA device current at hsg_create() (" + std::to_string((ctx)->device) + ") is not current (" + std::to_string(dev_) + ")"; \
    return HSG_ESTATE; } } while (0)
#define HSG_FAIL(ctx, code, msg) do { (ctx)->err = (msg); return (code); } while (0)
#define HSG_CUDA(ctx, expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) { \
  (ctx)->err = std::string(#expr) + ": " + cudaGetErrorString(e_); return HSG_ECUDA; } } while (0)
#define HSG_LAUNCHED(ctx) do { ++(ctx)->launches; cudaError_t e_ = cudaGetLastError(); if (e_ != cudaSuccess) { \
  (ctx)->err = std::string("kernel launch: ") + cudaGetErrorString(e_); return HSG_ECUDA; } } while (0)

extern "C" {

const char* hsg_version(void) { return "hsg 0.2 (sm_100a)"; }

int hsg_query_bytes(const hsg_desc* desc, size_t* state_bytes, size_t* scratch_bytes) {
  const int rc = check_desc(desc);
  if (rc != HSG_OK) return rc;
  const Geom g = make_geom(desc);
  if (state_bytes) *state_bytes = state_layout(g).total;
  if (scratch_bytes) *scratch_bytes = scratch_layout(g).total;
  return HSG_OK;
}

int hsg_create(const hsg_desc* desc, void* dev_state, size_t state_bytes, void* dev_scratch, size_t scratch_bytes,
               void* cuda_stream, hsg_ctx** out) {
  if (!out) return HSG_EINVAL;
  *out = nullptr;
  const int rc = check_desc(desc);
  if (rc != HSG_OK) return rc;
  const Geom g = make_geom(desc);
  const StateLayout sl = state_layout(g);
  const ScratchLayout cl = scratch_layout(g);
  if (!dev_state || !dev_scratch || state_bytes < sl.total || scratch_bytes < cl.total) return HSG_EINVAL;
  if (((uintptr_t)dev_state % kAlign) || ((uintptr_t)dev_scratch % kAlign)) return HSG_EINVAL;
  hsg_ctx* c = new (std::nothrow) hsg_ctx();
  if (!c) return HSG_EINVAL;
  c->g = g;
  if (cudaGetDevice(&c->device) != cudaSuccess ||
      cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, c->device) != cudaSuccess) { delete c; return HSG_ECUDA; }
  c->key.k0 = (uint32_t)(desc->seed & 0xFFFFFFFFull);
  c->key.k1 = (uint32_t)(desc->seed >> 32);
  c->stream = (cudaStream_t)cuda_stream;
  char* s = (char*)dev_state; char* w = (char*)dev_scratch;
  c->spins = (float*)(s + sl.spins); c->jh = (float*)(s + sl.jh);
  c->slot_of_temp = (int32_t*)(s + sl.slot_of_temp); c->temp_of_slot = (int32_t*)(s + sl.temp_of_slot);
  c->beta = (float*)(s + sl.beta); c->cs_table = (double*)(s + sl.cs_table);
  c->e_slot = (double*)(s + sl.e_slot); c->m_slot = (double*)(s + sl.m_slot);
  c->e_partial = (double*)(w + cl.e_partial); c->q_partial = (double*)(w + cl.q_partial);
  c->diag_moved = (long long*)(s + sl.diag_moved); c->diag_trav = (long long*)(s + sl.diag_trav); c->diag_last = (int32_t*)(s + sl.diag_last);
  c->diag_on = false; c->diag_passes = 0;
  c->k_hb = 0; c->k_pt = 0; c->have_disorder = false; c->have_spins = false; c->energy_valid = false;
  c->sweep_kernel_opt = HSG_KERNEL_AUTO; c->fuse_energy = true; c->last_kernel = "none"; c->launches = 0;
  c->fast_math = (desc->flags & HSG_FLAG_FAST_MATH) != 0;

  // small host-computed tables: beta_t = (float)(1.0/(double)T_t); cos/sin(2 pi x / L) in fp64
  std::vector<float> beta(g.T);
  for (int t = 0; t < g.T; ++t) beta[t] = (float)(1.0 / (double)desc->temps_host[t]);
  std::vector<double> cs(2 * (size_t)g.L);
  const double two_pi = 6.283185307179586476925286766559;
  for (int x = 0; x < g.L; ++x) {
    const double ph = two_pi * (double)x / (double)g.L;
    cs[2 * x] = std::cos(ph); cs[2 * x + 1] = std::sin(ph);
  }
  // pageable host memory: cudaMemcpyAsync stages it before returning, so the vectors may go out of scope
  cudaError_t e = cudaMemcpyAsync(c->beta, beta.data(), sizeof(float) * g.T, cudaMemcpyHostToDevice, c->stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(c->cs_table, cs.data(), sizeof(double) * cs.size(), cudaMemcpyHostToDevice, c->stream);
  if (e != cudaSuccess) { delete c; return HSG_ECUDA; }
  init_perm_kernel<<<blocks_for(g.R), kThreads, 0, c->stream>>>(g, c->slot_of_temp, c->temp_of_slot);
  ++c->launches;
  if (cudaGetLastError() != cudaSuccess) { delete c; return HSG_ECUDA; }
  *out = c;
  return HSG_OK;
}

int hsg_destroy(hsg_ctx* ctx) {
  if (!ctx) return HSG_EINVAL;
  delete ctx;
  return HSG_OK;
}

const char* hsg_last_error(const hsg_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }
uint64_t hsg_launch_count(const hsg_ctx* ctx) { return ctx ? ctx->launches : 0; }
const char* hsg_last_sweep_kernel(const hsg_ctx* ctx) { return ctx ? ctx->last_kernel : "none"; }

int hsg_set_option(hsg_ctx* ctx, int option, int value) {
  if (!ctx) return HSG_EINVAL;
  if (option == HSG_OPT_SWEEP_KERNEL) {
    if (value < HSG_KERNEL_AUTO || value > HSG_KERNEL_ZMARCH) HSG_FAIL(ctx, HSG_EINVAL, "unknown sweep kernel");
    if (value == HSG_KERNEL_ZMARCH && !zmarch_supported(ctx->g)) HSG_FAIL(ctx, HSG_EUNSUPPORTED, "zmarch kernel does not support this geometry");
    ctx->sweep_kernel_opt = value;
    return HSG_OK;
  }
  if (option == HSG_OPT_FUSE_ENERGY) {
    ctx->fuse_energy = value != 0;
    return HSG_OK;
  }
  HSG_FAIL(ctx, HSG_EINVAL, "unknown option");
}

int hsg_set_disorder(hsg_ctx* ctx, const float* J_dev, const float* H_dev) {
  HSG_ENTER(ctx);
  if (!J_dev) HSG_FAIL(ctx, HSG_EINVAL, "J_dev is null");
  pack_disorder_kernel<<<blocks_for((long long)ctx->g.D * ctx->g.N), kThreads, 0, ctx->stream>>>(ctx->g, J_dev, H_dev, ctx->jh);
  HSG_LAUNCHED(ctx);
  ctx->have_disorder = true;
  ctx->energy_valid = false;
  return HSG_OK;
}

int hsg_init_spins(hsg_ctx* ctx) {
  HSG_ENTER(ctx);
  init_spins_kernel<<<blocks_for((long long)ctx->g.R * ctx->g.N), kThreads, 0, ctx->stream>>>(ctx->g, ctx->key, ctx->temp_of_slot, ctx->spins);
  HSG_LAUNCHED(ctx);
  ctx->have_spins = true;
  ctx->energy_valid = false;
  return HSG_OK;
}

int hsg_set_spins(hsg_ctx* ctx, const float* S_dev) {
  HSG_ENTER(ctx);
  if (!S_dev) HSG_FAIL(ctx, HSG_EINVAL, "S_dev is null");
  convert_spins_kernel<true><<<blocks_for((long long)ctx->g.R * ctx->g.N), kThreads, 0, ctx->stream>>>(
      ctx->g, ctx->slot_of_temp, ctx->spins, const_cast<float*>(S_dev));
  HSG_LAUNCHED(ctx);
  ctx->have_spins = true;
  ctx->energy_valid = false;
  return HSG_OK;
}

int hsg_get_spins(hsg_ctx* ctx, float* S_dev) {
  HSG_ENTER(ctx);
  if (!S_dev) HSG_FAIL(ctx, HSG_EINVAL, "S_dev is null");
  if (!ctx->have_spins) HSG_FAIL(ctx, HSG_ESTATE, "spins not set");
  convert_spins_kernel<false><<<blocks_for((long long)ctx->g.R * ctx->g.N), kThreads, 0, ctx->stream>>>(
      ctx->g, ctx->slot_of_temp, ctx->spins, S_dev);
  HSG_LAUNCHED(ctx);
  return HSG_OK;
}

// ------------------------------------------------------------------ sweeps
static int launch_generic_sweep(hsg_ctx* ctx, bool hb) {
  const Geom& g = ctx->g;
  SweepArgs a{g, ctx->spins, ctx->jh, ctx->temp_of_slot, ctx->beta, ctx->key, ctx->k_hb};
  const int V = (g.Lh % 4 == 0) ? 4 : (g.Lh % 2 == 0) ? 2 : 1;
  const long long n = (long long)g.R * g.L * g.L * (g.Lh / V);
  for (int colour = 0; colour < 2; ++colour) {
    const unsigned nb = blocks_for(n);
    const bool fm = hb && ctx->fast_math;
    if (V == 4) { if (fm) sweep_generic_kernel<4, true, true><<<nb, kThreads, 0, ctx->stream>>>(a, colour); else if (hb) sweep_generic_kernel<4, true><<<nb, kThreads, 0, ctx->stream>>>(a, colour); else sweep_generic_kernel<4, false><<<nb, kThreads, 0, ctx->stream>>>(a, colour); }
    else if (V == 2) { if (fm) sweep_generic_kernel<2, true, true><<<nb, kThreads, 0, ctx->stream>>>(a, colour); else if (hb) sweep_generic_kernel<2, true><<<nb, kThreads, 0, ctx->stream>>>(a, colour); else sweep_generic_kernel<2, false><<<nb, kThreads, 0, ctx->stream>>>(a, colour); }
    else { if (fm) sweep_generic_kernel<1, true, true><<<nb, kThreads, 0, ctx->stream>>>(a, colour); else if (hb) sweep_generic_kernel<1, true><<<nb, kThreads, 0, ctx->stream>>>(a, colour); else sweep_generic_kernel<1, false><<<nb, kThreads, 0, ctx->stream>>>(a, colour); }
    HSG_LAUNCHED(ctx);
  }
  return HSG_OK;
}

int hsg_sweep(hsg_ctx* ctx, int n_or, int n_hb) {
  HSG_ENTER(ctx);
  if (n_or < 0 || n_hb < 0) HSG_FAIL(ctx, HSG_EINVAL, "negative sweep count");
  if (!ctx->have_disorder || !ctx->have_spins) HSG_FAIL(ctx, HSG_ESTATE, "hsg_sweep before disorder and spins were set");
  if (n_or + n_hb == 0) return HSG_OK;
  ctx->energy_valid = false;
  int kernel = ctx->sweep_kernel_opt;
  if (kernel == HSG_KERNEL_AUTO) kernel = zmarch_supported(ctx->g) ? HSG_KERNEL_ZMARCH : HSG_KERNEL_GENERIC;
  if (kernel == HSG_KERNEL_ZMARCH) {
    // the final sweep of the call also reduces E and m of every slot
    ZmarchArgs a{ctx->g, ctx->spins, ctx->jh, ctx->temp_of_slot, ctx->beta, ctx->key, ctx->k_hb, n_or, n_hb,
                 ctx->fuse_energy ? ctx->e_slot : nullptr, ctx->m_slot, ctx->fast_math ? 1 : 0};
    int n_launch = 0;
    const cudaError_t e = zmarch_launch(a, ctx->stream, &n_launch, ctx->sm_count);
    ctx->launches += (unsigned long long)n_launch;
    if (e != cudaSuccess) { ctx->err = std::string("zmarch launch: ") + cudaGetErrorString(e); return HSG_ECUDA; }
    ctx->k_hb += (unsigned long long)n_hb;
    ctx->last_kernel = "zmarch";
    ctx->energy_valid = ctx->fuse_energy;
    return HSG_OK;
  }
  for (int s = 0; s < n_or; ++s) { const int rc = launch_generic_sweep(ctx, false); if (rc != HSG_OK) return rc; }
  for (int s = 0; s < n_hb; ++s) {
    const int rc = launch_generic_sweep(ctx, true);
    if (rc != HSG_OK) return rc;
    ++ctx->k_hb;
  }
  ctx->last_kernel = "generic";
  return HSG_OK;
}

// ------------------------------------------------------------------ energy, parallel tempering, measurements
static int enqueue_energy_mag(hsg_ctx* ctx) {
  const Geom& g = ctx->g;
  if (ctx->energy_valid) return HSG_OK;          // spins unchanged since the last reduction
  const int V = vec_width(g), ZB = reduce_zb(g, V), n_chunks = (g.L + ZB - 1) / ZB;
  const unsigned nb = (unsigned)((long long)g.R * n_chunks);
  if (V == 4) energy_mag_kernel<4><<<nb, kThreads, 0, ctx->stream>>>(g, ZB, ctx->spins, ctx->jh, ctx->e_partial);
  else if (V == 2) energy_mag_kernel<2><<<nb, kThreads, 0, ctx->stream>>>(g, ZB, ctx->spins, ctx->jh, ctx->e_partial);
  else energy_mag_kernel<1><<<nb, kThreads, 0, ctx->stream>>>(g, ZB, ctx->spins, ctx->jh, ctx->e_partial);
  HSG_LAUNCHED(ctx);
  finalize_energy_kernel<<<blocks_for((long long)g.R * 4), kThreads, 0, ctx->stream>>>(g, n_chunks, ctx->e_partial, ctx->e_slot, ctx->m_slot);
  HSG_LAUNCHED(ctx);
  ctx->energy_valid = true;
  return HSG_OK;
}

int hsg_energy(hsg_ctx* ctx, double* E_dev) {
  HSG_ENTER(ctx);
  if (!E_dev) HSG_FAIL(ctx, HSG_EINVAL, "E_dev is null");
  if (!ctx->have_disorder || !ctx->have_spins) HSG_FAIL(ctx, HSG_ESTATE, "hsg_energy before disorder and spins were set");
  const int rc = enqueue_energy_mag(ctx);
  if (rc != HSG_OK) return rc;
  gather_by_temp_kernel<<<blocks_for(ctx->g.R), kThreads, 0, ctx->stream>>>(ctx->g, 1, ctx->slot_of_temp, ctx->e_slot, E_dev);
  HSG_LAUNCHED(ctx);
  return HSG_OK;
}

int hsg_pt_swap(hsg_ctx* ctx, int32_t* accepted_dev) {
  HSG_ENTER(ctx);
  if (!ctx->have_disorder || !ctx->have_spins) HSG_FAIL(ctx, HSG_ESTATE, "hsg_pt_swap before disorder and spins were set");
  const int rc = enqueue_energy_mag(ctx);
  if (rc != HSG_OK) return rc;
  pt_swap_kernel<<<blocks_for((long long)ctx->g.D * ctx->g.O), kThreads, 0, ctx->stream>>>(
      ctx->g, ctx->key, ctx->k_pt, ctx->beta, ctx->e_slot, ctx->slot_of_temp, ctx->temp_of_slot, accepted_dev,
      ctx->diag_on ? PtDiag{ctx->diag_moved, ctx->diag_trav, ctx->diag_last} : PtDiag{nullptr, nullptr, nullptr});
  HSG_LAUNCHED(ctx);
  ++ctx->k_pt;
  if (ctx->diag_on) ++ctx->diag_passes;
  return HSG_OK;
}

int hsg_measure(hsg_ctx* ctx, double* E_dev, double* M_dev, double* q0_dev, double* qk_dev) {
  HSG_ENTER(ctx);
  if (!ctx->have_disorder || !ctx->have_spins) HSG_FAIL(ctx, HSG_ESTATE, "hsg_measure before disorder and spins were set");
  const Geom& g = ctx->g;
  if (E_dev || M_dev) {
    const int rc = enqueue_energy_mag(ctx);
    if (rc != HSG_OK) return rc;
    if (E_dev) { gather_by_temp_kernel<<<blocks_for(g.R), kThreads, 0, ctx->stream>>>(g, 1, ctx->slot_of_temp, ctx->e_slot, E_dev); HSG_LAUNCHED(ctx); }
    if (M_dev) { gather_by_temp_kernel<<<blocks_for((long long)g.R * 3), kThreads, 0, ctx->stream>>>(g, 3, ctx->slot_of_temp, ctx->m_slot, M_dev); HSG_LAUNCHED(ctx); }
  }
  const int P = g.O * (g.O - 1) / 2;
  if ((q0_dev || qk_dev) && P > 0) {
    const long long n_sys = (long long)g.D * P * g.T;
    const int V = vec_width(g);
    int ZB, n_chunks, nt;
    reduction_shape(g, V, &ZB, &n_chunks, &nt);
    const unsigned nb = (unsigned)(n_sys * n_chunks);
    if (V == 4) overlap_kernel<4><<<nb, nt, 0, ctx->stream>>>(g, ZB, ctx->spins, ctx->slot_of_temp, ctx->cs_table, ctx->q_partial);
    else if (V == 2) overlap_kernel<2><<<nb, nt, 0, ctx->stream>>>(g, ZB, ctx->spins, ctx->slot_of_temp, ctx->cs_table, ctx->q_partial);
    else overlap_kernel<1><<<nb, nt, 0, ctx->stream>>>(g, ZB, ctx->spins, ctx->slot_of_temp, ctx->cs_table, ctx->q_partial);
    HSG_LAUNCHED(ctx);
    finalize_overlap_kernel<<<blocks_for(n_sys * 9), kThreads, 0, ctx->stream>>>(g, (int)n_sys, n_chunks, ctx->q_partial, q0_dev, qk_dev);
    HSG_LAUNCHED(ctx);
  }
  return HSG_OK;
}

// ------------------------------------------------------------------ field case, chirality, PT diagnostics
int hsg_measure_field(hsg_ctx* ctx, double* chi_dev) {
  HSG_ENTER(ctx);
  if (!chi_dev) HSG_FAIL(ctx, HSG_EINVAL, "chi_dev is null");
  if (!ctx->have_spins) HSG_FAIL(ctx, HSG_ESTATE, "hsg_measure_field before spins were set");
  const Geom& g = ctx->g;
  if (g.O < 4) HSG_FAIL(ctx, HSG_EUNSUPPORTED, "hsg_measure_field needs four replicas (PAPER.md:77)");
  const int V = vec_width(g);
  int ZB, n_chunks, nt;
  reduction_shape(g, V, &ZB, &n_chunks, &nt);
  const int n_dt = g.D * g.T;
  const unsigned nb = (unsigned)((long long)n_dt * n_chunks);
  if (V == 4) field_trace_kernel<4><<<nb, nt, 0, ctx->stream>>>(g, ZB, ctx->spins, ctx->slot_of_temp, ctx->cs_table, ctx->q_partial);
  else if (V == 2) field_trace_kernel<2><<<nb, nt, 0, ctx->stream>>>(g, ZB, ctx->spins, ctx->slot_of_temp, ctx->cs_table, ctx->q_partial);
  else field_trace_kernel<1><<<nb, nt, 0, ctx->stream>>>(g, ZB, ctx->spins, ctx->slot_of_temp, ctx->cs_table, ctx->q_partial);
  HSG_LAUNCHED(ctx);
  finalize_field_kernel<<<blocks_for(n_dt), kThreads, 0, ctx->stream>>>(n_dt, n_chunks, ctx->q_partial, chi_dev);
  HSG_LAUNCHED(ctx);
  return HSG_OK;
}

int hsg_measure_chiral(hsg_ctx* ctx, double* qc0_dev, double* qck_dev) {
  HSG_ENTER(ctx);
  if (!ctx->have_spins) HSG_FAIL(ctx, HSG_ESTATE, "hsg_measure_chiral before spins were set");
  const Geom& g = ctx->g;
  const int P = g.O * (g.O - 1) / 2;
  if (P == 0 || (!qc0_dev && !qck_dev)) return HSG_OK;
  const int V = vec_width(g);
  int ZB, n_chunks, nt;
  reduction_shape(g, V, &ZB, &n_chunks, &nt);
  const long long n_sys = (long long)g.D * P * g.T;
  const unsigned nb = (unsigned)(n_sys * n_chunks);
  if (V == 4) chiral_kernel<4><<<nb, nt, 0, ctx->stream>>>(g, ZB, ctx->spins, ctx->slot_of_temp, ctx->cs_table, ctx->q_partial);
  else if (V == 2) chiral_kernel<2><<<nb, nt, 0, ctx->stream>>>(g, ZB, ctx->spins, ctx->slot_of_temp, ctx->cs_table, ctx->q_partial);
  else chiral_kernel<1><<<nb, nt, 0, ctx->stream>>>(g, ZB, ctx->spins, ctx->slot_of_temp, ctx->cs_table, ctx->q_partial);
  HSG_LAUNCHED(ctx);
  finalize_chiral_kernel<<<blocks_for(n_sys * 3), kThreads, 0, ctx->stream>>>(g, (int)n_sys, n_chunks, ctx->q_partial, qc0_dev, qck_dev);
  HSG_LAUNCHED(ctx);
  return HSG_OK;
}

int hsg_xi_second_moment(double chi_0, double chi_kmin, int32_t L, double* xi_host) {
  if (!xi_host || L < 2 || !(chi_kmin > 0.0) || !(chi_0 >= chi_kmin)) return HSG_EINVAL;
  const double kmin = 6.283185307179586476925286766559 / (double)L;
  *xi_host = std::sqrt(chi_0 / chi_kmin - 1.0) / (2.0 * std::sin(0.5 * kmin));
  return HSG_OK;
}

int hsg_pt_diag_reset(hsg_ctx* ctx) {
  HSG_ENTER(ctx);
  pt_diag_reset_kernel<<<blocks_for((long long)ctx->g.D * ctx->g.O), kThreads, 0, ctx->stream>>>(
      ctx->g, ctx->slot_of_temp, ctx->diag_moved, ctx->diag_trav, ctx->diag_last);
  HSG_LAUNCHED(ctx);
  ctx->diag_on = true; ctx->diag_passes = 0;
  return HSG_OK;
}

int hsg_pt_diag_get(hsg_ctx* ctx, int64_t* moved_dev, int64_t* traversals_dev, double* p_diff_dev, uint64_t* n_pass_host) {
  HSG_ENTER(ctx);
  if (!ctx->diag_on) HSG_FAIL(ctx, HSG_ESTATE, "hsg_pt_diag_get before hsg_pt_diag_reset");
  const size_t nb = sizeof(long long) * ctx->g.R;
  if (moved_dev) HSG_CUDA(ctx, cudaMemcpyAsync(moved_dev, ctx->diag_moved, nb, cudaMemcpyDeviceToDevice, ctx->stream));
  if (traversals_dev) HSG_CUDA(ctx, cudaMemcpyAsync(traversals_dev, ctx->diag_trav, nb, cudaMemcpyDeviceToDevice, ctx->stream));
  if (p_diff_dev) {
    pt_diag_pdiff_kernel<<<blocks_for(ctx->g.T), kThreads, 0, ctx->stream>>>(ctx->g, ctx->diag_passes, ctx->diag_moved, p_diff_dev);
    HSG_LAUNCHED(ctx);
  }
  if (n_pass_host) *n_pass_host = ctx->diag_passes;
  return HSG_OK;
}

// ------------------------------------------------------------------ arithmetic self-test
int hsg_selftest_arith(void* cuda_stream, uint64_t seed, uint64_t n, unsigned long long* counts_dev) {
  if (!counts_dev) return HSG_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (cudaMemsetAsync(counts_dev, 0, 3 * sizeof(unsigned long long), st) != cudaSuccess) return HSG_ECUDA;
  PhiloxKey key{(uint32_t)seed, (uint32_t)(seed >> 32)};
  selftest_arith_kernel<<<148 * 8, kThreads, 0, st>>>(key, n, counts_dev);
  return cudaGetLastError() == cudaSuccess ? HSG_OK : HSG_ECUDA;
}

// ------------------------------------------------------------------ checkpoint
int hsg_get_state(hsg_ctx* ctx, int32_t* slot_of_temp_dev, uint64_t counters_host[2]) {
  HSG_ENTER(ctx);
  if (slot_of_temp_dev)
    HSG_CUDA(ctx, cudaMemcpyAsync(slot_of_temp_dev, ctx->slot_of_temp, sizeof(int32_t) * ctx->g.R, cudaMemcpyDeviceToDevice, ctx->stream));
  if (counters_host) { counters_host[0] = ctx->k_hb; counters_host[1] = ctx->k_pt; }
  return HSG_OK;
}

int hsg_set_state(hsg_ctx* ctx, const int32_t* slot_of_temp_dev, const uint64_t counters_host[2]) {
  HSG_ENTER(ctx);
  if (slot_of_temp_dev) {
    // NOTE: the caller must pass a valid permutation per (sample, replica); spins stay in their slots.
    set_perm_kernel<<<blocks_for(ctx->g.R), kThreads, 0, ctx->stream>>>(ctx->g, slot_of_temp_dev, ctx->slot_of_temp, ctx->temp_of_slot);
    HSG_LAUNCHED(ctx);
  }
  if (counters_host) { ctx->k_hb = counters_host[0]; ctx->k_pt = counters_host[1]; }
  return HSG_OK;
}

}  // extern "C"
