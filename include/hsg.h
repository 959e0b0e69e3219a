/* hsg.h — C ABI of the B200 Heisenberg-spin-glass Monte Carlo engine.
 *
 * One data-parallel hot path of Yavors'kii & Weigel, "Optimized GPU simulation of continuous-spin
 * glass models" (arXiv 1204.6192; citations are /root/reference/PAPER.md line numbers): Monte Carlo
 * sweeps of the 3D Edwards-Anderson Heisenberg spin glass in a random field,
 *
 *     H = - sum_<ij> J_ij s_i.s_j - sum_i H_i.s_i            (Eq. 1; each bond once)
 *
 * for D disorder samples x O replicas x T temperatures at once, with checkerboard
 * over-relaxation (Eq. 3) and heat-bath (Eq. 2) sweeps, parallel-tempering swaps (Eq. 4) and the
 * E / m / q^{mu nu}(k) reductions (Eqs. 5, 6).  DESIGN.md §3 fixes every arithmetic detail.
 *
 * Conventions
 *   - Every pointer named *_dev is DEVICE memory owned by the caller (e.g. a torch tensor); pointers
 *     named *_host are host memory.  The library never allocates or frees device memory: the caller
 *     provides `dev_state` / `dev_scratch` of the sizes hsg_query_bytes() returns and keeps them alive
 *     until hsg_destroy().  The layout inside them is private.
 *   - Every call only ENQUEUES work on the CUDA stream given to hsg_create() (a cudaStream_t passed
 *     as void*; NULL = the legacy default stream) and returns without synchronising; outputs are valid
 *     once the caller has synchronised that stream.  The device current at hsg_create() must be
 *     current at every later call (checked: HSG_ESTATE otherwise); contexts on different devices of one
 *     process are independent.
 *   - Site index i = x + L*(y + L*z), x fastest.  N = L^3.
 *     J_dev[d][dir][i]: coupling of the bond from site i to site i+e_dir (dir 0,1,2 = x,y,z), periodic.
 *     H_dev[d][c][i]  : component c of the field at site i.
 *     S_dev[d][o][t][c][i]: component c of spin i of (sample d, replica o, TEMPERATURE index t).
 *     All user-visible arrays are indexed by temperature index (0 = lowest T), never by the internal
 *     memory slot a configuration sits in.
 *   - P = O(O-1)/2 replica pairs in the order (0,1),(0,2),...,(1,2),...
 *   - Return value: HSG_OK (0) or a negative error code; no exceptions, no exit().  Text of the last
 *     error: hsg_last_error().  A context is not thread-safe; distinct contexts are independent.
 *   - Determinism: the same descriptor, disorder, start spins and call sequence give bit-identical
 *     results on every run, whatever kernel variant or grid is used (checkerboard independence,
 *     PAPER.md:119, plus the counter-based random stream of DESIGN.md §3.5).
 */
#ifndef HSG_H_
#define HSG_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
  HSG_OK = 0,
  HSG_EINVAL = -1,       /* null pointer, odd or too small L, non-ascending temperatures, size mismatch */
  HSG_ESTATE = -2,       /* e.g. sweep before disorder or spins were set */
  HSG_EUNSUPPORTED = -3, /* lattice size / option not supported by the selected kernel */
  HSG_ECUDA = -4         /* CUDA launch or runtime error; see hsg_last_error() */
};

/* kernel selection for hsg_sweep (hsg_set_option(HSG_OPT_SWEEP_KERNEL, ...)) */
enum {
  HSG_KERNEL_AUTO = 0,     /* fastest kernel that supports L */
  HSG_KERNEL_GENERIC = 1,  /* one launch per colour, neighbours straight from global memory; any even L */
  HSG_KERNEL_ZMARCH = 2    /* one launch per hsg_sweep call: both colours of every sweep fused in a z-marching pass */
};
enum {
  HSG_OPT_SWEEP_KERNEL = 1,
  HSG_OPT_FUSE_ENERGY = 2  /* 1 (default): the z-marching kernel reduces E and m of every system in the final
                              sweep of each hsg_sweep call, so hsg_pt_swap / hsg_measure / hsg_energy right
                              after it need no extra pass over the spins; 0: always use the separate
                              reduction kernel.  Values agree to fp64 summation order (~1e-15 relative). */
};

/* hsg_desc.flags */
enum {
  HSG_FLAG_FAST_MATH = 1   /* VARIANT of the heat-bath update (Table 1 rows PAPER.md:211,215,218: "fast_math"): the
                              same draw — same uniforms, inverse CDF and frame — with the correctly rounded divisions, square
                              roots and fixed series of DESIGN.md §3.3-3.4 replaced by the special-function unit's approximations
                              (rsqrt, ex2, lg2, rcp, sqrt, sin, cos).  Over-relaxation, energies, swaps and measurements are
                              unchanged.  Runs are still deterministic, but NOT bit-identical to the reference arithmetic: one
                              heat-bath update from equal inputs differs per spin component by at most
                              sqrt(2e-6 (1 + 1/a)), a = beta |h| (median ~ 1e-6 (1 + 1/a)); DESIGN.md §3.9. */
};

typedef struct hsg_ctx hsg_ctx; /* opaque, host side */

typedef struct {
  int32_t L;             /* lattice edge, even, >= 2 */
  int32_t n_samples;     /* D >= 1 disorder samples held by this context */
  int32_t n_replicas;    /* O >= 1 (overlaps need >= 2) */
  int32_t n_temps;       /* T >= 1 */
  const float* temps_host; /* T temperatures, strictly ascending, > 0; copied at create.
                              beta_t = (float)(1.0/(double)temps[t]) */
  uint64_t seed;         /* Philox key */
  uint64_t sample_offset;/* global id of local sample 0: random streams are keyed by the global id
                            sample_offset+d, so a job sharded by sample over several GPUs
                            reproduces the single-GPU run */
  uint32_t flags;        /* HSG_FLAG_* bits; 0 = the reference arithmetic of DESIGN.md §3 */
} hsg_desc;
/* Limits checked by hsg_query_bytes / hsg_create (HSG_EINVAL otherwise): L^3 < 2^31 (the site index is a 32-bit word
 * of the random-stream counter) and (sample_offset + D) * O * T < 2^32 (so is the global system id). */

/* Sizes of the two caller-owned device buffers for this descriptor. */
int hsg_query_bytes(const hsg_desc* desc, size_t* state_bytes, size_t* scratch_bytes);

/* Create a context over caller-owned device buffers (256-byte aligned).  Enqueues initialisation of the
 * permutation (configuration t holds temperature t) on `cuda_stream`. */
int hsg_create(const hsg_desc* desc, void* dev_state, size_t state_bytes, void* dev_scratch,
               size_t scratch_bytes, void* cuda_stream, hsg_ctx** out);

/* Frees the host-side context only. */
int hsg_destroy(hsg_ctx* ctx);

/* Quenched disorder.  J_dev [D][3][N]; H_dev [D][3][N] or NULL for zero field.  The
 * arrays are re-packed into the private layout; the caller may free them after synchronising. */
int hsg_set_disorder(hsg_ctx* ctx, const float* J_dev, const float* H_dev);

/* Start configuration: uniform on the sphere from the INIT domain of the random stream
 * (DESIGN.md §3.5), for the temperature index each configuration currently holds. */
int hsg_init_spins(hsg_ctx* ctx);

/* Copy spins in / out, S_dev [D][O][T][3][N] fp32 by temperature index. */
int hsg_set_spins(hsg_ctx* ctx, const float* S_dev);
int hsg_get_spins(hsg_ctx* ctx, float* S_dev);

/* n_or over-relaxation sweeps, THEN n_hb heat-bath sweeps of every system.
 * One sweep = all even sites ((x+y+z)%2 == 0), then all odd sites.
 * OR:  s' = 2 (s.h)/(h.h) h - s,  h = H_i + sum_j J_ij s_j                  (Eq. 3)
 * HB:  s' ~ exp(beta h.s) from two uniforms of the Philox stream keyed by
 *      (seed, sample, replica, temperature index, site, heat-bath sweep counter) (Eq. 2)
 * The heat-bath sweep counter advances by one per HB sweep. */
int hsg_sweep(hsg_ctx* ctx, int n_or, int n_hb);

/* Total energy (Eq. 1, every nearest-neighbour bond once) of every system, E_dev [D][O][T] by temperature
 * index.  Precision as PAPER.md:185: the site terms s_i.h_i (odd sites, h_i the local field of PAPER.md:37) and s_i.H_i
 * (even sites) in single precision, their sum over the lattice in double. */
int hsg_energy(hsg_ctx* ctx, double* E_dev);

/* One parallel-tempering pass (Eq. 4): for each (sample, replica), pairs (t, t+1) for
 * t = 0..T-2 in this order, swap accepted with probability min[1, exp(dbeta*dE)],
 * dE = E_{t+1}-E_t, dbeta = beta_{t+1}-beta_t in fp64, energies as hsg_energy recomputed from the spins.
 * accepted_dev [D][O][T-1] int32 (1 = swapped) or NULL.  The PT counter advances by one per call. */
int hsg_pt_swap(hsg_ctx* ctx, int32_t* accepted_dev);

/* Measurements, all fp64, any pointer may be NULL:
 *   E_dev  [D][O][T]            total energy
 *   M_dev  [D][O][T][3]         m = (1/N) sum_i s_i
 *   q0_dev [D][P][T][3][3]      q^{mu nu}(0)      = (1/N) sum_i s_i^{mu(a)} s_i^{nu(b)}         (Eq. 5)
 *   qk_dev [D][P][T][3][3][2]   q^{mu nu}(k_min)  = (1/N) sum_i s_i^{mu(a)} s_i^{nu(b)} e^{+i k x_i},
 *                               k_min = (2 pi/L)(1,0,0), last index (re, im)        (Eq. 6)
 * for replica pairs a<b holding the same temperature. */
int hsg_measure(hsg_ctx* ctx, double* E_dev, double* M_dev, double* q0_dev, double* qk_dev);

/* Checkpoint: slot_of_temp_dev [D][O][T] int32 = configuration slot (0..T-1 within its (d,o) group, in
 * hsg_init order) that holds temperature t; counters_host = {heat-bath sweep counter, PT counter}.
 * hsg_get_state synchronises nothing: slot_of_temp_dev is written on the stream.
 * Restore order: hsg_set_state(permutation) FIRST, then hsg_set_spins — spins arrive by temperature index and are
 * stored in the slot the permutation in force at that moment assigns; a later hsg_set_state re-labels the
 * configurations without moving them. */
int hsg_get_state(hsg_ctx* ctx, int32_t* slot_of_temp_dev, uint64_t counters_host[2]);
int hsg_set_state(hsg_ctx* ctx, const int32_t* slot_of_temp_dev, const uint64_t counters_host[2]);

/* Field-case observables (Eqs. 9-11): the susceptibility summands of Eq. (10) from four real replicas
 * (1),(2),(3),(4) = replicas 0,1,2,3 of every sample, all at temperature index t, for k = 0 and
 * k_min = (2 pi/L)(1,0,0):
 *   chi_1(k) = sum_{i,j} sum_{mu,nu} s_i^{mu(1)} s_j^{nu(1)} s_i^{mu(2)} s_j^{nu(2)} e^{ik.(R_i-R_j)}
 *   chi_2(k) = ...                   s_i^{mu(1)} s_j^{nu(1)} s_i^{mu(3)} s_j^{nu(4)} ...
 *   chi_3(k) = ...                   s_i^{mu(1)} s_j^{nu(2)} s_i^{mu(3)} s_j^{nu(4)} ...
 * chi_dev [D][T][2 (k = 0, k_min)][3 (chi_1, chi_2, chi_3)][2 (re, im)] fp64.  The thermal average of Eq. (10) is the
 * caller's mean over measurements; Eq. (11): chi_SG(k) = (1/N) [chi_1 - 2 chi_2 + chi_3]_J.  Needs O >= 4
 * (HSG_EUNSUPPORTED otherwise).  Evaluated as products of A_ab(k) = sum_i (s_i^(a).s_i^(b)) e^{ik x_i}. */
int hsg_measure_field(hsg_ctx* ctx, double* chi_dev);

/* Chiral sector: local chirality kappa_i^alpha = s_{i+alpha} . (s_i x s_{i-alpha}) (Eq. 12, alpha = x,y,z,
 * periodic; formed in single precision in the operation order of DESIGN.md §3.8) and the chiral overlaps (Eq. 13)
 *   qc0_dev [D][P][T][3]     q_c^alpha(0)     = (1/N) sum_i kappa_i^{alpha(a)} kappa_i^{alpha(b)}
 *   qck_dev [D][P][T][3][2]  q_c^alpha(k_min) = (1/N) sum_i kappa_i^{alpha(a)} kappa_i^{alpha(b)} e^{+i k x_i}   (re, im)
 * for replica pairs a<b at the same temperature (fp64 products and sums); either pointer may be NULL.
 * chi_CG^alpha(k) = N <|q_c^alpha(k)|^2> (Eq. 14) and xi_c (Eq. 15, hsg_xi_second_moment) are the caller's averages. */
int hsg_measure_chiral(hsg_ctx* ctx, double* qc0_dev, double* qck_dev);

/* Second-moment correlation length, Eq. (8) (and Eq. 15): xi = sqrt(chi(0)/chi(k_min) - 1) / (2 sin(k_min/2)),
 * |k_min| = 2 pi/L.  Host arithmetic on host values; HSG_EINVAL if chi_kmin <= 0 or the ratio is below 1. */
int hsg_xi_second_moment(double chi_0, double chi_kmin, int32_t L, double* xi_host);

/* Parallel-tempering diagnostics (PAPER.md:197 and Fig. 3), accumulated on the device by hsg_pt_swap once
 * hsg_pt_diag_reset() has been called (which zeroes them and marks the configurations that start at an end point):
 *   moved_dev      [D][O][T] int64, by temperature index: passes after which the copy that held T_t had left it
 *   traversals_dev [D][O][T] int64, by configuration slot: arrivals at one end point of the ladder after the last touch
 *                  of the other one; N_tunn ("a replica travels a closed loop between T_1 and T_{R_T}") = traversals / 2
 *   p_diff_dev     [T] fp64: moved summed over (d,o) / (D O n_pass) — the quantity of Fig. 3
 *   n_pass_host    passes counted since the reset.  Any pointer may be NULL. */
int hsg_pt_diag_reset(hsg_ctx* ctx);
int hsg_pt_diag_get(hsg_ctx* ctx, int64_t* moved_dev, int64_t* traversals_dev, double* p_diff_dev, uint64_t* n_pass_host);

/* Tuning / test hooks (HSG_OPT_*).  Results never depend on them. */
int hsg_set_option(hsg_ctx* ctx, int option, int value);

/* Number of kernel launches enqueued by this context so far (for bench.py's gpu_launches). */
uint64_t hsg_launch_count(const hsg_ctx* ctx);

/* Name of the sweep kernel the last hsg_sweep used ("generic", "zmarch"; "none" before the first sweep). */
const char* hsg_last_sweep_kernel(const hsg_ctx* ctx);

/* Test hook: compares the kernels' branch-free IEEE division / square root with the
 * compiler's correctly rounded ones on n pseudo-random operand sets; counts_dev[0] = division mismatches,
 * counts_dev[1] = square-root mismatches, counts_dev[2] = division mismatches on divisors whose mantissa is all ones (the
 * one exceptional case of the Newton scheme, counted apart) (device memory, 3 x uint64, zeroed by the call). */
int hsg_selftest_arith(void* cuda_stream, uint64_t seed, uint64_t n, unsigned long long* counts_dev);

const char* hsg_last_error(const hsg_ctx* ctx);
const char* hsg_version(void);

#ifdef __cplusplus
}
#endif
#endif /* HSG_H_ */
