// hsg_oracle.cpp — ORACLE. TEST INFRASTRUCTURE ONLY, NOT PART OF THE PRODUCT PATH.
//
// Plain, slow, serial (per system) CPU implementation of the hot path of
// Yavors'kii & Weigel, "Optimized GPU simulation of continuous-spin glass models"
// (arXiv 1204.6192): Monte Carlo sweeps (over-relaxation + heat bath), parallel
// tempering and the E / M / overlap measurements of the 3D Edwards-Anderson
// Heisenberg spin glass in a random field.  Written from PAPER.md and the readings
// listed in DESIGN.md §3; it shares no code with the CUDA path (paper_1204_6192_b200/).
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may build, load or call this file.
//
// Two instantiations of one template:
//   Real = double : the physics truth used by the closed-form pins.
//   Real = float  : the trajectory reference for the GPU.  PAPER.md:185 fixes the
//                   precision ("spins being represented in single precision and
//                   aggregate quantities ... in double precision"), and a chaotic
//                   fp32 trajectory can only be compared with an fp32 trajectory
//                   (DESIGN.md §3 "numeric contract").  In this instantiation every
//                   floating-point operation is an individually rounded IEEE-754
//                   binary32 operation in the order DESIGN.md §3 states (explicit
//                   fused multiply-adds, correctly rounded division and square
//                   root), and exp/log/sin/cos are the fixed series of DESIGN.md §3.4.
//                   Compile with -ffp-contract=off so the compiler adds no fusion
//                   of its own (cf. PAPER.md:220 on FMA contraction).
//
// Pins: tests/test_oracle_*.py (-m "not gpu") — Langevin law, OR invariants, beta=0,
// two-/four-spin clusters against quadrature, PT in a uniform field, overlap
// identities, brute force on L=4, Philox against an independent numpy restatement
// and published known-answer vectors.  No function here is "parity unpinned".
//
// Layouts (all C-order):
//   site index  i = x + L*(y + L*z), x fastest
//   J[d][dir][i]  coupling of the bond from site i to i+e_dir (dir 0,1,2 = x,y,z), periodic
//   H[d][c][i]    field component c at site i
//   S[d][o][t][c][i] spins, t = TEMPERATURE index (0 = lowest T), c = component
//   system id (Philox) = ((sample_offset+d)*O + o)*T + t
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <thread>
#include <algorithm>
#include <type_traits>

namespace {

// --------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), DESIGN.md §3.5.  Replaces the
// paper's multiply-with-carry generator (which the authors planned to
// replace).  Counter-based: out = philox(counter[4], key[2]).
// --------------------------------------------------------------------------------------
inline void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;   // multipliers
  const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;   // Weyl key increments
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    if (round > 0) { k0 += W0; k1 += W1; }
    const uint64_t p0 = (uint64_t)M0 * c0;
    const uint64_t p1 = (uint64_t)M1 * c2;
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    const uint32_t n0 = hi1 ^ c1 ^ k0;
    const uint32_t n1 = lo1;
    const uint32_t n2 = hi0 ^ c3 ^ k1;
    const uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

enum : uint32_t { DOMAIN_INIT = 0, DOMAIN_HB = 1, DOMAIN_PT = 2 };

// counter packing, DESIGN.md §3.5
inline void make_counter(uint32_t c0, uint64_t k, uint32_t c2, uint32_t domain, uint32_t ctr[4]) {
  ctr[0] = c0;
  ctr[1] = (uint32_t)(k & 0xFFFFFFFFull);
  ctr[2] = c2;
  ctr[3] = ((uint32_t)(k >> 32) & 0x0FFFFFFFu) | (domain << 28);
}

// 23-bit midpoint uniform in (0,1): u = ((w >> 9) + 1/2) * 2^-23.  Exactly representable
// in binary32 and binary64, never 0 or 1.  DESIGN.md §3.5 ("two random
// numbers distributed uniformly between 0 and 1").
template <class Real> inline Real u01(uint32_t w) {
  return (Real)(w >> 9) * (Real)(1.0 / 8388608.0) + (Real)(1.0 / 16777216.0);   // exact in both types
}

// --------------------------------------------------------------------------------------
// Elementary arithmetic.  For Real=float every call is one IEEE-754 binary32 rounding.
// --------------------------------------------------------------------------------------
inline float  fma_(float a, float b, float c)    { return __builtin_fmaf(a, b, c); }
inline double fma_(double a, double b, double c) { return __builtin_fma(a, b, c); }
inline float  sqrt_(float a)  { return __builtin_sqrtf(a); }
inline double sqrt_(double a) { return __builtin_sqrt(a); }

// --------------------------------------------------------------------------------------
// the three transcendental steps of the heat-bath draw.
//   omexp(x)  = 1 - exp(-x),      x >= 0
//   log1m(y)  = ln(1 - y),        0 < y < 1
//   sincos2pi(u) = (sin 2*pi*u, cos 2*pi*u), 0 < u < 1
// double: the C library.  float: fixed Taylor / atanh series of binary32 operations
// (so that an independent implementation can reproduce every bit).
// --------------------------------------------------------------------------------------
inline double omexp(double x) { return -std::expm1(-x); }
inline double log1m(double y) { return std::log1p(-y); }
inline void sincos2pi(double u, double& s, double& c) {
  const double two_pi = 6.283185307179586476925286766559;
  s = std::sin(two_pi * u); c = std::cos(two_pi * u);
}

inline float uint_as_float(uint32_t u) { float f; std::memcpy(&f, &u, 4); return f; }
inline uint32_t float_as_uint(float f) { uint32_t u; std::memcpy(&u, &f, 4); return u; }

inline float omexp(float x) {
  // exp(-x) = 2^-k * exp(-r),  k = rint(x*log2(e)),  r = x - k*ln2 (two-term Cody-Waite).
  // expm1(s), s=-r, |s| <= ln2/2: Taylor s + s^2/2! + ... + s^8/8!  (truncation < 6e-10 relative).
  const float xc = x < 80.0f ? x : 80.0f;                  // 2^-k stays a normal number
  const float kf = __builtin_rintf(xc * 1.44269504088896341f);
  float r = fma_(-kf, 0.693145751953125f, xc);             // ln2_hi (exact in 16 bits)
  r = fma_(-kf, 1.42860682030941723e-6f, r);               // ln2_lo
  const float s = -r;
  float p = 1.0f / 40320.0f;
  p = fma_(p, s, 1.0f / 5040.0f);
  p = fma_(p, s, 1.0f / 720.0f);
  p = fma_(p, s, 1.0f / 120.0f);
  p = fma_(p, s, 1.0f / 24.0f);
  p = fma_(p, s, 1.0f / 6.0f);
  p = fma_(p, s, 0.5f);
  p = p * s;
  p = fma_(p, s, s);                                       // p = expm1(s)
  const int k = (int)kf;
  const float c = uint_as_float((uint32_t)(127 - k) << 23);  // 2^-k exactly
  return fma_(-c, p, 1.0f - c);                            // (1 - 2^-k) - 2^-k * expm1(s)
}

inline float log1m(float y) {
  // ln(1-y) = e*ln2 + ln(1+f):  y < 1/4: f = -y, e = 0;  else 1-y = m*2^e with m in [2/3,4/3), f = m-1.
  // ln(1+f) = 2 atanh(s), s = f/(2+f): 2s(1 + s^2/3 + s^4/5 + s^6/7 + s^8/9), |s| <= 1/5.
  float f, ef;
  if (y < 0.25f) { f = -y; ef = 0.0f; }
  else {
    const float u = 1.0f - y;
    const uint32_t bits = float_as_uint(u);
    const int32_t e = (int32_t)(bits - 0x3f2aaaabu) >> 23;       // floor(log2(u / (2/3)))
    const float m = uint_as_float(bits - ((uint32_t)e << 23));
    f = m - 1.0f; ef = (float)e;
  }
  const float s = f / (2.0f + f);
  const float z = s * s;
  float p = 1.0f / 9.0f;
  p = fma_(p, z, 1.0f / 7.0f);
  p = fma_(p, z, 1.0f / 5.0f);
  p = fma_(p, z, 1.0f / 3.0f);
  p = p * z;
  p = fma_(p, s, s);                                       // atanh(s)
  return fma_(ef, 0.693147180559945309f, p + p);
}

inline void sincos2pi(float u, float& sn, float& cs) {
  // q = rint(4u) in {0..4}, r = u - q/4 (exact), |r| <= 1/8; Taylor series of sin/cos(2*pi*r) in r.
  const float qf = __builtin_rintf(4.0f * u);
  const float r = fma_(-0.25f, qf, u);
  const float z = r * r;
  // sin(2 pi r) = r*(S1 + S3 z + S5 z^2 + S7 z^3 + S9 z^4),  S_k = (-1)^((k-1)/2) (2 pi)^k / k!
  float ps = 42.0586939448225f;              //  (2pi)^9/9!
  ps = fma_(ps, z, -76.7058597530614f);      // -(2pi)^7/7!
  ps = fma_(ps, z, 81.6052492760750f);       //  (2pi)^5/5!
  ps = fma_(ps, z, -41.3417022403998f);      // -(2pi)^3/3!
  ps = fma_(ps, z, 6.28318530717959f);       //  2pi
  const float s0 = ps * r;
  // cos(2 pi r) = 1 + z*(C2 + C4 z + C6 z^2 + C8 z^3 + C10 z^4),  C_k = (-1)^(k/2) (2 pi)^k / k!
  float pc = -26.4262567832749f;             // -(2pi)^10/10!
  pc = fma_(pc, z, 60.2446413718766f);       //  (2pi)^8/8!
  pc = fma_(pc, z, -85.4568172066937f);      // -(2pi)^6/6!
  pc = fma_(pc, z, 64.9393940226683f);       //  (2pi)^4/4!
  pc = fma_(pc, z, -19.7392088021787f);      // -(2pi)^2/2!
  const float c0 = fma_(pc, z, 1.0f);
  const int q = (int)qf & 3;
  if (q == 0)      { sn =  s0; cs =  c0; }
  else if (q == 1) { sn =  c0; cs = -s0; }
  else if (q == 2) { sn = -s0; cs = -c0; }
  else             { sn = -c0; cs =  s0; }
}

// --------------------------------------------------------------------------------------
// Single-spin moves.
// --------------------------------------------------------------------------------------

// Over-relaxation, Eq. (3):  s' = 2 (s.h)/(h.h) h - s.   DESIGN.md §3.2.
template <class Real>
inline void or_reflect(const Real s[3], const Real h[3], Real out[3]) {
  const Real sh = fma_(s[2], h[2], fma_(s[1], h[1], s[0] * h[0]));
  const Real hh = fma_(h[2], h[2], fma_(h[1], h[1], h[0] * h[0]));
  if (!(hh >= (Real)1e-30)) { out[0] = s[0]; out[1] = s[1]; out[2] = s[2]; return; }   // zero field: identity
  const Real f = (sh + sh) / hh;
  out[0] = fma_(f, h[0], -s[0]);
  out[1] = fma_(f, h[1], -s[1]);
  out[2] = fma_(f, h[2], -s[2]);
}

// Heat bath, Eq. (2): s' ~ exp(beta h.s), drawn from two uniforms.
// cos(theta) by inversion of the CDF (e^{a c} - e^{-a})/(e^{a} - e^{-a}), a = beta|h|:
//   t = 1 - cos(theta) = -ln(1 - (1-u1)(1 - e^{-2a})) / a ;
// azimuth phi = 2 pi u2 in the orthonormal frame (e1, e2, n) of DESIGN.md §3.3.
template <class Real>
inline void hb_draw(const Real h[3], Real beta, Real u1, Real u2, Real out[3]) {
  const Real hh = fma_(h[2], h[2], fma_(h[1], h[1], h[0] * h[0]));
  Real a, n[3];
  if (!(hh >= (Real)1e-30)) { a = 0; n[0] = 0; n[1] = 0; n[2] = 1; }
  else {
    const Real hn = sqrt_(hh);
    const Real inv = (Real)1 / hn;
    n[0] = h[0] * inv; n[1] = h[1] * inv; n[2] = h[2] * inv;
    a = beta * hn;
  }
  const Real v = (Real)1 - u1;                       // exact
  Real t;
  if (a < (Real)1e-4) {
    const Real t0 = v + v;                           // t = 2v(1 - a u1) + O(a^2)
    t = fma_(-(a * u1), t0, t0);
  } else {
    const Real E = omexp(a + a);
    const Real y = v * E;
    t = -log1m(y) / a;
  }
  t = t < (Real)0 ? (Real)0 : (t > (Real)2 ? (Real)2 : t);
  const Real ct = (Real)1 - t;
  const Real st = sqrt_(t * ((Real)2 - t));
  Real sp, cp;
  sincos2pi(u2, sp, cp);
  // frame: sigma = sign(n_z) (+1 at 0), A = -1/(sigma + n_z)
  const Real sg = n[2] >= (Real)0 ? (Real)1 : (Real)-1;
  const Real A = (Real)-1 / (sg + n[2]);
  const Real xa = n[0] * A, ya = n[1] * A;
  const Real B = n[1] * xa;
  const Real e1[3] = { fma_(sg * n[0], xa, (Real)1), sg * B, -(sg * n[0]) };
  const Real e2[3] = { B, fma_(n[1], ya, sg), -n[1] };
  const Real p = st * cp, q = st * sp;
  for (int c = 0; c < 3; ++c) out[c] = fma_(q, e2[c], fma_(p, e1[c], ct * n[c]));
}

// --------------------------------------------------------------------------------------
// The simulation.
// --------------------------------------------------------------------------------------
template <class Real>
struct Sim {
  int L, D, O, T; long N;
  uint64_t seed, sample_offset;
  uint64_t k_hb = 0, k_pt = 0;
  std::vector<float> temps;            // [T] ascending
  std::vector<float> beta;             // [T] beta_t = (float)(1.0/(double)temps[t])
  std::vector<float> J, H;             // [D][3][N]
  // configurations are stored by SLOT (memory position); conf_of_temp[(d*O+o)*T + t] = slot
  // (0..T-1 inside the (d,o) group) whose configuration currently holds temperature t.
  std::vector<Real> S;                 // [D][O][slot][3][N]
  std::vector<int32_t> conf_of_temp;   // [D][O][T]
  bool have_disorder = false, have_spins = false;
  // parallel-tempering diagnostics of PAPER.md:197 / Fig. 3, see pt_diag_reset()
  bool diag_on = false;
  uint64_t diag_passes = 0;
  std::vector<int64_t> diag_moved;     // [D][O][T] by TEMPERATURE index: passes after which the copy that held T_t had left it
  std::vector<int64_t> diag_trav;      // [D][O][slot] end-to-end traversals T_1 <-> T_{R_T} of every configuration
  std::vector<int8_t> diag_last;       // [D][O][slot] end point touched last: +1 = T_1, -1 = T_{R_T}, 0 = none yet

  Sim(int L_, int D_, int O_, int T_, const float* temps_, uint64_t seed_, uint64_t off)
      : L(L_), D(D_), O(O_), T(T_), N((long)L_ * L_ * L_), seed(seed_), sample_offset(off),
        temps(temps_, temps_ + T_), beta(T_), J((size_t)D_ * 3 * N, 0.f), H((size_t)D_ * 3 * N, 0.f),
        S((size_t)D_ * O_ * T_ * 3 * N, (Real)0), conf_of_temp((size_t)D_ * O_ * T_) {
    for (int t = 0; t < T; ++t) beta[t] = (float)(1.0 / (double)temps[t]);
    for (int g = 0; g < D * O; ++g) for (int t = 0; t < T; ++t) conf_of_temp[(size_t)g * T + t] = t;
  }
  Real* spins_of_slot(int d, int o, int slot) { return &S[(((size_t)d * O + o) * T + slot) * 3 * N]; }
  Real* spins_of_temp(int d, int o, int t) { return spins_of_slot(d, o, conf_of_temp[((size_t)d * O + o) * T + t]); }
  uint32_t system_id(int d, int o, int t) const { return (uint32_t)(((sample_offset + (uint64_t)d) * O + o) * T + t); }
  void key(uint32_t k[2]) const { k[0] = (uint32_t)seed; k[1] = (uint32_t)(seed >> 32); }

  long nbr(long i, int dir, int sign) const {   // periodic neighbour of site i
    const int x = (int)(i % L), y = (int)((i / L) % L), z = (int)(i / ((long)L * L));
    int c[3] = {x, y, z};
    c[dir] = (c[dir] + sign + L) % L;
    return c[0] + (long)L * (c[1] + (long)L * c[2]);
  }

  // local field: h = H_i + sum_j J_ij s_j ; fixed order x+,x-,y+,y-,z+,z- 
  void local_field(const Real* s, const float* Jd, const float* Hd, long i, Real h[3]) const {
    for (int c = 0; c < 3; ++c) h[c] = (Real)Hd[(size_t)c * N + i];
    for (int dir = 0; dir < 3; ++dir) {
      const long ip = nbr(i, dir, +1), im = nbr(i, dir, -1);
      const Real Jp = (Real)Jd[(size_t)dir * N + i];     // bond i -> i+e_dir
      const Real Jm = (Real)Jd[(size_t)dir * N + im];    // bond (i-e_dir) -> i
      for (int c = 0; c < 3; ++c) h[c] = fma_(Jp, s[(size_t)c * N + ip], h[c]);
      for (int c = 0; c < 3; ++c) h[c] = fma_(Jm, s[(size_t)c * N + im], h[c]);
    }
  }

  // uniform spins on S^2 from the INIT domain: cos(theta) = 2u1-1, phi = 2 pi u2 about z.
  void init_spins() {
    uint32_t k[2]; key(k);
    for (int d = 0; d < D; ++d) for (int o = 0; o < O; ++o) for (int t = 0; t < T; ++t) {
      Real* s = spins_of_temp(d, o, t);
      for (long i = 0; i < N; ++i) {
        uint32_t ctr[4], w[4];
        make_counter((uint32_t)i, 0, system_id(d, o, t), DOMAIN_INIT, ctr);
        philox4x32_10(ctr, k, w);
        const Real u1 = u01<Real>(w[0]), u2 = u01<Real>(w[1]);
        const Real ct = fma_((Real)2, u1, (Real)-1);
        const Real st = sqrt_(fma_(-ct, ct, (Real)1));
        Real sp, cp; sincos2pi(u2, sp, cp);
        s[i] = st * cp; s[N + i] = st * sp; s[2 * N + i] = ct;
      }
    }
    have_spins = true;
  }

  // one full sweep of one configuration: colour 0 = even sites ((x+y+z)%2==0), then colour 1
  // (reading 9: global two-colour sweeps).
  void sweep_system(int d, int o, int t, bool heat_bath) {
    Real* s = spins_of_temp(d, o, t);
    const float* Jd = &J[(size_t)d * 3 * N];
    const float* Hd = &H[(size_t)d * 3 * N];
    const Real b = (Real)beta[t];
    const uint32_t sid = system_id(d, o, t);
    uint32_t k[2]; key(k);
    for (int colour = 0; colour < 2; ++colour)
      for (int z = 0; z < L; ++z) for (int y = 0; y < L; ++y) for (int x = 0; x < L; ++x) {
        if (((x + y + z) & 1) != colour) continue;
        const long i = x + (long)L * (y + (long)L * z);
        Real h[3], cur[3] = { s[i], s[N + i], s[2 * N + i] }, out[3];
        local_field(s, Jd, Hd, i, h);
        if (heat_bath) {
          // one Philox call serves the two same-colour sites x and x+2 whose compact index
          // j = x>>1 is (even, odd): counter word 0 = the site with even j; that site takes output words 0, 1,
          // its partner words 2, 3.
          const int odd = (x >> 1) & 1;
          uint32_t ctr[4], w[4];
          make_counter((uint32_t)(i - 2 * odd), k_hb, sid, DOMAIN_HB, ctr);
          philox4x32_10(ctr, k, w);
          hb_draw<Real>(h, b, u01<Real>(w[2 * odd]), u01<Real>(w[2 * odd + 1]), out);
        } else {
          or_reflect<Real>(cur, h, out);
        }
        s[i] = out[0]; s[N + i] = out[1]; s[2 * N + i] = out[2];
      }
  }

  // hsg_sweep(n_or, n_hb): n_or OR sweeps, THEN n_hb HB sweeps (reading 8).
  void sweep(int n_or, int n_hb, int n_threads) {
    const long R = (long)D * O * T;
    for (int sw = 0; sw < n_or + n_hb; ++sw) {
      const bool hb = sw >= n_or;
      auto work = [&](long r0, long r1) {
        for (long r = r0; r < r1; ++r) {
          const int t = (int)(r % T), o = (int)((r / T) % O), d = (int)(r / ((long)T * O));
          sweep_system(d, o, t, hb);
        }
      };
      if (n_threads <= 1) work(0, R);
      else {   // systems are independent; each system stays serial
        std::vector<std::thread> th;
        const int nt = (int)std::min<long>(n_threads, R);
        for (int k = 0; k < nt; ++k) th.emplace_back(work, R * k / nt, R * (k + 1) / nt);
        for (auto& x : th) x.join();
      }
      if (hb) ++k_hb;
    }
  }

  // PAPER.md:26 Eq. (1), each nearest-neighbour bond once (reading 1), in the bipartite form: every bond joins an
  // even and an odd site, so  E = - sum_{i odd} s_i . h_i  -  sum_{i even} s_i . H_i  with h_i = H_i + sum_j J_ij s_j
  // the local field of the moves.  Site terms in the spins' precision Real with the fixed FMA order of
  // the moves, the sum over sites in double ("spins ... single precision and aggregate quantities ...
  // double precision", reading 11).
  double energy_of(const Real* s, int d) const {
    const float* Jd = &J[(size_t)d * 3 * N];
    const float* Hd = &H[(size_t)d * 3 * N];
    double E = 0.0;
    for (int z = 0; z < L; ++z) for (int y = 0; y < L; ++y) for (int x = 0; x < L; ++x) {
      const long i = x + (long)L * (y + (long)L * z);
      Real h[3];
      if ((x + y + z) & 1) local_field(s, Jd, Hd, i, h);
      else for (int c = 0; c < 3; ++c) h[c] = (Real)Hd[(size_t)c * N + i];
      const Real e = fma_(s[2 * N + i], h[2], fma_(s[N + i], h[1], s[i] * h[0]));
      E -= (double)e;
    }
    return E;
  }
  void energy(double* E /*[D][O][T]*/) {
    for (int d = 0; d < D; ++d) for (int o = 0; o < O; ++o) for (int t = 0; t < T; ++t)
      E[((size_t)d * O + o) * T + t] = energy_of(spins_of_temp(d, o, t), d);
  }

  // PAPER.md:26 Eq. (1) exactly as written, the plain definition:  E = - sum_<ij> J_ij s_i.s_j - sum_i H_i.s_i ,
  // every nearest-neighbour bond once (the three forward bonds x+, y+, z+ of every site; reading 1), every product
  // and the whole sum in double from the stored spins, sites in index order.  No local field, no colours, no
  // single-precision intermediate: this is what energy_of() (the PAPER.md:185 reading the moves and the
  // parallel-tempering decisions use) is pinned against, and what the GPU energies are bounded against.
  double energy_plain_of(const Real* s, int d) const {
    const float* Jd = &J[(size_t)d * 3 * N];
    const float* Hd = &H[(size_t)d * 3 * N];
    double E = 0.0;
    for (long i = 0; i < N; ++i) {
      for (int dir = 0; dir < 3; ++dir) {
        const long ip = nbr(i, dir, +1);
        double dot = 0.0;
        for (int c = 0; c < 3; ++c) dot += (double)s[(size_t)c * N + i] * (double)s[(size_t)c * N + ip];
        E -= (double)Jd[(size_t)dir * N + i] * dot;
      }
      for (int c = 0; c < 3; ++c) E -= (double)Hd[(size_t)c * N + i] * (double)s[(size_t)c * N + i];
    }
    return E;
  }
  void energy_plain(double* E /*[D][O][T]*/) {
    for (int d = 0; d < D; ++d) for (int o = 0; o < O; ++o) for (int t = 0; t < T; ++t)
      E[((size_t)d * O + o) * T + t] = energy_plain_of(spins_of_temp(d, o, t), d);
  }

  // Parallel tempering, Eq. (4): pairs (t, t+1) from the lowest temperature upwards,
  // accept with min[1, exp(dbeta*dE)], dE = E_{t+1}-E_t, dbeta = beta_{t+1}-beta_t.  One chain per (d,o).
  void pt_swap(int32_t* accepted /*[D][O][T-1] or null*/) {
    std::vector<double> E((size_t)D * O * T);
    energy(E.data());
    const std::vector<int32_t> before = conf_of_temp;          // (diagnostics only)
    uint32_t k[2]; key(k);
    for (int d = 0; d < D; ++d) for (int o = 0; o < O; ++o) {
      double* Eg = &E[((size_t)d * O + o) * T];
      int32_t* cf = &conf_of_temp[((size_t)d * O + o) * T];
      for (int t = 0; t + 1 < T; ++t) {
        const double x = ((double)beta[t + 1] - (double)beta[t]) * (Eg[t + 1] - Eg[t]);
        uint32_t ctr[4], w[4];
        make_counter((uint32_t)t, k_pt, (uint32_t)((sample_offset + (uint64_t)d) * O + o), DOMAIN_PT, ctr);
        philox4x32_10(ctr, k, w);
        const double u = u01<double>(w[0]);
        const bool acc = (x >= 0.0) || (std::log(u) < x);
        if (acc) { std::swap(cf[t], cf[t + 1]); std::swap(Eg[t], Eg[t + 1]); }
        if (accepted) accepted[((size_t)d * O + o) * (T - 1) + t] = acc ? 1 : 0;
      }
    }
    ++k_pt;
    if (diag_on) pt_diag_update(before);
  }

  // ---- Parallel-tempering diagnostics (Fig. 3) ----
  // p_diff(T_t): "the probability that, after a parallel tempering update, a copy of the system at T_t will diffuse to
  // neighboring temperatures": per pass and (d,o), the copy (configuration slot) that held T_t before the pass holds
  // another temperature after it.  Tunnelling: "a replica travels a closed loop between the temperature end points T_1
  // and T_{R_T}": every arrival of a configuration at one end point after it last touched the OTHER one is one
  // traversal; a closed loop = two traversals (N_tunn = traversals / 2, integer division, per configuration).
  void pt_diag_touch() {
    for (int g = 0; g < D * O; ++g)
      for (int e = 0; e < 2; ++e) {
        const int t_end = e == 0 ? 0 : T - 1;
        const int8_t tag = e == 0 ? 1 : -1;
        const size_t s = (size_t)g * T + conf_of_temp[(size_t)g * T + t_end];
        if (diag_last[s] == -tag) ++diag_trav[s];
        diag_last[s] = tag;
      }
  }
  void pt_diag_reset() {
    diag_on = true; diag_passes = 0;
    diag_moved.assign((size_t)D * O * T, 0); diag_trav.assign((size_t)D * O * T, 0); diag_last.assign((size_t)D * O * T, 0);
    pt_diag_touch();                      // the configurations that START at an end point have touched it
  }
  void pt_diag_update(const std::vector<int32_t>& before) {
    for (size_t r = 0; r < before.size(); ++r) diag_moved[r] += (conf_of_temp[r] != before[r]) ? 1 : 0;
    ++diag_passes;
    pt_diag_touch();
  }
  void pt_diag_get(int64_t* moved, int64_t* trav, uint64_t* n_pass, double* p_diff /*[T]*/) const {
    if (moved) std::copy(diag_moved.begin(), diag_moved.end(), moved);
    if (trav) std::copy(diag_trav.begin(), diag_trav.end(), trav);
    if (n_pass) *n_pass = diag_passes;
    if (p_diff) for (int t = 0; t < T; ++t) {
      double acc = 0.0;
      for (int g = 0; g < D * O; ++g) acc += (double)diag_moved[(size_t)g * T + t];
      p_diff[t] = diag_passes ? acc / ((double)D * O * (double)diag_passes) : 0.0;
    }
  }

  // Measurements: E per system; m = (1/N) sum_i s_i; overlap tensor PAPER.md:53-58 Eqs. (5),(6)
  // q^{mu nu}(k) = (1/N) sum_i s_i^{mu(a)} s_i^{nu(b)} e^{+i k x_i} for replica pairs a<b at the same
  // temperature, k = 0 and k_min = (2 pi/L)(1,0,0).  All sums in double.
  void measure(double* E, double* M, double* q0, double* qk) {
    if (E) energy(E);
    if (M) for (int d = 0; d < D; ++d) for (int o = 0; o < O; ++o) for (int t = 0; t < T; ++t) {
      const Real* s = spins_of_temp(d, o, t);
      for (int c = 0; c < 3; ++c) {
        double acc = 0.0;
        for (long i = 0; i < N; ++i) acc += (double)s[(size_t)c * N + i];
        M[(((size_t)d * O + o) * T + t) * 3 + c] = acc / (double)N;
      }
    }
    if (!q0 && !qk) return;
    const int P = O * (O - 1) / 2;
    const double two_pi = 6.283185307179586476925286766559;
    for (int d = 0; d < D; ++d) {
      int p = 0;
      for (int a = 0; a < O; ++a) for (int b = a + 1; b < O; ++b, ++p) for (int t = 0; t < T; ++t) {
        const Real* sa = spins_of_temp(d, a, t);
        const Real* sb = spins_of_temp(d, b, t);
        for (int mu = 0; mu < 3; ++mu) for (int nu = 0; nu < 3; ++nu) {
          double r0 = 0.0, re = 0.0, im = 0.0;
          for (long i = 0; i < N; ++i) {
            const double pr = (double)sa[(size_t)mu * N + i] * (double)sb[(size_t)nu * N + i];
            const double ph = two_pi * (double)(i % L) / (double)L;
            r0 += pr; re += pr * std::cos(ph); im += pr * std::sin(ph);
          }
          const size_t idx = ((((size_t)d * P + p) * T + t) * 3 + mu) * 3 + nu;
          if (q0) q0[idx] = r0 / (double)N;
          if (qk) { qk[2 * idx] = re / (double)N; qk[2 * idx + 1] = im / (double)N; }
        }
      }
    }
  }
};

// --------------------------------------------------------------------------------------
// Field-case observables, Eqs. (9)-(11): four real replicas (1),(2),(3),(4) = replicas 0,1,2,3 of a
// sample, all at the same temperature index.  One measurement contributes the summands of Eq. (10):
//   chi_1(k) = sum_{i,j} sum_{mu,nu} s_i^{mu(1)} s_j^{nu(1)} s_i^{mu(2)} s_j^{nu(2)} e^{ik.(R_i-R_j)}
//   chi_2(k) = sum_{i,j} sum_{mu,nu} s_i^{mu(1)} s_j^{nu(1)} s_i^{mu(3)} s_j^{nu(4)} e^{ik.(R_i-R_j)}
//   chi_3(k) = sum_{i,j} sum_{mu,nu} s_i^{mu(1)} s_j^{nu(2)} s_i^{mu(3)} s_j^{nu(4)} e^{ik.(R_i-R_j)}
// for k = 0 and k_min = (2 pi/L)(1,0,0); the thermal average <.> is the caller's running mean over
// measurements and Eq. (11) chi_SG(k) = (1/N)[chi_1 - 2 chi_2 + chi_3]_J its linear combination.  All arithmetic in
// double.  Output chi[D][T][2 (k = 0, k_min)][3 (chi_1, chi_2, chi_3)][2 (re, im)].
//
// chi_field_plain: the definition written out — the double sum over sites and components, nothing factored.  O(N^2).
// chi_field      : the same numbers from A_ab(k) = sum_i (s_i^(a) . s_i^(b)) e^{ik x_i}; in Eq. (10) site i always
//                  carries the index mu in both of its factors and site j the index nu, so the sums over (i, mu) and
//                  (j, nu) factor:  chi_1 = |A_12|^2, chi_2 = A_13 conj(A_14), chi_3 = A_13 conj(A_24).  O(N); pinned
//                  against chi_field_plain in tests/test_oracle_field_chiral.py.
// --------------------------------------------------------------------------------------
template <class Real>
void chi_field_plain_one(Sim<Real>& sim, int d, int t, double* out /*[2][3][2]*/) {
  const long N = sim.N; const int L = sim.L;
  const Real* s[4];
  for (int r = 0; r < 4; ++r) s[r] = sim.spins_of_temp(d, r, t);
  const double two_pi = 6.283185307179586476925286766559;
  for (int ik = 0; ik < 2; ++ik) {
    const double kx = ik == 0 ? 0.0 : two_pi / (double)L;
    double acc[3][2] = {{0, 0}, {0, 0}, {0, 0}};
    for (long i = 0; i < N; ++i) for (long j = 0; j < N; ++j) {
      const double ph = kx * (double)((i % L) - (j % L));
      const double co = std::cos(ph), si = std::sin(ph);
      for (int mu = 0; mu < 3; ++mu) for (int nu = 0; nu < 3; ++nu) {
        const double i1 = (double)s[0][(size_t)mu * N + i], i2 = (double)s[1][(size_t)mu * N + i], i3 = (double)s[2][(size_t)mu * N + i];
        const double j1 = (double)s[0][(size_t)nu * N + j], j2 = (double)s[1][(size_t)nu * N + j], j4 = (double)s[3][(size_t)nu * N + j];
        const double c1 = i1 * j1 * i2 * j2;        // s_i^{mu(1)} s_j^{nu(1)} s_i^{mu(2)} s_j^{nu(2)}
        const double c2 = i1 * j1 * i3 * j4;        // s_i^{mu(1)} s_j^{nu(1)} s_i^{mu(3)} s_j^{nu(4)}
        const double c3 = i1 * j2 * i3 * j4;        // s_i^{mu(1)} s_j^{nu(2)} s_i^{mu(3)} s_j^{nu(4)}
        acc[0][0] += c1 * co; acc[0][1] += c1 * si;
        acc[1][0] += c2 * co; acc[1][1] += c2 * si;
        acc[2][0] += c3 * co; acc[2][1] += c3 * si;
      }
    }
    for (int c = 0; c < 3; ++c) { out[(ik * 3 + c) * 2] = acc[c][0]; out[(ik * 3 + c) * 2 + 1] = acc[c][1]; }
  }
}

template <class Real>
void chi_field_one(Sim<Real>& sim, int d, int t, double* out /*[2][3][2]*/) {
  const long N = sim.N; const int L = sim.L;
  const Real* s[4];
  for (int r = 0; r < 4; ++r) s[r] = sim.spins_of_temp(d, r, t);
  const double two_pi = 6.283185307179586476925286766559;
  const int pa[4] = {0, 0, 0, 1}, pb[4] = {1, 2, 3, 3};     // A_12, A_13, A_14, A_24
  for (int ik = 0; ik < 2; ++ik) {
    double A[4][2];
    for (int p = 0; p < 4; ++p) {
      double re = 0.0, im = 0.0;
      for (long i = 0; i < N; ++i) {
        double dot = 0.0;
        for (int mu = 0; mu < 3; ++mu) dot += (double)s[pa[p]][(size_t)mu * N + i] * (double)s[pb[p]][(size_t)mu * N + i];
        const double ph = ik == 0 ? 0.0 : two_pi * (double)(i % L) / (double)L;
        re += dot * std::cos(ph); im += dot * std::sin(ph);
      }
      A[p][0] = re; A[p][1] = im;
    }
    double* o = out + ik * 6;
    o[0] = A[0][0] * A[0][0] + A[0][1] * A[0][1]; o[1] = 0.0;                                   // |A_12|^2
    o[2] = A[1][0] * A[2][0] + A[1][1] * A[2][1]; o[3] = A[1][1] * A[2][0] - A[1][0] * A[2][1];  // A_13 conj(A_14)
    o[4] = A[1][0] * A[3][0] + A[1][1] * A[3][1]; o[5] = A[1][1] * A[3][0] - A[1][0] * A[3][1];  // A_13 conj(A_24)
  }
}

template <class Real>
void chi_field_all(Sim<Real>& sim, double* chi, bool plain, int n_threads) {
  const int D = sim.D, T = sim.T;
  auto work = [&](int r0, int r1) {
    for (int r = r0; r < r1; ++r) {
      if (plain) chi_field_plain_one(sim, r / T, r % T, chi + (size_t)r * 12);
      else chi_field_one(sim, r / T, r % T, chi + (size_t)r * 12);
    }
  };
  const int n = D * T, nt = std::max(1, std::min(n_threads, n));
  if (nt == 1) { work(0, n); return; }
  std::vector<std::thread> th;
  for (int k = 0; k < nt; ++k) th.emplace_back(work, n * k / nt, n * (k + 1) / nt);
  for (auto& x : th) x.join();
}

// --------------------------------------------------------------------------------------
// Chiral sector, Eqs. (12), (13):
//   kappa_i^alpha = s_{i+alpha} . (s_i x s_{i-alpha}),  alpha = x, y, z (periodic)                              (12)
//   q_c^alpha(k)  = (1/N) sum_i kappa_i^{alpha(a)} kappa_i^{alpha(b)} e^{ik.R_i}                               (13)
// for replica pairs a < b at the same temperature, k = 0 and k_min = (2 pi/L)(1,0,0) for every alpha (the paper defines
// one k_min; reading 22).  The local chirality is a per-site quantity of the spins and is formed
// in the spins' precision Real with this fixed operation order:
//   c = s_i x s_{i-alpha}:  c_x = fma(b_y, m_z, -(b_z*m_y)), c_y = fma(b_z, m_x, -(b_x*m_z)), c_z = fma(b_x, m_y, -(b_y*m_x))
//   kappa = fma(p_z, c_z, fma(p_y, c_y, p_x*c_x)),   p = s_{i+alpha}, b = s_i, m = s_{i-alpha};
// the product kappa^(a) kappa^(b) and the sums are double.  chi_CG (Eq. 14) and xi_c (Eq. 15) are the caller's averages.
// Output qc0[D][P][T][3], qck[D][P][T][3][2 (re, im)].
// --------------------------------------------------------------------------------------
template <class Real>
Real chirality(const Sim<Real>& sim, const Real* s, long i, int alpha) {
  const long N = sim.N;
  const long ip = sim.nbr(i, alpha, +1), im = sim.nbr(i, alpha, -1);
  const Real p[3] = { s[ip], s[N + ip], s[2 * N + ip] };
  const Real b[3] = { s[i], s[N + i], s[2 * N + i] };
  const Real m[3] = { s[im], s[N + im], s[2 * N + im] };
  const Real cx = fma_(b[1], m[2], -(b[2] * m[1]));
  const Real cy = fma_(b[2], m[0], -(b[0] * m[2]));
  const Real cz = fma_(b[0], m[1], -(b[1] * m[0]));
  return fma_(p[2], cz, fma_(p[1], cy, p[0] * cx));
}

template <class Real>
void measure_chiral(Sim<Real>& sim, double* qc0, double* qck, double* kappa_out /*[D][O][T][3][N] or null*/) {
  const int D = sim.D, O = sim.O, T = sim.T, L = sim.L; const long N = sim.N;
  const int P = O * (O - 1) / 2;
  const double two_pi = 6.283185307179586476925286766559;
  std::vector<Real> ka((size_t)3 * N), kb((size_t)3 * N);
  if (kappa_out)
    for (int d = 0; d < D; ++d) for (int o = 0; o < O; ++o) for (int t = 0; t < T; ++t) {
      const Real* s = sim.spins_of_temp(d, o, t);
      for (int al = 0; al < 3; ++al) for (long i = 0; i < N; ++i)
        kappa_out[((((size_t)d * O + o) * T + t) * 3 + al) * N + i] = (double)chirality(sim, s, i, al);
    }
  if (!qc0 && !qck) return;
  for (int d = 0; d < D; ++d) {
    int p = 0;
    for (int a = 0; a < O; ++a) for (int b = a + 1; b < O; ++b, ++p) for (int t = 0; t < T; ++t) {
      const Real* sa = sim.spins_of_temp(d, a, t);
      const Real* sb = sim.spins_of_temp(d, b, t);
      for (int al = 0; al < 3; ++al) {
        double r0 = 0.0, re = 0.0, im = 0.0;
        for (long i = 0; i < N; ++i) {
          const double pr = (double)chirality(sim, sa, i, al) * (double)chirality(sim, sb, i, al);
          const double ph = two_pi * (double)(i % L) / (double)L;
          r0 += pr; re += pr * std::cos(ph); im += pr * std::sin(ph);
        }
        const size_t idx = (((size_t)d * P + p) * T + t) * 3 + al;
        if (qc0) qc0[idx] = r0 / (double)N;
        if (qck) { qck[2 * idx] = re / (double)N; qck[2 * idx + 1] = im / (double)N; }
      }
    }
  }
}

struct Handle { int precision; Sim<float>* f; Sim<double>* d; };

}  // namespace

#define ORC_DISPATCH(h, expr) do { Handle* H_ = (Handle*)(h); if (H_->precision == 32) { auto& sim = *H_->f; expr; } else { auto& sim = *H_->d; expr; } } while (0)

extern "C" {

// ---- unit-level entry points (used by the pins) ----
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) { philox4x32_10(ctr, key, out); }
double orc_u01(uint32_t w) { return u01<double>(w); }
float orc_u01_f32(uint32_t w) { return u01<float>(w); }
float orc_spec_omexp_f32(float x) { return omexp(x); }
float orc_spec_log1m_f32(float y) { return log1m(y); }
void orc_spec_sincos2pi_f32(float u, float* s, float* c) { sincos2pi(u, *s, *c); }
void orc_or_reflect_f32(const float s[3], const float h[3], float out[3]) { or_reflect<float>(s, h, out); }
void orc_or_reflect_f64(const double s[3], const double h[3], double out[3]) { or_reflect<double>(s, h, out); }
void orc_hb_draw_f32(const float h[3], float beta, float u1, float u2, float out[3]) { hb_draw<float>(h, beta, u1, u2, out); }
void orc_hb_draw_f64(const double h[3], double beta, double u1, double u2, double out[3]) { hb_draw<double>(h, beta, u1, u2, out); }
// many heat-bath draws of one spin in a fixed field from the Philox stream (HB domain, site 0, system 0,
// sweep counter k = 0..n-1); out[n][3].  For the Langevin-law pin.
void orc_hb_sample(int precision, const double h[3], double beta, uint64_t seed, long n, double* out) {
  uint32_t k[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
  for (long j = 0; j < n; ++j) {
    uint32_t ctr[4], w[4];
    make_counter(0u, (uint64_t)j, 0u, DOMAIN_HB, ctr);
    philox4x32_10(ctr, k, w);
    if (precision == 32) {
      const float hf[3] = { (float)h[0], (float)h[1], (float)h[2] }; float o[3];
      hb_draw<float>(hf, (float)beta, u01<float>(w[0]), u01<float>(w[1]), o);
      out[3 * j] = o[0]; out[3 * j + 1] = o[1]; out[3 * j + 2] = o[2];
    } else {
      hb_draw<double>(h, beta, u01<double>(w[0]), u01<double>(w[1]), out + 3 * j);
    }
  }
}

// ---- simulation object ----
void* orc_create(int L, int D, int O, int T, const float* temps, uint64_t seed, uint64_t sample_offset, int precision) {
  if (L < 2 || (L & 1) || D < 1 || O < 1 || T < 1 || !temps || (precision != 32 && precision != 64)) return nullptr;
  for (int t = 0; t < T; ++t) { if (!(temps[t] > 0.f)) return nullptr; if (t > 0 && !(temps[t] > temps[t - 1])) return nullptr; }
  Handle* h = new Handle{precision, nullptr, nullptr};
  if (precision == 32) h->f = new Sim<float>(L, D, O, T, temps, seed, sample_offset);
  else h->d = new Sim<double>(L, D, O, T, temps, seed, sample_offset);
  return h;
}
void orc_destroy(void* h) { if (!h) return; Handle* H_ = (Handle*)h; delete H_->f; delete H_->d; delete H_; }

void orc_set_disorder(void* h, const float* J, const float* Hf /*may be null*/) {
  ORC_DISPATCH(h, {
    std::copy(J, J + sim.J.size(), sim.J.begin());
    if (Hf) std::copy(Hf, Hf + sim.H.size(), sim.H.begin()); else std::fill(sim.H.begin(), sim.H.end(), 0.f);
    sim.have_disorder = true;
  });
}
void orc_init_spins(void* h) { ORC_DISPATCH(h, sim.init_spins()); }
// S[d][o][t][3][N] by temperature index, as double (exact for the float instantiation)
void orc_set_spins(void* h, const double* S) {
  ORC_DISPATCH(h, {
    const size_t n3 = (size_t)3 * sim.N;
    for (int d = 0; d < sim.D; ++d) for (int o = 0; o < sim.O; ++o) for (int t = 0; t < sim.T; ++t) {
      auto* dst = sim.spins_of_temp(d, o, t);
      const double* src = S + (((size_t)d * sim.O + o) * sim.T + t) * n3;
      for (size_t j = 0; j < n3; ++j) dst[j] = (std::remove_reference_t<decltype(*dst)>)src[j];
    }
    sim.have_spins = true;
  });
}
void orc_get_spins(void* h, double* S) {
  ORC_DISPATCH(h, {
    const size_t n3 = (size_t)3 * sim.N;
    for (int d = 0; d < sim.D; ++d) for (int o = 0; o < sim.O; ++o) for (int t = 0; t < sim.T; ++t) {
      const auto* src = sim.spins_of_temp(d, o, t);
      double* dst = S + (((size_t)d * sim.O + o) * sim.T + t) * n3;
      for (size_t j = 0; j < n3; ++j) dst[j] = (double)src[j];
    }
  });
}
void orc_sweep(void* h, int n_or, int n_hb, int n_threads) { ORC_DISPATCH(h, sim.sweep(n_or, n_hb, n_threads)); }
void orc_energy(void* h, double* E) { ORC_DISPATCH(h, sim.energy(E)); }
void orc_energy_plain(void* h, double* E) { ORC_DISPATCH(h, sim.energy_plain(E)); }
void orc_pt_swap(void* h, int32_t* accepted) { ORC_DISPATCH(h, sim.pt_swap(accepted)); }
void orc_measure(void* h, double* E, double* M, double* q0, double* qk) { ORC_DISPATCH(h, sim.measure(E, M, q0, qk)); }
// slot_of_temp[D][O][T] and counters {k_hb, k_pt}
void orc_get_state(void* h, int32_t* slot_of_temp, uint64_t counters[2]) {
  ORC_DISPATCH(h, {
    if (slot_of_temp) std::copy(sim.conf_of_temp.begin(), sim.conf_of_temp.end(), slot_of_temp);
    if (counters) { counters[0] = sim.k_hb; counters[1] = sim.k_pt; }
  });
}
// field-case observables (Eq. 10): chi[D][T][2][3][2]; plain != 0: the O(N^2) definition, else the factored form.  Needs O >= 4.
int orc_chi_field(void* h, double* chi, int plain, int n_threads) {
  int rc = 0;
  ORC_DISPATCH(h, { if (sim.O < 4) rc = -1; else chi_field_all(sim, chi, plain != 0, n_threads); });
  return rc;
}
// chirality (Eqs. 12, 13): qc0[D][P][T][3], qck[D][P][T][3][2], optionally the local chiralities kappa[D][O][T][3][N]
void orc_measure_chiral(void* h, double* qc0, double* qck, double* kappa) { ORC_DISPATCH(h, measure_chiral(sim, qc0, qck, kappa)); }
// Eq. (8) / Eq. (15): second-moment correlation length from chi(0), chi(k_min)
double orc_xi_second_moment(double chi_0, double chi_k, int L) {
  const double kmin = 6.283185307179586476925286766559 / (double)L;
  return std::sqrt(chi_0 / chi_k - 1.0) / (2.0 * std::sin(0.5 * kmin));
}
// parallel-tempering diagnostics (Fig. 3)
void orc_pt_diag_reset(void* h) { ORC_DISPATCH(h, sim.pt_diag_reset()); }
void orc_pt_diag_get(void* h, int64_t* moved, int64_t* trav, uint64_t* n_pass, double* p_diff) { ORC_DISPATCH(h, sim.pt_diag_get(moved, trav, n_pass, p_diff)); }
void orc_set_counters(void* h, const uint64_t counters[2]) { ORC_DISPATCH(h, { sim.k_hb = counters[0]; sim.k_pt = counters[1]; }); }

}  // extern "C"
