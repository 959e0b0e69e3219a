// sanitizer_main.cpp — stand-alone program around zmarch_driver.cpp for tests/test_zmarch_sanitizers_on_host.py: the sweep
// kernel on the host execution model (emu.h) built as an EXECUTABLE with -fsanitize=thread or -fsanitize=address (a
// sanitised shared object cannot be loaded into an unsanitised python).  Inputs are arbitrary numbers on heap blocks of
// exactly the sizes the C ABI states, so that a read or write past any array is seen.  No result is checked here (the
// bit-for-bit comparison with the oracle is tests/test_zmarch_on_host.py); compile with -DEMU_L=8|16|32|64.
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <vector>

#define SAN_CAT2(a, b) a##b
#define SAN_CAT(a, b) SAN_CAT2(a, b)
extern "C" int SAN_CAT(emu_zmarch_l, EMU_L)(int G, int mode, int D, int O, int T, const float* temps, unsigned long long seed,
                                             unsigned long long sample_offset, unsigned long long k_hb, int n_or, int n_hb,
                                             const float* J, const float* H, float* S, double* E, double* M, int fast_math);

static uint64_t state = 0x9E3779B97F4A7C15ull;
static float unit() {                       // xorshift64*, mapped to (-1, 1)
  state ^= state >> 12; state ^= state << 25; state ^= state >> 27;
  return (float)((double)((state * 0x2545F4914F6CDD1Dull) >> 11) / 4503599627370496.0 - 1.0);
}

int main(int argc, char** argv) {
  if (argc < 8) { std::fprintf(stderr, "usage: %s G D O T n_or n_hb mode [fast_math]\n", argv[0]); return 64; }
  const int L = EMU_L, G = std::atoi(argv[1]), D = std::atoi(argv[2]), O = std::atoi(argv[3]), T = std::atoi(argv[4]);
  const int n_or = std::atoi(argv[5]), n_hb = std::atoi(argv[6]), mode = std::atoi(argv[7]), fast = argc > 8 ? std::atoi(argv[8]) : 0;
  const size_t N = (size_t)L * L * L, R = (size_t)D * O * T;
  std::vector<float> J(D * 3 * N), H(D * 3 * N), S(R * 3 * N), temps(T);
  for (float& x : J) x = 1.5f * unit();
  for (float& x : H) x = 0.1f * unit();
  for (int t = 0; t < T; ++t) temps[t] = 0.1f + 0.05f * (float)t;
  for (size_t r = 0; r < R; ++r)
    for (size_t i = 0; i < N; ++i) {
      float a = unit(), b = unit(), c = unit();
      const float n = std::sqrt(a * a + b * b + c * c) + 1e-6f;
      S[(r * 3 + 0) * N + i] = a / n; S[(r * 3 + 1) * N + i] = b / n; S[(r * 3 + 2) * N + i] = c / n;
    }
  std::vector<double> E(R), M(3 * R);
  const int rc = SAN_CAT(emu_zmarch_l, EMU_L)(G, mode, D, O, T, temps.data(), 11ull, 3ull, 0ull, n_or, n_hb, J.data(), H.data(),
                                               S.data(), E.data(), M.data(), fast);
  double e = 0.0;
  for (double x : E) e += x;
  std::printf("L=%d G=%d D=%d O=%d T=%d rc=%d sum E=%.6f\n", L, G, D, O, T, rc, e);
  return rc == 0 ? 0 : 1;
}
