"""One small pass of the hot path through the C ABI, for compute-sanitizer (memcheck / racecheck / synccheck):

    compute-sanitizer --tool racecheck python tests/sanitizer_case.py L D O T n_or n_hb [kernel]

runs hsg_init_spins, hsg_sweep(n_or, n_hb) twice (the second call exercises the fused E/m reduction on warm rings),
hsg_pt_swap and hsg_measure, and prints a checksum.  The records kept under profiles/ name this command.
Not collected by pytest (no test_ prefix)."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import hsg_inputs  # noqa: E402


def main():
    L, D, O, T, n_or, n_hb = (int(x) for x in sys.argv[1:7])
    kernel = sys.argv[7] if len(sys.argv) > 7 else "auto"
    import paper_1204_6192_b200 as hsg
    temps = hsg_inputs.geometric_ladder(0.08, 0.30, T)
    eng = hsg.hsg_create(L, D, O, temps, 5, kernel=kernel)
    eng.set_disorder(hsg_inputs.couplings(L, D, 5), hsg_inputs.gaussian_field(L, D, 0.1, 5))
    eng.init_spins()
    for _ in range(2):
        eng.sweep(n_or, n_hb)
    acc = eng.pt_swap()
    E, M, q0, qk = eng.measure()
    eng.synchronize()
    print(f"sanitizer_case L={L} D={D} O={O} T={T} sweep({n_or},{n_hb}) x2 kernel={eng.last_sweep_kernel()} "
          f"sum|S|={eng.get_spins().abs().sum().item():.6f} sumE={E.sum().item():.9f} acc={int(acc.sum().item())}")


if __name__ == "__main__":
    main()
