"""Parallel-tempering diagnostics (Fig. 3): the accumulator against a brute-force tracker on oracle runs
(CPU), and — on the GPU — the paper's qualitative finding and its one printed number, N_tunn ~ 3 closed loops per
configuration in 2 x 10^4 steps on a geometric ladder at L = 8 (a weak sanity check: the paper does not print the
temperature interval of that run next to the number; "parity unpinned" in the sense of DESIGN.md)."""
import numpy as np
import pytest
import torch

import hsg_inputs
import oracle
from paper_1204_6192_b200.pt_diagnostics import PtDiagnostics


def test_accumulator_matches_a_brute_force_tracker_on_an_oracle_run():
    L, D, O, T, steps = 4, 2, 2, 5, 400
    temps = hsg_inputs.geometric_ladder(0.4, 2.0, T)
    sim = oracle.Oracle(L, D, O, temps, 9, precision=32)
    sim.set_disorder(hsg_inputs.couplings(L, D, 3), None); sim.init_spins()
    perm0 = np.asarray(sim.get_state()[0]).reshape(D, O, T)
    diag = PtDiagnostics(perm=torch.from_numpy(perm0.copy()))
    # brute force: follow every configuration slot through the temperatures
    last = np.zeros((D, O, T), dtype=int); trav = np.zeros((D, O, T), dtype=int); moved = np.zeros((D, O, T), dtype=int)
    def touch(perm):
        for d in range(D):
            for o in range(O):
                for t_end, tag in ((0, 1), (T - 1, -1)):
                    s = perm[d, o, t_end]
                    if last[d, o, s] == -tag:
                        trav[d, o, s] += 1
                    last[d, o, s] = tag
    touch(perm0)
    prev = perm0
    for _ in range(steps):
        sim.sweep(1, 1); sim.pt_swap()
        perm = np.asarray(sim.get_state()[0]).reshape(D, O, T)
        diag.after_pt_swap(torch.from_numpy(perm.copy()))
        moved += (perm != prev)
        touch(perm); prev = perm
    assert np.array_equal(diag.n_tunnel(), trav // 2)
    np.testing.assert_allclose(diag.p_diff(), moved.mean(axis=(0, 1)) / steps)
    assert trav.sum() > 0 and (np.sort(perm, axis=2) == np.arange(T)).all()


@pytest.mark.gpu
def test_geometric_ladder_tunnels_and_the_arithmetic_one_stalls_at_low_temperature():
    import paper_1204_6192_b200 as hsg
    L, D, O, T, steps = 8, 16, 2, 32, 20000             # 10 OR + 1 HB + 1 PT pass per step, H = 0
    J = hsg_inputs.couplings(L, D, 31)
    res = {}
    for name, temps in (("geometric", hsg_inputs.geometric_ladder(0.1, 0.6, T)),
                        ("arithmetic", np.linspace(0.1, 0.6, T).astype(np.float32))):
        eng = hsg.hsg_create(L, D, O, temps, 77)
        eng.set_disorder(J, None); eng.init_spins()
        diag = PtDiagnostics(eng)
        for _ in range(steps):
            eng.sweep(10, 1); eng.pt_swap(want_flags=False); diag.after_pt_swap()
        res[name] = (diag.n_tunnel().mean(), diag.p_diff())
    (ng, pg), (na, pa) = res["geometric"], res["arithmetic"]
    assert 1.0 < ng < 10.0                              # paper: N_tunn ~ 3 (same order; measured here: ~5)
    assert na < 0.7 * ng                                # the arithmetic ladder tunnels less
    assert pg[1:-1].min() > 0.4 and pg[1:-1].max() < 0.8          # geometric: p_diff flat over the ladder (Fig. 3)
    assert pa[0] < 0.05 < pg[0] and pa[1] < 0.15                  # arithmetic: exchanges at the lowest temperatures starved
