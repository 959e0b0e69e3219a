"""Parallel-tempering diagnostics (Fig. 3).  CPU: the oracle's tracker against a brute-force tracker that
follows every configuration through the permutations.  GPU: the device counters of hsg_pt_swap against the oracle's,
element by element on the same seeds (they must be identical, since the swap decisions are), and — as a separate sanity
check — the paper's qualitative finding and its one printed number, N_tunn ~ 3 closed loops per configuration in 2 x 10^4
steps on a geometric ladder at L = 8 (weak: the paper does not print the temperature interval of that run next to the
number; "parity unpinned" in the sense of DESIGN.md)."""
import numpy as np
import pytest

import hsg_inputs
import oracle


def test_oracle_tracker_matches_a_brute_force_tracker():
    L, D, O, T, steps = 4, 2, 2, 5, 400
    temps = hsg_inputs.geometric_ladder(0.4, 2.0, T)
    sim = oracle.Oracle(L, D, O, temps, 9, precision=32)
    sim.set_disorder(hsg_inputs.couplings(L, D, 3), None); sim.init_spins()
    sim.sweep(0, 2); sim.pt_swap(); sim.pt_swap()             # start from a scrambled permutation
    perm0 = np.asarray(sim.get_state()[0]).reshape(D, O, T).copy()
    sim.pt_diag_reset()
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
        perm = np.asarray(sim.get_state()[0]).reshape(D, O, T).copy()
        moved += (perm != prev)
        touch(perm); prev = perm
    m, tr, n, p = sim.pt_diag_get()
    assert n == steps
    assert np.array_equal(m, moved) and np.array_equal(tr, trav)
    np.testing.assert_allclose(p, moved.mean(axis=(0, 1)) / steps, rtol=1e-15)
    assert trav.sum() > 0 and (trav // 2).sum() > 0 and (np.sort(perm, axis=2) == np.arange(T)).all()
    # a reset starts over
    sim.pt_diag_reset()
    m, tr, n, p = sim.pt_diag_get()
    assert n == 0 and m.sum() == 0 and tr.sum() == 0 and (p == 0).all()


def test_tracker_on_a_hand_made_walk():
    """T = 2, one chain: the two configurations exchange on every accepted pass; each exchange is a traversal for both
    (they start at opposite end points), so after n accepted passes: traversals = n each, loops = n // 2."""
    L, T = 4, 2
    temps = np.array([5.0, 5.000001], dtype=np.float32)       # equal temperatures: dbeta*dE ~ 0 -> (almost) always accepted
    sim = oracle.Oracle(L, 1, 1, temps, 3, precision=32)
    sim.set_disorder(hsg_inputs.couplings(L, 1, 3), None); sim.init_spins()
    sim.pt_diag_reset()
    n_acc = 0
    for _ in range(7):
        sim.sweep(0, 1)
        n_acc += int(sim.pt_swap().sum())
    m, tr, n, p = sim.pt_diag_get()
    assert n == 7 and n_acc >= 5
    assert (tr[0, 0] == n_acc).all() and (m[0, 0] == n_acc).all()
    np.testing.assert_allclose(p, n_acc / 7)


@pytest.mark.gpu
@pytest.mark.parametrize("kernel", ["generic", "zmarch"])
def test_device_counters_match_the_oracle_tracker_element_by_element(kernel):
    import paper_1204_6192_b200 as hsg
    from paper_1204_6192_b200.pt_diagnostics import PtDiagnostics
    L, D, O, T, steps = 8, 3, 2, 6, 300
    temps = hsg_inputs.geometric_ladder(0.8, 0.9, T)             # warm and closely spaced: tunnels within a few hundred passes
    J = hsg_inputs.couplings(L, D, 31); H = hsg_inputs.gaussian_field(L, D, 0.1, 31)
    eng = hsg.hsg_create(L, D, O, temps, 77, kernel=kernel)
    orc = oracle.Oracle(L, D, O, temps, 77, precision=32, n_threads=8)
    for s in (eng, orc):
        s.set_disorder(J, H); s.init_spins()
    for _ in range(3):                                          # scramble first: the reset must read the CURRENT permutation
        eng.sweep(1, 1); orc.sweep(1, 1); eng.pt_swap(); orc.pt_swap()
    diag = PtDiagnostics(eng); orc.pt_diag_reset()
    for step in range(steps):
        eng.sweep(2, 1); orc.sweep(2, 1)
        acc = eng.pt_swap().cpu().numpy()
        assert np.array_equal(acc, orc.pt_swap()), step
    moved, trav, p_diff, n = eng.pt_diag_get()
    m_o, t_o, n_o, p_o = orc.pt_diag_get()
    assert n == n_o == steps
    assert np.array_equal(moved.cpu().numpy(), m_o) and np.array_equal(trav.cpu().numpy(), t_o)
    np.testing.assert_allclose(p_diff.cpu().numpy(), p_o, rtol=1e-15)
    assert np.array_equal(diag.n_tunnel(), t_o // 2) and (t_o // 2).sum() > 0
    np.testing.assert_allclose(diag.p_diff(), p_o, rtol=1e-15)


@pytest.mark.gpu
def test_geometric_ladder_tunnels_and_the_arithmetic_one_stalls_at_low_temperature():
    import paper_1204_6192_b200 as hsg
    from paper_1204_6192_b200.pt_diagnostics import PtDiagnostics
    L, D, O, T, steps = 8, 16, 2, 32, 20000             # 10 OR + 1 HB + 1 PT pass per step, H = 0
    J = hsg_inputs.couplings(L, D, 31)
    res = {}
    for name, temps in (("geometric", hsg_inputs.geometric_ladder(0.1, 0.6, T)),
                        ("arithmetic", np.linspace(0.1, 0.6, T).astype(np.float32))):
        eng = hsg.hsg_create(L, D, O, temps, 77)
        eng.set_disorder(J, None); eng.init_spins()
        diag = PtDiagnostics(eng)
        for _ in range(steps):
            eng.sweep(10, 1); eng.pt_swap(want_flags=False)
        assert diag.n_pass() == steps
        res[name] = (diag.n_tunnel().mean(), diag.p_diff())
    (ng, pg), (na, pa) = res["geometric"], res["arithmetic"]
    assert 1.0 < ng < 10.0                              # paper: N_tunn ~ 3 (same order; measured here: ~5)
    assert na < 0.7 * ng                                # the arithmetic ladder tunnels less
    assert pg[1:-1].min() > 0.4 and pg[1:-1].max() < 0.8          # geometric: p_diff flat over the ladder (Fig. 3)
    assert pa[0] < 0.05 < pg[0] and pa[1] < 0.15                  # arithmetic: exchanges at the lowest temperatures starved
