"""Pins for the oracle's measurements: magnetisation and the overlap tensor q^{mu nu}(k) of
PAPER.md:53-58 (Eqs. 5, 6) at k = 0 and k_min = (2 pi/L)(1,0,0).  CPU only."""
import numpy as np

import hsg_inputs
import oracle


def _sim(L, D, O, T, precision=32):
    temps = hsg_inputs.geometric_ladder(0.1, 0.3, T)
    sim = oracle.Oracle(L, D, O, temps, 3, precision=precision)
    sim.set_disorder(hsg_inputs.couplings(L, D, 4), hsg_inputs.gaussian_field(L, D, 0.1, 4))
    return sim


def test_overlap_brute_force_and_magnetisation():
    L, D, O, T = 4, 2, 3, 2            # three replicas -> pairs (0,1),(0,2),(1,2)
    sim = _sim(L, D, O, T)
    S = hsg_inputs.unit_spins(L, D, O, T, 12)
    sim.set_spins(S)
    E, M, q0, qk = sim.measure()
    S64 = S.astype(np.float64)
    np.testing.assert_allclose(M, S64.mean(axis=(4, 5, 6)), atol=1e-14)
    np.testing.assert_allclose(E, sim.energy(), atol=0)
    x = np.arange(L)
    phase = np.exp(2j * np.pi * x / L)                       # e^{+i k x}, k along x (fastest index)
    pairs = [(0, 1), (0, 2), (1, 2)]
    for p, (a, b) in enumerate(pairs):
        for d in range(D):
            for t in range(T):
                ref0 = np.einsum("mzyx,nzyx->mn", S64[d, a, t], S64[d, b, t]) / L**3
                refk = np.einsum("mzyx,nzyx,x->mn", S64[d, a, t], S64[d, b, t], phase) / L**3
                np.testing.assert_allclose(q0[d, p, t], ref0, atol=1e-14)
                np.testing.assert_allclose(qk[d, p, t, :, :, 0], refk.real, atol=1e-14)
                np.testing.assert_allclose(qk[d, p, t, :, :, 1], refk.imag, atol=1e-14)


def test_identical_replicas_have_unit_trace_and_rotation_invariant_q2():
    L, D, O, T = 4, 1, 2, 2
    sim = _sim(L, D, O, T, precision=64)
    S = hsg_inputs.unit_spins(L, D, O, T, 13).astype(np.float64)
    S[:, 1] = S[:, 0]
    sim.set_spins(S)
    _, _, q0, _ = sim.measure()
    np.testing.assert_allclose(np.trace(q0[0, 0, 0]), 1.0, atol=1e-7)      # fp32-rounded unit vectors
    # replica 2 = R * replica 1: q -> q R^T, Frobenius norm unchanged
    th = 0.7
    R = np.array([[np.cos(th), -np.sin(th), 0], [np.sin(th), np.cos(th), 0], [0, 0, 1]]) @ np.array([[1, 0, 0], [0, 0.6, -0.8], [0, 0.8, 0.6]])
    S2 = S.copy()
    S2[:, 1] = np.einsum("ab,dtbzyx->dtazyx", R, S[:, 0])
    sim.set_spins(S2)
    _, _, q0r, _ = sim.measure()
    for t in range(T):
        np.testing.assert_allclose(q0r[0, 0, t], q0[0, 0, t] @ R.T, atol=1e-12)
        np.testing.assert_allclose((q0r[0, 0, t]**2).sum(), (q0[0, 0, t]**2).sum(), atol=1e-12)


def test_plane_wave_overlap():
    """replica 1 = (cos kx, sin kx, 0) with k = 2 pi/L, replica 2 = (1,0,0):
    q^{xx}(k_min) = 1/2, q^{yx}(k_min) = i/2, everything else and all of q(0) zero."""
    L, D, O, T = 8, 1, 2, 1
    sim = _sim(L, D, O, T, precision=64)
    S = np.zeros((D, O, T, 3, L, L, L))
    x = np.arange(L)
    S[0, 0, 0, 0] = np.cos(2 * np.pi * x / L)[None, None, :]
    S[0, 0, 0, 1] = np.sin(2 * np.pi * x / L)[None, None, :]
    S[0, 1, 0, 0] = 1.0
    sim.set_spins(S)
    _, M, q0, qk = sim.measure()
    np.testing.assert_allclose(q0, 0, atol=1e-15)
    ref = np.zeros((3, 3, 2)); ref[0, 0, 0] = 0.5; ref[1, 0, 1] = 0.5
    np.testing.assert_allclose(qk[0, 0, 0], ref, atol=1e-15)
    np.testing.assert_allclose(M[0, 1, 0], [1, 0, 0], atol=0)
    np.testing.assert_allclose(M[0, 0, 0], 0, atol=1e-15)
    # a wave along y is invisible to k_min = (2 pi/L)(1,0,0)
    S[0, 0, 0, 0] = np.cos(2 * np.pi * x / L)[None, :, None]
    S[0, 0, 0, 1] = np.sin(2 * np.pi * x / L)[None, :, None]
    sim.set_spins(S)
    np.testing.assert_allclose(sim.measure()[3], 0, atol=1e-15)


def test_measure_follows_the_temperature_labels_after_a_swap():
    """q pairs the two replicas that hold the SAME temperature, whatever slot they sit in."""
    L, D, O, T = 4, 1, 2, 4
    temps = hsg_inputs.geometric_ladder(1.0, 4.0, T)          # hot ladder: swaps are frequent
    sim = oracle.Oracle(L, D, O, temps, 19, precision=32)
    sim.set_disorder(hsg_inputs.couplings(L, D, 4), None); sim.init_spins()
    moved = False
    for _ in range(10):
        sim.sweep(1, 1)
        acc = sim.pt_swap()
        S = sim.get_spins()                                    # by temperature index
        _, M, q0, _ = sim.measure()
        for t in range(T):
            ref = np.einsum("mzyx,nzyx->mn", S[0, 0, t], S[0, 1, t]) / L**3
            np.testing.assert_allclose(q0[0, 0, t], ref, atol=1e-14)
        np.testing.assert_allclose(M, S.mean(axis=(4, 5, 6)), atol=1e-14)
        moved |= bool(acc[0, 0].any() != acc[0, 1].all())
    perm, _ = sim.get_state()
    assert not (perm[0, 0] == perm[0, 1]).all() or moved
