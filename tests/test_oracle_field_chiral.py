"""Pins for the oracle's field-case observables (Eqs. 8-11) and chiral sector (PAPER.md:94-109,
Eqs. 12-15): brute force on small lattices, frozen / inverted / rotated replicas, a conical spiral with a closed-form
chirality, and a free-spin model whose connected susceptibility is known in closed form.  CPU only."""
import math

import numpy as np
import pytest

import hsg_inputs
import oracle


def langevin(a):
    return 1.0 / np.tanh(a) - 1.0 / a


def _sim(L, D, O, T, precision=64, n_threads=4):
    temps = hsg_inputs.geometric_ladder(0.1, 0.3, T)
    sim = oracle.Oracle(L, D, O, temps, 3, precision=precision, n_threads=n_threads)
    sim.set_disorder(hsg_inputs.couplings(L, D, 4), hsg_inputs.gaussian_field(L, D, 0.1, 4))
    return sim


def _rot(th=0.7):
    return np.array([[np.cos(th), -np.sin(th), 0], [np.sin(th), np.cos(th), 0], [0, 0, 1]]) @ np.array([[1, 0, 0], [0, 0.6, -0.8], [0, 0.8, 0.6]])


# ---------------------------------------------------------------------- field case, Eqs. (9)-(11)
def _chi_einsum(S4, L):
    """Eq. (10) literally, as einsums over (mu, i) and (nu, j) with the phase e^{ik(x_i - x_j)}.  S4[4][3][N]."""
    N = L**3
    x = np.arange(N) % L
    out = np.zeros((2, 3), dtype=complex)
    for ik, k in enumerate((0.0, 2 * np.pi / L)):
        ph = np.exp(1j * k * x)
        s1, s2, s3, s4 = S4
        out[ik, 0] = np.einsum("mi,nj,mi,nj,i,j->", s1, s1, s2, s2, ph, ph.conj())
        out[ik, 1] = np.einsum("mi,nj,mi,nj,i,j->", s1, s1, s3, s4, ph, ph.conj())
        out[ik, 2] = np.einsum("mi,nj,mi,nj,i,j->", s1, s2, s3, s4, ph, ph.conj())
    return out


@pytest.mark.parametrize("precision", [64, 32])
def test_chi_field_plain_and_factored_match_the_einsum_of_eq10(precision):
    L, D, O, T = 4, 2, 4, 2
    sim = _sim(L, D, O, T, precision)
    S = hsg_inputs.unit_spins(L, D, O, T, 31)
    sim.set_spins(S)
    plain, fact = sim.chi_field(plain=True), sim.chi_field(plain=False)
    N = L**3
    for d in range(D):
        for t in range(T):
            ref = _chi_einsum(S[d, :, t].astype(np.float64).reshape(4, 3, N), L)
            for got in (plain, fact):
                np.testing.assert_allclose(got[d, t, :, :, 0], ref.real, rtol=0, atol=1e-9)
                np.testing.assert_allclose(got[d, t, :, :, 1], ref.imag, rtol=0, atol=1e-9)
    np.testing.assert_allclose(fact, plain, rtol=0, atol=1e-9)
    assert np.abs(plain[:, :, 0, :, 1]).max() < 1e-9              # k = 0: real
    assert np.abs(plain[:, :, 1, 1:, 1]).max() > 1e-3             # chi_2, chi_3 of ONE measurement at k_min are complex
    assert (plain[:, :, :, 0, 0] >= 0).all() and np.abs(plain[:, :, :, 0, 1]).max() < 1e-9   # chi_1 = |.|^2


def test_chi_field_needs_four_replicas_and_uses_the_first_four():
    sim = _sim(4, 1, 3, 1)
    sim.set_spins(hsg_inputs.unit_spins(4, 1, 3, 1, 1))
    with pytest.raises(ValueError):
        sim.chi_field()
    S = hsg_inputs.unit_spins(4, 1, 5, 1, 2)
    a = _sim(4, 1, 5, 1); a.set_spins(S)
    b = _sim(4, 1, 4, 1); b.set_spins(S[:, :4])
    np.testing.assert_array_equal(a.chi_field(), b.chi_field())


def test_frozen_replicas_have_no_connected_part_and_rotations_change_nothing():
    L, D, T = 4, 1, 2
    N = L**3
    sim = _sim(L, D, 4, T)
    S = hsg_inputs.unit_spins(L, D, 4, T, 7).astype(np.float64)
    S[:, 1] = S[:, 0]; S[:, 2] = S[:, 0]; S[:, 3] = S[:, 0]       # <s s> = <s><s>: chi_ij = 0
    sim.set_spins(S)
    chi = sim.chi_field(plain=True)
    np.testing.assert_allclose(chi[:, :, 0, :, 0], N**2, rtol=1e-6)            # (sum_i s_i.s_i)^2, fp32-rounded unit vectors
    conn = chi[..., 0, :] - 2 * chi[..., 1, :] + chi[..., 2, :]
    assert np.abs(conn).max() < 1e-7 * N**2
    # a global rotation of all four replicas (the field rotates with them) leaves every summand unchanged
    S = hsg_inputs.unit_spins(L, D, 4, T, 8).astype(np.float64)
    sim.set_spins(S); c0 = sim.chi_field()
    sim.set_spins(np.einsum("ab,dotbzyx->dotazyx", _rot(), S)); c1 = sim.chi_field()
    np.testing.assert_allclose(c1, c0, atol=1e-9)
    # exchanging the roles (3) <-> (4) conjugates nothing in chi_1 and maps chi_2 -> conj-partner A_14 conj(A_13)
    S2 = S.copy(); S2[:, 2], S2[:, 3] = S[:, 3], S[:, 2]
    sim.set_spins(S2); c2 = sim.chi_field()
    np.testing.assert_allclose(c2[..., 0, :], c0[..., 0, :], atol=1e-9)
    np.testing.assert_allclose(c2[..., 1, 0], c0[..., 1, 0], atol=1e-9)
    np.testing.assert_allclose(c2[..., 1, 1], -c0[..., 1, 1], atol=1e-9)


def test_connected_chi_sg_of_free_spins_in_a_field_matches_its_closed_form():
    """J = 0, |H_i| = H0 with random directions: sites are independent, so chi_ij^{mu nu} = delta_ij C_i^{mu nu} and Eq. (9)
    gives chi_SG(k) = (1/N) sum_i ||C_i||_F^2 for EVERY k, with ||C||_F^2 = (1 - 2 L(a)/a - L(a)^2)^2 + 2 (L(a)/a)^2,
    a = beta H0 (longitudinal and two transverse variances of one spin in a field).  Four heat-bath replicas, Eq. (11)."""
    L, D, O, T, H0 = 4, 8, 4, 2, 1.5
    temps = np.array([0.8, 1.7], dtype=np.float32)
    N = L**3
    H = hsg_inputs.fixed_radius_field(L, D, H0, 5)
    sim = oracle.Oracle(L, D, O, temps, 77, precision=32, n_threads=4)
    sim.set_disorder(np.zeros((D, 3, L, L, L), np.float32), H); sim.init_spins()
    sim.sweep(0, 2)
    acc = []
    for _ in range(600):
        sim.sweep(0, 1)                                            # J = 0: every heat-bath sweep is an independent draw
        acc.append(sim.chi_field())
    acc = np.array(acc)                                            # [n][D][T][2][3][2]
    conn = (acc[..., 0, :] - 2 * acc[..., 1, :] + acc[..., 2, :]) / N      # Eq. (11) summand, [n][D][T][2][re/im]
    beta = (1.0 / temps.astype(np.float64)).astype(np.float32).astype(np.float64)
    a = beta * H0
    exact = (1 - 2 * langevin(a) / a - langevin(a)**2)**2 + 2 * (langevin(a) / a)**2
    est = conn.mean(axis=(0, 1))                                   # [T][2][2]: thermal and disorder average
    blocks = conn.reshape(30, -1, D, T, 2, 2).mean(axis=(1, 2))
    err = blocks.std(axis=0, ddof=1) / math.sqrt(30)
    for ik in range(2):
        assert (np.abs(est[:, ik, 0] - exact) < 4.5 * err[:, ik, 0] + 1e-6).all(), (est[:, ik, 0], exact, err[:, ik, 0])
        assert (np.abs(est[:, ik, 1]) < 4.5 * err[:, ik, 1] + 1e-6).all()
    # the disconnected parts alone are far from it: chi_1/N contains (sum_i m_i^2)^2 / N ~ N m^4
    assert (acc[..., 0, 0, 0].mean(axis=(0, 1)) / N > 1.25 * exact).all()


def test_xi_second_moment_is_eq8():
    # Ornstein-Zernike form chi(k) = chi0 / (1 + xi^2 khat^2), khat = 2 sin(k/2): Eq. (8) returns xi exactly
    for L in (4, 8, 32):
        for xi in (0.3, 2.0, 11.0):
            khat2 = (2 * math.sin(math.pi / L))**2
            assert abs(oracle.xi_second_moment(5.0, 5.0 / (1 + xi * xi * khat2), L) - xi) < 1e-12 * max(1, xi)
    assert oracle.xi_second_moment(2.0, 2.0, 8) == 0.0


# ---------------------------------------------------------------------- chirality, Eqs. (12)-(13)
def _kappa_np(s):
    """kappa^alpha = s_{i+alpha} . (s_i x s_{i-alpha}) with np.roll / np.cross; s[3][z][y][x] -> [3 alpha][z][y][x]."""
    out = []
    for ax in (3, 2, 1):                                   # alpha = x, y, z -> axes of s[c, z, y, x]
        p, m = np.roll(s, -1, axis=ax), np.roll(s, 1, axis=ax)
        out.append((p * np.cross(s, m, axis=0)).sum(axis=0))
    return np.array(out)


@pytest.mark.parametrize("precision,tol", [(64, 1e-15), (32, 6 * 2.0**-24)])
def test_chirality_and_chiral_overlap_brute_force(precision, tol):
    L, D, O, T = 4, 2, 3, 2
    sim = _sim(L, D, O, T, precision)
    S = hsg_inputs.unit_spins(L, D, O, T, 41)
    sim.set_spins(S)
    qc0, qck, kap = sim.measure_chiral(want_kappa=True)
    S64 = S.astype(np.float64)
    ref = np.array([[[_kappa_np(S64[d, o, t]) for t in range(T)] for o in range(O)] for d in range(D)])
    assert np.abs(kap - ref).max() <= tol
    assert np.abs(kap).max() > 0.5
    # the overlaps are formed from the oracle's own kappa (whatever its precision) in double
    x = np.arange(L)
    ph = np.exp(2j * np.pi * x / L)
    for p, (a, b) in enumerate([(0, 1), (0, 2), (1, 2)]):
        r0 = (kap[:, a] * kap[:, b]).mean(axis=(3, 4, 5))                           # [D][T][3]
        rk = (kap[:, a] * kap[:, b] * ph).mean(axis=(3, 4, 5))
        np.testing.assert_allclose(qc0[:, p], r0, atol=1e-15)
        np.testing.assert_allclose(qck[:, p, :, :, 0], rk.real, atol=1e-15)
        np.testing.assert_allclose(qck[:, p, :, :, 1], rk.imag, atol=1e-15)


def test_chirality_special_configurations():
    L, D, O, T = 8, 1, 2, 1
    sim = _sim(L, D, O, T, 64)
    x = np.arange(L)
    # collinear spins (any signs): kappa = 0
    S = np.zeros((D, O, T, 3, L, L, L)); S[:, :, :, 2] = np.where(np.random.default_rng(1).random((L, L, L)) < 0.5, -1.0, 1.0)
    sim.set_spins(S)
    qc0, qck, kap = sim.measure_chiral(want_kappa=True)
    assert np.abs(kap).max() == 0 and np.abs(qc0).max() == 0
    # coplanar spiral: three coplanar vectors have no volume
    th = 2 * np.pi * x / L
    S = np.zeros((D, O, T, 3, L, L, L)); S[:, :, :, 0] = np.cos(th); S[:, :, :, 1] = np.sin(th)
    sim.set_spins(S)
    assert np.abs(sim.measure_chiral(want_kappa=True)[2]).max() < 1e-15
    # conical spiral along x, s = (sin f cos(theta x), sin f sin(theta x), cos f): kappa^x = -2 sin(theta)(1 - cos(theta)) cos f sin^2 f
    # at every site; nothing changes along y, z: kappa^y = kappa^z = 0 (two equal vectors)
    f, theta = 0.9, 2 * np.pi * 3 / L
    S = np.zeros((D, O, T, 3, L, L, L))
    S[:, :, :, 0] = np.sin(f) * np.cos(theta * x); S[:, :, :, 1] = np.sin(f) * np.sin(theta * x); S[:, :, :, 2] = np.cos(f)
    sim.set_spins(S)
    qc0, qck, kap = sim.measure_chiral(want_kappa=True)
    k_exact = -2 * np.sin(theta) * (1 - np.cos(theta)) * np.cos(f) * np.sin(f)**2
    np.testing.assert_allclose(kap[0, 0, 0, 0], k_exact, atol=1e-15)
    assert np.abs(kap[0, 0, 0, 1:]).max() < 1e-15
    np.testing.assert_allclose(qc0[0, 0, 0], [k_exact**2, 0, 0], atol=1e-15)
    np.testing.assert_allclose(qck[0, 0, 0], 0, atol=1e-15)                     # uniform chirality: no k_min component
    # the opposite handedness (theta -> -theta) flips the sign of kappa
    S[:, 1, :, 1] *= -1                                                         # replica 2: mirror y -> left-handed
    sim.set_spins(S)
    np.testing.assert_allclose(sim.measure_chiral()[0][0, 0, 0], [-k_exact**2, 0, 0], atol=1e-15)
    # chirality wave: replica 1's handedness alternates with cos(2 pi x / L) -> visible at k_min only
    S = np.zeros((D, O, T, 3, L, L, L))
    S[:, :, :, 0] = np.sin(f) * np.cos(theta * x); S[:, :, :, 1] = np.sin(f) * np.sin(theta * x); S[:, :, :, 2] = np.cos(f)
    sim.set_spins(S)
    kap = sim.measure_chiral(want_kappa=True)[2]
    assert np.allclose(kap[0, 0], kap[0, 1])


def test_chiral_overlap_symmetries():
    L, D, O, T = 4, 1, 2, 2
    sim = _sim(L, D, O, T, 64)
    S = hsg_inputs.unit_spins(L, D, O, T, 43).astype(np.float64)
    sim.set_spins(S); q0, qk = sim.measure_chiral()
    # inversion s -> -s of ONE replica: kappa is odd (three factors), q_c changes sign
    S1 = S.copy(); S1[:, 1] *= -1
    sim.set_spins(S1); a0, ak = sim.measure_chiral()
    np.testing.assert_allclose(a0, -q0, atol=1e-15); np.testing.assert_allclose(ak, -qk, atol=1e-15)
    # inversion of BOTH: unchanged; improper rotation (mirror) of one replica: sign flip; proper rotations: invariant
    sim.set_spins(-S); b0, _ = sim.measure_chiral()
    np.testing.assert_allclose(b0, q0, atol=1e-15)
    S2 = S.copy(); S2[:, 1] = np.einsum("ab,dtbzyx->dtazyx", _rot(), S[:, 1])
    sim.set_spins(S2); c0, ck = sim.measure_chiral()
    np.testing.assert_allclose(c0, q0, atol=1e-13); np.testing.assert_allclose(ck, qk, atol=1e-13)
    S3 = S.copy(); S3[:, 1, :, 0] *= -1                                         # mirror x of replica 2
    sim.set_spins(S3); d0, _ = sim.measure_chiral()
    np.testing.assert_allclose(d0, -q0, atol=1e-15)
    # identical replicas: q_c(0) = mean kappa^2 >= 0
    S4 = S.copy(); S4[:, 1] = S[:, 0]
    sim.set_spins(S4); e0, _, kap = sim.measure_chiral(want_kappa=True)
    np.testing.assert_allclose(e0[0, 0], (kap[0, 0]**2).mean(axis=(2, 3, 4)), atol=1e-15)
