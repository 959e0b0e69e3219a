"""Pins for the oracle's sweeps, energy and parallel tempering against closed forms and quadrature
(BASELINE.json north_star: OR conserves energy, Langevin law, E=0 at beta=0, two- and four-spin
clusters against integrated partition functions; SURVEY.md §8(c) pins).  CPU only."""
import math

import numpy as np
import pytest
from scipy import special

import hsg_inputs
import oracle
from tests import philox_np as pnp


def langevin(a):
    return 1.0 / np.tanh(a) - 1.0 / a


# ---------------------------------------------------------------------- energy: independent restatements
def energy_roll(S, J, H):
    """E = -sum_<ij> J_ij s_i.s_j - sum_i H_i.s_i with np.roll (forward bonds once). S[3,z,y,x], J[3,z,y,x]."""
    E = 0.0
    for d, ax in enumerate((3, 2, 1)):          # dir x,y,z  -> array axes of S[c,z,y,x]
        E -= (J[d] * (S * np.roll(S, -1, axis=ax)).sum(axis=0)).sum()
    if H is not None:
        E -= (H * S).sum()
    return E


def local_field_roll(S, J, H):
    h = np.zeros_like(S) if H is None else H.astype(np.float64).copy()
    for d, ax in enumerate((3, 2, 1)):
        h += J[d][None] * np.roll(S, -1, axis=ax)                       # bond i -> i+e
        h += np.roll(J[d], 1, axis=ax - 1)[None] * np.roll(S, 1, axis=ax)  # bond (i-e) -> i
    return h


def energy_bound(N, J=None, H=None):
    """|E_fp32form - E_plain| bound of DESIGN.md §3.6: each colour-1 site term carries at most 9 roundings of 2^-24
    relative to sum|J||s||s| + |H||s| <~ 8 (colour-0 terms: 3 roundings of |H|), i.e. N/2 * 9 * 2^-24 * 8."""
    return N / 2 * 9 * 2.0**-24 * 8


def test_energy_plain_is_eq1_and_matches_three_algebraically_equal_forms():
    """oracle.energy_plain = PAPER.md:26 Eq. (1) as written (forward bonds once, fp64): against three independent numpy
    restatements, in both instantiations (the fp32 one holds fp32 spins; the arithmetic of energy_plain is fp64 either way)."""
    L, D, O, T = 4, 2, 2, 3
    temps = hsg_inputs.geometric_ladder(0.1, 0.3, T)
    J = hsg_inputs.couplings(L, D, 5); H = hsg_inputs.gaussian_field(L, D, 0.3, 5)
    S = hsg_inputs.unit_spins(L, D, O, T, 5)
    par = np.indices((L, L, L)).sum(axis=0) % 2
    for precision in (64, 32):
        sim = oracle.Oracle(L, D, O, temps, 1, precision=precision)
        sim.set_disorder(J, H); sim.set_spins(S)
        Ep = sim.energy_plain()
        for d in range(D):
            for o in range(O):
                for t in range(T):
                    s = S[d, o, t].astype(np.float64); Jd = J[d].astype(np.float64); Hd = H[d].astype(np.float64)
                    e1 = energy_roll(s, Jd, Hd)
                    hJ = local_field_roll(s, Jd, None)
                    e2 = -0.5 * (s * hJ).sum() - (Hd * s).sum()
                    e3 = -((s * (hJ + Hd)).sum(axis=0) * (par == 1)).sum() - ((Hd * s).sum(axis=0) * (par == 0)).sum()
                    assert abs(Ep[d, o, t] - e1) < 1e-11 and abs(e1 - e2) < 1e-11 and abs(e1 - e3) < 1e-11
        # zero field path (H = None)
        sim.set_disorder(J, None)
        assert abs(sim.energy_plain()[0, 0, 0] - energy_roll(S[0, 0, 0].astype(np.float64), J[0].astype(np.float64), None)) < 1e-11


def test_energy_plain_brute_force_bond_list():
    """Every bond once: an explicit python loop over sites and the three forward neighbours (a dropped direction, a bond
    counted twice, a wrong periodic wrap or a transposed J index all fail here)."""
    L = 4
    J = hsg_inputs.couplings(L, 1, 6); H = hsg_inputs.gaussian_field(L, 1, 0.5, 6)
    S = hsg_inputs.unit_spins(L, 1, 1, 1, 6)
    sim = oracle.Oracle(L, 1, 1, [0.2], 1, precision=32)
    sim.set_disorder(J, H); sim.set_spins(S)
    s = S[0, 0, 0].astype(np.float64)
    E = 0.0
    for z in range(L):
        for y in range(L):
            for x in range(L):
                for d, (dx, dy, dz) in enumerate(((1, 0, 0), (0, 1, 0), (0, 0, 1))):
                    E -= float(J[0, d, z, y, x]) * float(s[:, z, y, x] @ s[:, (z + dz) % L, (y + dy) % L, (x + dx) % L])
                E -= float(H[0, :, z, y, x].astype(np.float64) @ s[:, z, y, x])
    assert abs(sim.energy_plain()[0, 0, 0] - E) < 1e-12
    # one ferromagnetic bond, aligned spins: E = -J
    J1 = np.zeros((1, 3, L, L, L), np.float32); J1[0, 1, 2, 3, 1] = 1.5      # y-bond leaving (x=1,y=3,z=2): wraps to y=0
    S1 = np.zeros((1, 1, 1, 3, L, L, L), np.float32); S1[0, 0, 0, 2] = 1.0
    sim.set_disorder(J1, None); sim.set_spins(S1)
    assert sim.energy_plain()[0, 0, 0] == -1.5 and sim.energy()[0, 0, 0] == -1.5
    S1[0, 0, 0, 2, 2, 0, 1] = -1.0                                             # flip the far end of that bond
    sim.set_spins(S1)
    assert sim.energy_plain()[0, 0, 0] == 1.5 and sim.energy()[0, 0, 0] == 1.5


@pytest.mark.parametrize("L", [4, 8, 12])
def test_energy_of_the_moves_reading_is_pinned_against_energy_plain(L):
    """oracle.energy (PAPER.md:185 reading: single-precision site terms s_i.h_i / s_i.H_i in the bipartite
    form, fp64 sum — what the parallel-tempering decisions use) against the plain definition: the fp64 instantiation agrees to
    summation-order rounding, the fp32 one inside the derived bound N/2 * 9 * 2^-24 * 8 (and is typically sqrt(N) smaller)."""
    D, O, T = 2, 2, 2
    temps = hsg_inputs.geometric_ladder(0.1, 0.3, T)
    J = hsg_inputs.couplings(L, D, 5 + L); H = hsg_inputs.gaussian_field(L, D, 0.3, 5 + L)
    S = hsg_inputs.unit_spins(L, D, O, T, 5 + L)
    N = L**3
    sim = oracle.Oracle(L, D, O, temps, 1, precision=64)
    sim.set_disorder(J, H); sim.set_spins(S)
    assert np.abs(sim.energy() - sim.energy_plain()).max() < 1e-13 * N
    sim32 = oracle.Oracle(L, D, O, temps, 1, precision=32)
    sim32.set_disorder(J, H); sim32.set_spins(S)
    E32, Ep = sim32.energy(), sim32.energy_plain()
    assert np.abs(Ep - sim.energy_plain()).max() == 0                          # same fp32 spins, same fp64 arithmetic
    assert np.abs(E32 - Ep).max() < energy_bound(N)
    assert np.abs(E32 - Ep).max() < 40 * math.sqrt(N) * 2.0**-24 * 8           # random-walk size, with margin
    assert np.abs(E32 - Ep).max() > 0                                          # it IS the single-precision form


# ---------------------------------------------------------------------- OR sweeps are microcanonical
@pytest.mark.parametrize("precision,n_sweeps,tol_e,tol_n", [(64, 100, 1e-12, 1e-12), (32, 100, 3e-5, 3e-5)])
def test_or_sweeps_conserve_energy_and_norm(precision, n_sweeps, tol_e, tol_n):
    L, D, O, T = 6, 1, 1, 2
    temps = [0.1, 0.2]
    sim = oracle.Oracle(L, D, O, temps, 3, precision=precision)
    sim.set_disorder(hsg_inputs.couplings(L, D, 8), hsg_inputs.gaussian_field(L, D, 0.1, 8))
    sim.init_spins()
    E0 = sim.energy()
    S0 = sim.get_spins()
    sim.sweep(n_sweeps, 0)
    E1 = sim.energy(); S1 = sim.get_spins()
    assert np.abs((E1 - E0) / E0).max() < tol_e * max(1, abs(L**3 / E0).max())
    assert np.abs((S1**2).sum(axis=3) - 1).max() < tol_n
    assert np.abs(S1 - S0).max() > 0.5          # and it actually moved
    _, cnt = sim.get_state()
    assert cnt[0] == 0                           # OR consumes no random numbers / HB counter


def test_one_or_sweep_equals_vectorised_two_colour_update():
    """Brute force: colour 0 from the old odd spins, then colour 1 from the new even spins."""
    L = 4
    J = hsg_inputs.couplings(L, 1, 21); H = hsg_inputs.gaussian_field(L, 1, 0.2, 21)
    S = hsg_inputs.unit_spins(L, 1, 1, 1, 21)
    sim = oracle.Oracle(L, 1, 1, [0.2], 1, precision=64)
    sim.set_disorder(J, H); sim.set_spins(S); sim.sweep(1, 0)
    got = sim.get_spins()[0, 0, 0]
    s = S[0, 0, 0].astype(np.float64); Jd = J[0].astype(np.float64); Hd = H[0].astype(np.float64)
    par = np.indices((L, L, L)).sum(axis=0) % 2
    for colour in (0, 1):
        h = local_field_roll(s, Jd, Hd)
        new = 2 * (s * h).sum(axis=0) / (h * h).sum(axis=0) * h - s
        s = np.where(par == colour, new, s)
    np.testing.assert_allclose(got, s, atol=1e-13)


# ---------------------------------------------------------------------- beta = 0
def test_energy_vanishes_at_infinite_temperature():
    L, D, O, T = 8, 2, 2, 2
    sim = oracle.Oracle(L, D, O, [1e29, 1e30], 17, precision=32)
    J = hsg_inputs.couplings(L, D, 9); H = hsg_inputs.gaussian_field(L, D, 0.1, 9)
    sim.set_disorder(J, H); sim.init_spins()
    es = []
    for _ in range(40):
        sim.sweep(0, 1)
        es.append(sim.energy())
    es = np.array(es)                                   # [40, D, O, T] independent configurations
    # Var(E) = sum_bonds J^2 <(s.s')^2> + sum_i |H_i|^2 <cos^2> = (sum J^2 + sum H^2)/3
    sigma = np.sqrt(((J.astype(np.float64)**2).sum(axis=(1, 2, 3, 4)) + (H.astype(np.float64)**2).sum(axis=(1, 2, 3, 4))) / 3)
    mean = es.mean(axis=0)
    n = es.shape[0]
    assert (np.abs(mean) < 4.5 * sigma[:, None, None] / math.sqrt(n)).all()
    # and the fluctuations have the predicted size
    ratio = es.std(axis=0) / sigma[:, None, None]
    assert (ratio > 0.6).all() and (ratio < 1.5).all()


# ---------------------------------------------------------------------- two-spin clusters
def _dimer_lattice(L, J0):
    """All couplings zero except the x-bonds leaving even-x sites: N/2 independent dimers of coupling J0."""
    J = np.zeros((1, 3, L, L, L), dtype=np.float32)
    J[0, 0, :, :, 0::2] = J0
    return J


@pytest.mark.parametrize("J0,T", [(1.0, 0.5), (-0.7, 0.2)])
def test_dimers_zero_field_closed_form(J0, T):
    """<s1.s2> = L(beta J0) for two spins coupled by J0 (integrate one spin out)."""
    L = 6
    sim = oracle.Oracle(L, 1, 1, [T], 23, precision=32)
    sim.set_disorder(_dimer_lattice(L, J0), None); sim.init_spins()
    sim.sweep(0, 20)
    acc = []
    for _ in range(1500):
        sim.sweep(0, 1)
        S = sim.get_spins()[0, 0, 0]
        acc.append((S[:, :, :, 0::2] * S[:, :, :, 1::2]).sum(axis=0).mean())
    acc = np.array(acc)
    beta = float(np.float32(1.0 / np.float64(np.float32(T))))
    exact = langevin(beta * float(np.float32(J0)))
    # successive sweeps are correlated: estimate the error from blocks
    blocks = acc.reshape(30, -1).mean(axis=1)
    err = blocks.std(ddof=1) / math.sqrt(len(blocks))
    assert abs(acc.mean() - exact) < 4.5 * err + 1e-5
    # the energy routine sees the same number: E = -J0 * sum over dimers of s1.s2 (plain Eq. 1 form: fp64 products)
    S = sim.get_spins()[0, 0, 0]
    e_dimers = -float(np.float32(J0)) * (S[:, :, :, 0::2] * S[:, :, :, 1::2]).sum()
    assert abs(sim.energy_plain()[0, 0, 0] - e_dimers) < 1e-9
    assert abs(sim.energy()[0, 0, 0] - e_dimers) < energy_bound(L**3)          # the single-precision reading, inside its bound


def _dimer_in_field_exact(beta, J0, h1, h2):
    """<E> of two spins, H = -J0 s1.s2 - h1.s1 - h2.s2: spin 2 integrated analytically,
    spin 1 by Gauss-Legendre (cos theta) x trapezoid (phi) quadrature of Z and dZ/dbeta."""
    x, w = np.polynomial.legendre.leggauss(96)
    phi = np.linspace(0, 2 * np.pi, 128, endpoint=False)
    ct, ph = np.meshgrid(x, phi, indexing="ij")
    st = np.sqrt(1 - ct**2)
    s1 = np.stack([st * np.cos(ph), st * np.sin(ph), ct])
    A = np.linalg.norm(J0 * s1 + np.asarray(h2)[:, None, None], axis=0)
    b1 = np.tensordot(np.asarray(h1), s1, axes=1)
    inner = np.sinh(beta * A) / (beta * A)                 # (1/4pi) int ds2 exp(beta A.s2)
    dinner = np.cosh(beta * A) / beta - np.sinh(beta * A) / (beta**2 * A)
    wgt = w[:, None] * (2 * np.pi / len(phi))
    Z = (wgt * np.exp(beta * b1) * inner).sum()
    dZ = (wgt * np.exp(beta * b1) * (b1 * inner + dinner)).sum()
    return -dZ / Z


def test_dimers_in_a_field_match_integrated_partition_function():
    L, J0, T = 6, 0.9, 0.4
    h1, h2 = np.array([0.3, -0.2, 0.5]), np.array([-0.4, 0.1, 0.25])
    H = np.zeros((1, 3, L, L, L), dtype=np.float32)
    H[0, :, :, :, 0::2] = h1[:, None, None, None]
    H[0, :, :, :, 1::2] = h2[:, None, None, None]
    sim = oracle.Oracle(L, 1, 1, [T], 29, precision=32)
    sim.set_disorder(_dimer_lattice(L, J0), H); sim.init_spins()
    sim.sweep(0, 20)
    es = []
    for _ in range(1500):
        sim.sweep(3, 1)                                   # OR sweeps in between must not change the law
        es.append(sim.energy()[0, 0, 0] / (L**3 / 2))
    es = np.array(es)
    beta = float(np.float32(1.0 / np.float64(np.float32(T))))
    exact = _dimer_in_field_exact(beta, float(np.float32(J0)), H[0, :, 0, 0, 0].astype(np.float64), H[0, :, 0, 0, 1].astype(np.float64))
    blocks = es.reshape(30, -1).mean(axis=1)
    err = blocks.std(ddof=1) / math.sqrt(len(blocks))
    assert abs(es.mean() - exact) < 4.5 * err + 1e-5


# ---------------------------------------------------------------------- four-spin clusters
def _bond_expectations_ring(K):
    """Classical Heisenberg ring, zero field: Z ~ sum_l (2l+1) prod_i i_l(K_i) (Legendre/transfer-matrix
    expansion, i_l = modified spherical Bessel).  <s_i.s_{i+1}> = d ln Z / d K_i."""
    K = np.asarray(K, dtype=np.float64)
    ls = np.arange(0, 60)
    lam = np.array([special.spherical_in(ls, k) for k in K])            # [bond, l]
    dlam = np.array([special.spherical_in(ls, k, derivative=True) for k in K])
    Z = ((2 * ls + 1) * lam.prod(axis=0)).sum()
    out = []
    for i in range(len(K)):
        others = np.delete(lam, i, axis=0).prod(axis=0)
        out.append(((2 * ls + 1) * dlam[i] * others).sum() / Z)
    return np.array(out)


@pytest.mark.parametrize("ring", [False, True])
def test_four_spin_chains_and_rings(ring):
    """L=4 lattice with only x-bonds: L^2 independent 4-chains (bond x=3->0 cut) or 4-rings (plaquette
    topology).  Open chain: <s_i.s_{i+1}> = L(beta J_i) (integrate from the free end); ring: series above."""
    L, T = 4, 0.35
    Jb = np.array([1.1, -0.8, 0.6, 0.0 if not ring else -1.3])
    J = np.zeros((1, 3, L, L, L), dtype=np.float32)
    for x in range(4):
        J[0, 0, :, :, x] = Jb[x]
    sim = oracle.Oracle(L, 1, 1, [T], 31 + ring, precision=32)
    sim.set_disorder(J, None); sim.init_spins()
    sim.sweep(0, 30)
    acc = []
    for _ in range(3000):
        sim.sweep(1, 1)
        S = sim.get_spins()[0, 0, 0]
        acc.append((S * np.roll(S, -1, axis=3)).sum(axis=0).mean(axis=(0, 1)))   # [x] bond x -> x+1
    acc = np.array(acc)
    beta = float(np.float32(1.0 / np.float64(np.float32(T))))
    K = beta * J[0, 0, 0, 0, :].astype(np.float64)
    # open chain: the end-to-end correlation <s_3.s_0> is the product of the three bond expectations
    exact = _bond_expectations_ring(K) if ring else np.append(langevin(K[:3]), langevin(K[:3]).prod())
    blocks = acc.reshape(30, -1, 4).mean(axis=1)
    err = blocks.std(axis=0, ddof=1) / math.sqrt(len(blocks))
    assert (np.abs(acc.mean(axis=0) - exact) < 4.5 * err + 1e-5).all(), (acc.mean(axis=0), exact)


def test_ring_series_reduces_to_open_chain_when_a_bond_is_cut():
    K = np.array([1.7, -2.2, 0.9, 1e-9])
    np.testing.assert_allclose(_bond_expectations_ring(K)[:3], langevin(K[:3]), atol=1e-8)


# ---------------------------------------------------------------------- parallel tempering, Eq. (4)
def test_pt_decisions_follow_eq4_with_the_documented_stream():
    """Recompute every decision outside the oracle: x = (beta_{t+1}-beta_t)(E_{t+1}-E_t), accept iff
    x >= 0 or ln u < x, pairs from the lowest temperature upwards, u from the PT Philox domain."""
    L, D, O, T, seed, off = 4, 3, 2, 6, 77, 2
    temps = hsg_inputs.geometric_ladder(0.5, 3.0, T)
    sim = oracle.Oracle(L, D, O, temps, seed, precision=32, sample_offset=off)
    sim.set_disorder(hsg_inputs.couplings(L, D, 13), hsg_inputs.gaussian_field(L, D, 0.1, 13))
    sim.init_spins()
    beta = (1.0 / temps.astype(np.float64)).astype(np.float32).astype(np.float64)
    perm = np.tile(np.arange(T), (D, O, 1))
    n_acc = 0
    for step in range(12):
        sim.sweep(1, 1)
        E = sim.energy()                       # by temperature index, before the swap pass
        acc = sim.pt_swap()
        for d in range(D):
            for o in range(O):
                e = E[d, o].copy()
                for t in range(T - 1):
                    w = pnp.draw(pnp.DOMAIN_PT, t, step, (off + d) * O + o, seed)
                    u = float(pnp.u01(w[0]))
                    x = (beta[t + 1] - beta[t]) * (e[t + 1] - e[t])
                    a = x >= 0 or math.log(u) < x
                    assert int(a) == acc[d, o, t]
                    if a:
                        e[[t, t + 1]] = e[[t + 1, t]]
                        perm[d, o, [t, t + 1]] = perm[d, o, [t + 1, t]]
                    n_acc += a
                np.testing.assert_allclose(sim.energy()[d, o], e, rtol=0, atol=1e-9)   # configurations moved with labels
        got, cnt = sim.get_state()
        np.testing.assert_array_equal(got, perm)
        assert cnt[1] == step + 1
        assert (np.sort(got, axis=2) == np.arange(T)).all()       # stays a permutation
    assert 0 < n_acc < 12 * D * O * (T - 1)                       # both outcomes occurred


def test_pt_keeps_every_temperature_canonical_free_spins_in_uniform_field():
    """J = 0, uniform field H0 z: exact <E>_t = -N H0 L(beta_t H0).  OR cannot equilibrate anything here and
    HB runs only every 3rd step, so the ladder stays canonical only if the swap rule (sign of Eq. 4
    included) is right.  A flipped sign is off by far more than the tolerance."""
    L, D, O, T, H0 = 4, 16, 1, 5, 1.0
    temps = hsg_inputs.geometric_ladder(0.4, 1.6, T)
    N = L**3
    J = np.zeros((D, 3, L, L, L), dtype=np.float32)
    H = np.zeros((D, 3, L, L, L), dtype=np.float32); H[:, 2] = H0
    sim = oracle.Oracle(L, D, O, temps, 41, precision=32)
    sim.set_disorder(J, H); sim.init_spins()
    for _ in range(30):
        sim.sweep(0, 1); sim.pt_swap()
    es, accs = [], []
    for step in range(900):
        sim.sweep(1, 1 if step % 3 == 0 else 0)
        accs.append(sim.pt_swap().mean())
        es.append(sim.energy().mean(axis=(0, 1)))
    es = np.array(es)
    beta = (1.0 / temps.astype(np.float64)).astype(np.float32).astype(np.float64)
    exact = -N * H0 * langevin(beta * H0)
    blocks = es.reshape(30, -1, T).mean(axis=1)
    err = blocks.std(axis=0, ddof=1) / math.sqrt(len(blocks))
    assert (np.abs(es.mean(axis=0) - exact) < 4.5 * err + 1e-3).all(), (es.mean(axis=0), exact, err)
    assert 0.05 < np.mean(accs) < 0.95
