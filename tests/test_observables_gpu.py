"""GPU parity of the SURVEY §8(f) observables through the C ABI against the oracle, element by element on the same seeded
inputs: field-case susceptibility summands chi_1..3, chiral overlaps, Eq. (8)."""
import numpy as np
import pytest

import hsg_inputs
import oracle

pytestmark = pytest.mark.gpu


def _pair(L, D, O, T, seed, h_r=0.1, sample_offset=0):
    import paper_1204_6192_b200 as hsg
    # a warm, closely spaced ladder (spacing ~ 1/L^1.5 keeps dbeta*dE = O(1)): parallel tempering scrambles the slots quickly
    temps = (0.6 * (1.0 + 0.08 / L ** 1.5 * np.arange(T))).astype(np.float32)
    J = hsg_inputs.couplings(L, D, seed, sample_offset)
    H = hsg_inputs.gaussian_field(L, D, h_r, seed, sample_offset) if h_r > 0 else None
    eng = hsg.hsg_create(L, D, O, temps, seed, sample_offset=sample_offset)
    orc = oracle.Oracle(L, D, O, temps, seed, precision=32, sample_offset=sample_offset, n_threads=8)
    for s in (eng, orc):
        s.set_disorder(J, H); s.init_spins()
    n_acc = 0
    for _ in range(4):
        eng.sweep(1, 1); orc.sweep(1, 1)
        acc = orc.pt_swap()
        assert np.array_equal(eng.pt_swap().cpu().numpy(), acc)
        n_acc += int(acc.sum())
    assert n_acc > 0 or T == 1                                   # the observables must follow the temperature labels
    return eng, orc


@pytest.mark.parametrize("L,D,O,T,plain", [(4, 2, 4, 3, True), (6, 1, 4, 2, True), (8, 2, 5, 4, True), (16, 2, 4, 3, False),
                                           (32, 1, 4, 2, False), (64, 1, 4, 1, False)])
def test_field_case_chi_matches_oracle(L, D, O, T, plain):
    """chi_1, chi_2, chi_3 of Eq. (10) at k = 0 and k_min: against the O(N^2) definition on the small lattices and against
    the oracle's factored form (pinned to the definition in tests/test_oracle_field_chiral.py) on the large ones."""
    eng, orc = _pair(L, D, O, T, seed=51 + L)
    chi = eng.measure_field().cpu().numpy()
    ref = orc.chi_field(plain=plain)
    N = L ** 3
    np.testing.assert_allclose(chi, ref, rtol=1e-11, atol=1e-13 * N * N)
    if not plain and L <= 16:
        np.testing.assert_allclose(chi, orc.chi_field(plain=True), rtol=1e-11, atol=1e-13 * N * N)
    assert np.abs(chi[..., 0, 0]).min() > 0 and (chi[..., 1:, 1] != 0).any()


def test_field_case_needs_four_replicas():
    import paper_1204_6192_b200 as hsg
    eng, _ = _pair(4, 1, 3, 2, seed=3)
    with pytest.raises(hsg.HsgError) as ei:
        eng.measure_field()
    assert ei.value.code == hsg.HSG_EUNSUPPORTED


@pytest.mark.parametrize("L,D,O,T", [(4, 2, 2, 3), (6, 1, 3, 2), (8, 2, 2, 4), (10, 1, 2, 2), (16, 2, 3, 3), (32, 1, 2, 4), (64, 1, 2, 1)])
def test_chiral_overlaps_match_oracle(L, D, O, T):
    """q_c^alpha(0), q_c^alpha(k_min) of Eq. (13): the local chiralities are single-precision with a fixed operation order on
    both sides (bit-identical), products and sums fp64 -> only the summation order differs."""
    eng, orc = _pair(L, D, O, T, seed=71 + L)
    qc0, qck = (x.cpu().numpy() for x in eng.measure_chiral())
    r0, rk = orc.measure_chiral()
    np.testing.assert_allclose(qc0, r0, rtol=0, atol=1e-14)
    np.testing.assert_allclose(qck, rk, rtol=0, atol=1e-14)
    assert np.abs(r0).max() > 1e-4
    # either output alone
    only0, none = eng.measure_chiral(out=(eng._new(qc0.shape, eng.torch.float64), None))
    assert none is None and np.array_equal(only0.cpu().numpy(), qc0)


def test_chiral_conical_spiral_closed_form_on_the_gpu():
    """kappa^x = -2 sin(theta)(1 - cos(theta)) cos(f) sin^2(f) for a conical spiral along x (tests/test_oracle_field_chiral.py)."""
    import paper_1204_6192_b200 as hsg
    L, f, m = 16, 0.9, 3
    theta = 2 * np.pi * m / L
    x = np.arange(L)
    S = np.zeros((1, 2, 1, 3, L, L, L), dtype=np.float32)
    S[:, :, :, 0] = np.sin(f) * np.cos(theta * x); S[:, :, :, 1] = np.sin(f) * np.sin(theta * x); S[:, :, :, 2] = np.cos(f)
    S[:, 1, :, 1] *= -1                                           # replica 2 left-handed
    eng = hsg.hsg_create(L, 1, 2, [0.5], 1)
    eng.set_spins(S)
    qc0, qck = (t.cpu().numpy() for t in eng.measure_chiral())
    k = -2 * np.sin(theta) * (1 - np.cos(theta)) * np.cos(f) * np.sin(f) ** 2
    np.testing.assert_allclose(qc0[0, 0, 0], [-k * k, 0, 0], atol=1e-7)
    np.testing.assert_allclose(qck[0, 0, 0], 0, atol=1e-7)


def test_xi_second_moment_matches_oracle():
    import paper_1204_6192_b200 as hsg
    for L, c0, ck in ((8, 3.0, 1.2), (32, 900.0, 14.5), (64, 2.0, 2.0)):
        assert hsg.hsg_xi_second_moment(c0, ck, L) == pytest.approx(oracle.xi_second_moment(c0, ck, L), rel=1e-15)
    with pytest.raises(hsg.HsgError):
        hsg.hsg_xi_second_moment(1.0, 2.0, 8)


def test_overlap_of_a_lattice_wider_than_a_block():
    """L = 258 (Lh = 129: odd, so one site per item and 2*129 items per row lane > 256 threads): the overlap, field and
    chiral reductions must take their items in several passes (q came back as zeros)."""
    import paper_1204_6192_b200 as hsg
    import torch
    L = 258
    eng = hsg.hsg_create(L, 1, 2, [0.5], 9)
    eng.set_disorder(torch.zeros((1, 3, L, L, L), dtype=torch.float32, device="cuda"), None)
    eng.init_spins()
    _, M, q0, qk = eng.measure(out=(None, eng._new((1, 2, 1, 3), torch.float64), eng._new((1, 1, 1, 3, 3), torch.float64),
                                    eng._new((1, 1, 1, 3, 3, 2), torch.float64)))
    S = eng.get_spins().to(torch.float64)
    ref = torch.einsum("mzyx,nzyx->mn", S[0, 0, 0], S[0, 1, 0]) / L ** 3
    np.testing.assert_allclose(q0[0, 0, 0].cpu().numpy(), ref.cpu().numpy(), atol=1e-12)
    ph = torch.exp(2j * torch.pi * torch.arange(L, device=S.device, dtype=torch.float64) / L)
    refk = torch.einsum("mzyx,nzyx,x->mn", S[0, 0, 0].to(torch.complex128), S[0, 1, 0].to(torch.complex128), ph) / L ** 3
    np.testing.assert_allclose(qk[0, 0, 0, :, :, 0].cpu().numpy(), refk.real.cpu().numpy(), atol=1e-12)
    np.testing.assert_allclose(qk[0, 0, 0, :, :, 1].cpu().numpy(), refk.imag.cpu().numpy(), atol=1e-12)
    assert float(q0.abs().max()) > 0


def test_descriptor_limits_and_device_check():
    import paper_1204_6192_b200 as hsg
    import torch
    temps = hsg_inputs.geometric_ladder(0.1, 0.3, 4)
    with pytest.raises(hsg.HsgError):
        hsg.hsg_query_bytes(8, 2, 2, temps, sample_offset=2 ** 32 // 8 - 1)      # (offset + D) * O * T reaches 2^32
    hsg.hsg_query_bytes(8, 2, 2, temps, sample_offset=2 ** 32 // 8 - 3)
    if torch.cuda.device_count() < 2:
        pytest.skip("one device: the two-device part needs two")
    engs = []
    for dev in (0, 1):
        e = hsg.hsg_create(32, 1, 2, temps, 5, device=f"cuda:{dev}")
        e.set_disorder(hsg_inputs.couplings(32, 1, 5), None); e.init_spins(); e.sweep(2, 1)
        engs.append(e)
    a, b = (e.get_spins().cpu().numpy() for e in engs)
    assert np.array_equal(a, b)
    with torch.cuda.device(1):                                   # the raw C call on the wrong device is refused
        assert hsg.lib().hsg_sweep(engs[0]._h, 1, 0) == hsg.HSG_ESTATE
