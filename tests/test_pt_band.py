"""CPU check of tests/pt_band.py (the excuse clause the GPU lockstep tests use)."""
import numpy as np
import pytest

from tests import philox_np as pnp
from tests.pt_band import excuse_or_fail


def test_band_excuse_is_exact():
    """The excuse clause itself: a flipped decision far from the threshold must fail, one inside the band must pass."""
    beta = np.array([10.0, 8.0, 6.0])
    seed, k_pt, O = 5, 7, 1
    u0 = float(pnp.u01(pnp.draw(pnp.DOMAIN_PT, 0, k_pt, 0, seed)[0]))
    # pair 0: x = dbeta * dE = ln u + 5e-5  (inside the band, x < 0); oracle rejects? ln u < x -> accept
    dE = (np.log(u0) + 5e-5) / (beta[1] - beta[0])
    E_pre = np.array([[[0.0, dE, dE]]])
    acc_o = np.array([[[1, 1]]]); acc_g = np.array([[[0, 1]]])
    excuse_or_fail(acc_g, acc_o, E_pre, beta, seed, k_pt, O)
    E_far = np.array([[[0.0, (np.log(u0) + 5e-3) / (beta[1] - beta[0]), 0.0]]])
    with pytest.raises(AssertionError):
        excuse_or_fail(acc_g, acc_o, E_far, beta, seed, k_pt, O)
    # a mismatch at the SECOND pair is judged with the energies after the first exchange
    u1 = float(pnp.u01(pnp.draw(pnp.DOMAIN_PT, 1, k_pt, 0, seed)[0]))
    e2 = 1.0 + (np.log(u1) - 3e-5) / (beta[2] - beta[1])           # after the accepted swap of pair 0 the walker carries E = 1.0
    E_pre2 = np.array([[[1.0, 0.5, e2]]])                          # pair 0: x = (8-10)(0.5-1.0) = 1 >= 0 -> accepted
    excuse_or_fail(np.array([[[1, 1]]]), np.array([[[1, 0]]]), E_pre2, beta, seed, k_pt, O)
