"""Pins for the oracle's single-spin moves against what the paper and the
mathematics fix: OR is a norm- and energy-preserving involution, HB reproduces the
Langevin law of Eq. (2).  CPU only."""
import math

import numpy as np
import pytest
from scipy import stats

import oracle


def langevin(a):
    return 1.0 / math.tanh(a) - 1.0 / a if a > 1e-6 else a / 3.0


# ------------------------------------------------------------------ spec series vs libm
def _ulp32(x):
    return float(np.spacing(np.float32(abs(x))))


def test_spec_omexp_matches_libm():
    xs = np.concatenate([np.logspace(-4, 2.2, 4000), np.linspace(2e-4, 100, 4000), [0.3465, 0.3466, 0.34657359]]).astype(np.float32)
    for x in xs:
        ref = -math.expm1(-float(x))
        assert abs(oracle.spec_omexp_f32(x) - ref) <= 2.0 * _ulp32(ref), x


def test_spec_log1m_matches_libm():
    ys = np.concatenate([np.logspace(-7.2, 0, 4000), np.linspace(1e-7, 1 - 2.0**-24, 4000), [0.25, 0.24999999, 1 / 3, 0.5]]).astype(np.float32)
    for y in ys:
        if y >= 1:
            continue
        ref = math.log1p(-float(y))
        assert abs(oracle.spec_log1m_f32(y) - ref) <= 4.0 * _ulp32(ref), y


def test_spec_sincos2pi_matches_libm():
    us = np.concatenate([np.linspace(2.0**-24, 1 - 2.0**-24, 8001), [0.125, 0.375, 0.625, 0.875, 0.25, 0.5, 0.75]]).astype(np.float32)
    for u in us:
        s, c = oracle.spec_sincos2pi_f32(u)
        assert abs(s - math.sin(2 * math.pi * float(u))) < 1.5e-7
        assert abs(c - math.cos(2 * math.pi * float(u))) < 1.5e-7
        assert abs(s * s + c * c - 1) < 4e-7


# ------------------------------------------------------------------ over-relaxation, Eq. (3)
@pytest.mark.parametrize("precision,tol", [(64, 1e-14), (32, 1e-6)])
def test_or_reflection_is_an_involution_preserving_norm_and_energy(precision, tol):
    rng = np.random.default_rng(3)
    for _ in range(200):
        s = rng.standard_normal(3); s /= np.linalg.norm(s)
        h = rng.standard_normal(3) * rng.uniform(0.01, 5)
        s1 = oracle.or_reflect(s, h, precision).astype(np.float64)
        sq = np.asarray(s, dtype=np.float32 if precision == 32 else np.float64).astype(np.float64)
        hq = np.asarray(h, dtype=np.float32 if precision == 32 else np.float64).astype(np.float64)
        assert abs(np.linalg.norm(s1) - 1) < tol                         # unit length kept
        assert abs(s1 @ hq - sq @ hq) < tol * max(1, np.linalg.norm(hq))  # s.h (the energy) kept
        # mirror image: component along h kept, perpendicular part flipped
        hh = hq / np.linalg.norm(hq)
        np.testing.assert_allclose(s1 - (s1 @ hh) * hh, -(sq - (sq @ hh) * hh), atol=tol)
        s2 = oracle.or_reflect(s1, h, precision).astype(np.float64)      # reflecting twice = identity
        np.testing.assert_allclose(s2, sq, atol=2 * tol)
    # zero field: identity
    np.testing.assert_array_equal(oracle.or_reflect([0.6, 0.0, 0.8], [0, 0, 0], 64), [0.6, 0.0, 0.8])


# ------------------------------------------------------------------ heat bath, Eq. (2)
@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("a", [0.0, 1e-5, 0.5, 1.0, 5.0, 20.0, 40.0, 150.0])
def test_hb_reproduces_langevin_law(precision, a):
    """<cos> = coth a - 1/a, <cos^2> = 1 - 2 L(a)/a, azimuth uniform; KS test against the exact CDF."""
    n = 200_000
    h = np.array([0.3, -1.2, 0.7]); hn = np.linalg.norm(h)
    beta = a / hn
    S = oracle.hb_sample(h, beta, seed=1000 + int(a * 10), n=n, precision=precision)
    np.testing.assert_allclose((S**2).sum(axis=1), 1.0, atol=1e-12 if precision == 64 else 5e-7)
    nh = h / hn
    c = S @ nh
    La = langevin(a)
    m2 = 1 - 2 * La / a if a > 1e-3 else 1 / 3
    var_c = m2 - La**2
    assert abs(c.mean() - La) < 4.5 * math.sqrt(var_c / n) + 1e-7
    # <cos^2>: variance of c^2 bounded by <c^4> <= 1
    assert abs((c**2).mean() - m2) < 4.5 * math.sqrt(max((c**4).mean() - m2**2, 1e-12) / n) + 1e-7
    # perpendicular part: zero mean, azimuth uniform
    perp = S - np.outer(c, nh)
    assert np.abs(perp.mean(axis=0)).max() < 4.5 * math.sqrt((1 - m2) / 2 / n) + 1e-7
    e1 = np.cross(nh, [1.0, 0, 0]); e1 /= np.linalg.norm(e1); e2 = np.cross(nh, e1)
    phi = np.arctan2(perp @ e2, perp @ e1)
    assert abs(np.cos(2 * phi).mean()) < 4.5 * math.sqrt(0.5 / n)
    assert abs(np.sin(2 * phi).mean()) < 4.5 * math.sqrt(0.5 / n)
    # distribution of cos(theta): CDF F(c) = (e^{a c} - e^{-a}) / (e^{a} - e^{-a})
    if a > 1e-3:
        cdf = lambda x: np.expm1(a * (np.clip(x, -1, 1) + 1)) / math.expm1(2 * a) if a < 300 else None
    else:
        cdf = lambda x: (np.clip(x, -1, 1) + 1) / 2
    assert stats.kstest(c, cdf).pvalue > 1e-3


@pytest.mark.parametrize("precision,tol", [(64, 1e-12), (32, 3e-6)])
def test_hb_map_is_the_inverse_cdf_and_frame_is_orthonormal(precision, tol):
    """s'.n = cos(theta) with cos(theta) = 1 + ln(u1 + (1-u1) e^{-2a})/a; the azimuthal part has length
    sin(theta) and turns by 90 degrees when u2 advances by 1/4 (right-handed orthonormal frame)."""
    rng = np.random.default_rng(11)
    for _ in range(300):
        h = rng.standard_normal(3) * rng.uniform(0.05, 4)
        if rng.uniform() < 0.2:
            h[2] = -abs(h[2]) * 5           # exercise the sigma = -1 branch, n_z close to -1
        beta = rng.uniform(0.5, 17)
        u1 = (rng.integers(0, 2**23) + 0.5) / 2**23
        u2 = (rng.integers(0, 2**21) + 0.5) / 2**23      # < 1/4 so that u2 + 1/4 stays in (0,1)
        hq = np.asarray(h, dtype=np.float32 if precision == 32 else np.float64).astype(np.float64)
        bq = float(np.float32(beta)) if precision == 32 else beta
        hn = np.linalg.norm(hq); n = hq / hn; a = bq * hn
        s = oracle.hb_draw(h, beta, u1, u2, precision).astype(np.float64)
        s90 = oracle.hb_draw(h, beta, u1, u2 + 0.25, precision).astype(np.float64)
        ct = 1 + math.log(u1 + (1 - u1) * math.exp(-2 * a)) / a
        assert abs(s @ n - ct) < tol * max(1.0, 1.0 / a)
        assert abs(np.linalg.norm(s) - 1) < tol
        p, p90 = s - (s @ n) * n, s90 - (s90 @ n) * n
        assert abs(p @ p90) < 10 * tol                       # perpendicular azimuthal directions
        np.testing.assert_allclose(np.cross(p, p90), (p @ p) * n, atol=10 * tol)  # right-handed about n


def test_hb_zero_field_is_uniform_about_z():
    S = oracle.hb_sample([0.0, 0.0, 0.0], 7.0, seed=5, n=100_000, precision=32)
    assert np.abs(S.mean(axis=0)).max() < 4.5 * math.sqrt(1 / 3 / 100_000)
    np.testing.assert_allclose((S**2).sum(axis=1), 1.0, atol=5e-7)
