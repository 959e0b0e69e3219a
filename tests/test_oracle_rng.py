"""Pins for the oracle's random stream: Philox4x32-10, the uniform mapping and the
counter packing.  CPU only."""
import os

import numpy as np

import oracle
from tests import philox_np as pnp

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


def _kat():
    rows = []
    for line in open(GOLDEN):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        w = [int(t, 16) for t in line.split()]
        rows.append((w[0:4], w[4:6], w[6:10]))
    return rows


def test_philox_known_answer_vectors():
    rows = _kat()
    assert len(rows) == 3
    for ctr, key, out in rows:
        assert list(oracle.philox4x32_10(ctr, key)) == out
        got = pnp.philox4x32_10(ctr[0], ctr[1], ctr[2], ctr[3], key[0], key[1])
        assert [int(g) for g in got] == out


def test_philox_oracle_vs_numpy_restatement():
    rng = np.random.default_rng(7)
    ctrs = rng.integers(0, 2**32, size=(2000, 4), dtype=np.uint64)
    key = rng.integers(0, 2**32, size=2, dtype=np.uint64)
    ref = np.stack(pnp.philox4x32_10(ctrs[:, 0], ctrs[:, 1], ctrs[:, 2], ctrs[:, 3], key[0], key[1]), axis=1)
    for i in range(0, 2000, 7):
        assert (oracle.philox4x32_10(ctrs[i], key) == ref[i]).all()


def test_uniform_mapping_is_exact_open_and_symmetric():
    L = oracle.lib()
    assert oracle.u01(0) == 2.0**-24
    assert oracle.u01(0xFFFFFFFF) == 1.0 - 2.0**-24
    assert oracle.u01(0x80000000) == 0.5 + 2.0**-24
    for w in (0, 1, 511, 512, 0x12345678, 0xFFFFFE00, 0xFFFFFFFF):
        u64 = oracle.u01(w)
        u32 = L.orc_u01_f32(w)
        assert u64 == ((w >> 9) + 0.5) / 2**23
        assert float(u32) == u64                       # exactly representable in binary32
        assert oracle.u01(w) + oracle.u01(w ^ 0xFFFFFFFF) == 1.0   # symmetric about 1/2


def test_init_spins_follow_the_documented_counter_packing():
    """init: c0 = site, c1 = 0, c2 = ((off+d)*O+o)*T+t, c3 = DOMAIN_INIT<<28; cos(theta)=2u1-1, phi=2 pi u2."""
    Lx, D, O, T, seed, off = 4, 2, 2, 3, 0x1234567_89ABCDEF, 5
    sim = oracle.Oracle(Lx, D, O, np.linspace(0.1, 0.3, T), seed, precision=64, sample_offset=off)
    sim.init_spins()
    S = sim.get_spins().reshape(D, O, T, 3, Lx**3)
    site = np.arange(Lx**3)
    for d in range(D):
        for o in range(O):
            for t in range(T):
                sysid = ((off + d) * O + o) * T + t
                w = pnp.draw(pnp.DOMAIN_INIT, site, 0, sysid, seed)
                u1, u2 = pnp.u01(w[0]), pnp.u01(w[1])
                ct = 2 * u1 - 1
                st = np.sqrt(1 - ct * ct)
                ref = np.stack([st * np.cos(2 * np.pi * u2), st * np.sin(2 * np.pi * u2), ct])
                np.testing.assert_allclose(S[d, o, t], ref, atol=1e-14)
    # and the result is uniform on the sphere: mean ~ 0, <s_c^2> ~ 1/3
    big = oracle.Oracle(8, 4, 2, np.linspace(0.1, 0.3, 4), 99, precision=32)
    big.init_spins()
    Sb = big.get_spins().reshape(-1, 3, 512).transpose(1, 0, 2).reshape(3, -1)
    n = Sb.shape[1]
    assert np.abs(Sb.mean(axis=1)).max() < 4 * np.sqrt(1 / 3 / n)
    assert np.abs((Sb**2).mean(axis=1) - 1 / 3).max() < 4 * np.sqrt(4 / 45 / n)
    np.testing.assert_allclose((Sb**2).sum(axis=0), 1.0, atol=3e-7)


def test_heat_bath_sweep_follows_the_documented_counter_packing():
    """HB: c1/c3 = sweep counter k_hb with DOMAIN_HB, c2 = ((off+d)*O+o)*T+t, and ONE Philox call per
    pair of same-colour sites x, x+2 with compact index j = x>>1 (even, odd): c0 = index of the even-j site, which takes
    words 0,1; its partner takes words 2,3.  Checked on a lattice without couplings, where the local field is H_i, so
    every new spin is hb_draw(H_i, beta_t, u1, u2) of exactly those two words — for two successive sweeps."""
    for Lx in (4, 6):                                   # Lh even and odd (unpaired last site of a row)
        D, O, T, seed, off = 2, 2, 2, 0xFEDCBA98_76543210, 3
        temps = np.array([0.5, 0.9], dtype=np.float32)
        N = Lx**3
        rng = np.random.default_rng(5)
        J = np.zeros((D, 3, Lx, Lx, Lx), dtype=np.float32)
        H = rng.standard_normal((D, 3, Lx, Lx, Lx)).astype(np.float32)
        sim = oracle.Oracle(Lx, D, O, temps, seed, precision=64, sample_offset=off)
        sim.set_disorder(J, H)
        sim.init_spins()
        site = np.arange(N)
        x = site % Lx
        odd = (x >> 1) & 1
        c0 = site - 2 * odd
        for k_hb in range(2):
            sim.sweep(0, 1)
            S = sim.get_spins().reshape(D, O, T, 3, N)
            for d in range(D):
                for o in range(O):
                    for t in range(T):
                        sysid = ((off + d) * O + o) * T + t
                        w = pnp.draw(pnp.DOMAIN_HB, c0, k_hb, sysid, seed)
                        u1 = np.where(odd == 1, pnp.u01(w[2]), pnp.u01(w[0]))
                        u2 = np.where(odd == 1, pnp.u01(w[3]), pnp.u01(w[1]))
                        beta = float(np.float32(1.0 / np.float64(temps[t])))
                        Hd = H[d].reshape(3, N).astype(np.float64)
                        for i in range(0, N, 7):        # a sample of the sites, every residue of x
                            ref = oracle.hb_draw(Hd[:, i], beta, u1[i], u2[i], precision=64)
                            np.testing.assert_allclose(S[d, o, t, :, i], ref, atol=1e-14)
        assert sim.get_state()[1][0] == 2
