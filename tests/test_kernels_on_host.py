"""The plain kernels of the library (paper_1204_6192_b200/csrc/hsg_kernels.cuh, hsg_observables.cuh: layout conversion, start
spins, the generic sweep kernel, energy / magnetisation / overlap reductions, parallel tempering with its diagnostics, the
field-case and chiral reductions) executed on the HOST with the launch shapes the library uses (csrc/hsg_shapes.h), and
compared with the oracle.  No GPU.  Companion of tests/test_zmarch_on_host.py (the fused sweep kernel); the execution model is
tests/host_emul/emu.h.  What this cannot see is the same as there: the hardware itself."""
import ctypes as C
import hashlib
import shutil
import subprocess
from pathlib import Path

import numpy as np
import pytest

import hsg_inputs
import oracle
from tests.test_device_math_on_host import fast_math_bound

ROOT = Path(__file__).resolve().parent.parent
CSRC = ROOT / "paper_1204_6192_b200" / "csrc"
HERE = Path(__file__).resolve().parent
SOURCES = [CSRC / "hsg_kernels.cuh", CSRC / "hsg_observables.cuh", CSRC / "hsg_shapes.h", CSRC / "hsg_layout.cuh", CSRC / "hsg_math.cuh",
           HERE / "host_math" / "cuda_runtime.h", HERE / "host_math" / "hsg_prim.cuh",
           HERE / "host_emul" / "emu.h", HERE / "host_emul" / "cuda_builtins.h", HERE / "host_emul" / "kernels_driver.cpp"]


@pytest.fixture(scope="module")
def lib(tmp_path_factory):
    tag = hashlib.sha1(b"".join(p.read_bytes() for p in SOURCES)).hexdigest()[:12]
    d = tmp_path_factory.mktemp(f"kernels_host_{tag}")
    for p in SOURCES:
        shutil.copy(p, d / p.name)
    flags = ["-O1", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-Wno-unknown-pragmas", "-shared", "-fPIC", "-pthread", "-I", str(d)]
    if oracle._cpu_has_fma():
        flags.append("-mfma")
    subprocess.run(["g++", *flags, str(d / "kernels_driver.cpp"), "-o", str(d / "libemuk.so")], check=True)
    L = C.CDLL(str(d / "libemuk.so"))
    vp, ull, i32 = C.c_void_p, C.c_ulonglong, C.c_int
    L.emuk_create.argtypes = [i32, i32, i32, i32, vp, ull, ull, i32]; L.emuk_create.restype = vp
    L.emuk_destroy.argtypes = [vp]
    L.emuk_set_disorder.argtypes = [vp, vp, vp]
    L.emuk_init_spins.argtypes = [vp]
    L.emuk_set_spins.argtypes = [vp, vp]; L.emuk_get_spins.argtypes = [vp, vp]
    L.emuk_set_perm.argtypes = [vp, vp]; L.emuk_get_perm.argtypes = [vp, vp]
    L.emuk_sweep_generic.argtypes = [vp, i32, i32]
    L.emuk_pt_swap.argtypes = [vp, vp]
    L.emuk_measure.argtypes = [vp, vp, vp, vp, vp]
    L.emuk_measure_field.argtypes = [vp, vp]; L.emuk_measure_field.restype = i32
    L.emuk_measure_chiral.argtypes = [vp, vp, vp]
    L.emuk_diag_reset.argtypes = [vp]
    L.emuk_diag_get.argtypes = [vp, vp, vp, vp]; L.emuk_diag_get.restype = ull
    L.emuk_selftest.argtypes = [ull, ull, vp]
    return L


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class Host:
    """The kernels on the host behind the method names of the binding."""

    def __init__(self, lib, L, D, O, temps, seed, sample_offset=0, fast=False):
        self.lib, self.L, self.D, self.O, self.T = lib, L, D, O, len(temps)
        self.N, self.P = L ** 3, O * (O - 1) // 2
        self.temps = np.ascontiguousarray(temps, dtype=np.float32)
        self.h = lib.emuk_create(L, D, O, self.T, _p(self.temps), seed, sample_offset, int(fast))

    def __del__(self):
        self.lib.emuk_destroy(self.h)

    def set_disorder(self, J, H=None):
        J = np.ascontiguousarray(J, dtype=np.float32); H = None if H is None else np.ascontiguousarray(H, dtype=np.float32)
        self.lib.emuk_set_disorder(self.h, _p(J), _p(H))

    def init_spins(self):
        self.lib.emuk_init_spins(self.h)

    def set_spins(self, S):
        S = np.ascontiguousarray(S, dtype=np.float32)
        self.lib.emuk_set_spins(self.h, _p(S))

    def get_spins(self):
        S = np.empty((self.D, self.O, self.T, 3, self.L, self.L, self.L), dtype=np.float32)
        self.lib.emuk_get_spins(self.h, _p(S))
        return S.astype(np.float64)

    def sweep(self, n_or, n_hb):
        self.lib.emuk_sweep_generic(self.h, n_or, n_hb)

    def pt_swap(self):
        acc = np.empty((self.D, self.O, max(self.T - 1, 0)), dtype=np.int32)
        self.lib.emuk_pt_swap(self.h, _p(acc))
        return acc

    def perm(self):
        p = np.empty((self.D, self.O, self.T), dtype=np.int32)
        self.lib.emuk_get_perm(self.h, _p(p))
        return p

    def measure(self, energy=True):
        E = np.empty((self.D, self.O, self.T)) if energy else None
        M = np.empty((self.D, self.O, self.T, 3)) if energy else None
        q0 = np.empty((self.D, self.P, self.T, 3, 3)); qk = np.empty((self.D, self.P, self.T, 3, 3, 2))
        self.lib.emuk_measure(self.h, _p(E), _p(M), _p(q0), _p(qk))
        return E, M, q0, qk

    def measure_field(self):
        chi = np.empty((self.D, self.T, 2, 3, 2))
        assert self.lib.emuk_measure_field(self.h, _p(chi)) == 0
        return chi

    def measure_chiral(self):
        qc0 = np.empty((self.D, self.P, self.T, 3)); qck = np.empty((self.D, self.P, self.T, 3, 2))
        self.lib.emuk_measure_chiral(self.h, _p(qc0), _p(qck))
        return qc0, qck

    def diag_reset(self):
        self.lib.emuk_diag_reset(self.h)

    def diag_get(self):
        moved = np.empty((self.D, self.O, self.T), dtype=np.int64); trav = np.empty((self.D, self.O, self.T), dtype=np.int64)
        p = np.empty(self.T)
        n = self.lib.emuk_diag_get(self.h, _p(moved), _p(trav), _p(p))
        return moved, trav, int(n), p


def _pair(lib, L, D, O, T, seed, h_r=0.1, sample_offset=0, warm=False, fast=False):
    if warm:      # a warm, closely spaced ladder: parallel tempering scrambles the slots within a few passes
        temps = (0.6 * (1.0 + 0.08 / L ** 1.5 * np.arange(T))).astype(np.float32)
    else:
        temps = hsg_inputs.geometric_ladder(0.08, 0.30, T) if T > 1 else np.array([0.2], dtype=np.float32)
    J = hsg_inputs.couplings(L, D, seed, sample_offset)
    H = hsg_inputs.gaussian_field(L, D, h_r, seed, sample_offset) if h_r > 0 else None
    dev = Host(lib, L, D, O, temps, seed, sample_offset, fast)
    orc = oracle.Oracle(L, D, O, temps, seed, precision=32, sample_offset=sample_offset, n_threads=8)
    for s in (dev, orc):
        s.set_disorder(J, H); s.init_spins()
    return dev, orc, J, H


@pytest.mark.parametrize("L,D,O,T", [(4, 2, 2, 3), (6, 1, 1, 2), (8, 1, 2, 4), (10, 2, 1, 3), (12, 1, 2, 2)])
def test_start_spins_layout_conversion_and_generic_sweeps_bit_for_bit(lib, L, D, O, T):
    """V = 4 (L = 8), 2 (L = 4, 12) and 1 (L = 6, 10) sites per thread; zero and non-zero sample offset."""
    dev, orc, _, _ = _pair(lib, L, D, O, T, seed=11 + L, sample_offset=L % 3)
    assert np.array_equal(dev.get_spins(), orc.get_spins())
    dev.sweep(3, 2); orc.sweep(3, 2)
    assert np.array_equal(dev.get_spins(), orc.get_spins())
    S = hsg_inputs.unit_spins(L, D, O, T, seed=9)
    dev.set_spins(S)
    assert np.array_equal(dev.get_spins(), S.astype(np.float32).astype(np.float64))


def test_parallel_tempering_observables_and_diagnostics_in_lockstep(lib):
    L, D, O, T = 4, 1, 3, 5
    dev, orc, _, _ = _pair(lib, L, D, O, T, seed=21, warm=True)
    n_acc = 0
    for step in range(24):
        if step == 5:
            dev.diag_reset(); orc.pt_diag_reset()          # the reset must read the CURRENT (scrambled) permutation
        dev.sweep(1, 1); orc.sweep(1, 1)
        acc = orc.pt_swap()
        assert np.array_equal(dev.pt_swap(), acc), step
        assert np.array_equal(dev.perm(), orc.get_state()[0])
        n_acc += int(acc.sum())
        if step % 8 == 7:
            E, M, q0, qk = dev.measure(); Eo, Mo, q0o, qko = orc.measure()
            np.testing.assert_allclose(E, Eo, rtol=1e-12)
            np.testing.assert_allclose(M, Mo, rtol=0, atol=1e-13)
            np.testing.assert_allclose(q0, q0o, rtol=0, atol=1e-13)
            np.testing.assert_allclose(qk, qko, rtol=0, atol=1e-13)
            assert np.abs(E - orc.energy_plain()).max() < L ** 3 / 2 * 9 * 2.0 ** -24 * 8
    assert n_acc > 10 and not np.array_equal(dev.perm(), np.broadcast_to(np.arange(T), (D, O, T)))
    assert np.array_equal(dev.get_spins(), orc.get_spins())
    moved, trav, n, p = dev.diag_get(); m_o, t_o, n_o, p_o = orc.pt_diag_get()
    assert n == n_o == 19 and np.array_equal(moved, m_o) and np.array_equal(trav, t_o) and trav.sum() > 0
    np.testing.assert_allclose(p, p_o, rtol=1e-15)


@pytest.mark.parametrize("L,D,O,T,plain", [(4, 2, 4, 3, True), (6, 1, 5, 2, True), (8, 1, 4, 2, True), (16, 1, 4, 2, False), (34, 1, 4, 1, False)])
def test_field_case_chi_on_the_host(lib, L, D, O, T, plain):
    """chi_1..3 of Eq. (10) after parallel tempering has moved the labels: against the O(N^2) definition on the small
    lattices, the oracle's factored form beyond.  L = 34: one site per thread and three chunks of planes per system."""
    dev, orc, _, _ = _pair(lib, L, D, O, T, seed=51 + L, warm=True)
    for _ in range(3 if L <= 16 else 1):
        dev.sweep(1, 1); orc.sweep(1, 1)
        assert np.array_equal(dev.pt_swap(), orc.pt_swap())
    N = L ** 3
    np.testing.assert_allclose(dev.measure_field(), orc.chi_field(plain=plain), rtol=1e-11, atol=1e-13 * N * N)


@pytest.mark.parametrize("L,D,O,T", [(4, 2, 2, 3), (6, 1, 3, 2), (8, 1, 2, 3), (16, 1, 2, 2), (34, 1, 2, 1)])
def test_chiral_overlaps_on_the_host(lib, L, D, O, T):
    dev, orc, _, _ = _pair(lib, L, D, O, T, seed=71 + L, warm=True)
    for _ in range(3 if L <= 16 else 1):
        dev.sweep(1, 1); orc.sweep(1, 1)
        assert np.array_equal(dev.pt_swap(), orc.pt_swap())
    qc0, qck = dev.measure_chiral(); r0, rk = orc.measure_chiral()
    np.testing.assert_allclose(qc0, r0, rtol=0, atol=1e-14)
    np.testing.assert_allclose(qck, rk, rtol=0, atol=1e-14)
    assert np.abs(r0).max() > 1e-5
    E, M, q0, qk = dev.measure(); Eo, Mo, q0o, qko = orc.measure()      # (the overlap kernel with chunks of planes at L = 34)
    np.testing.assert_allclose(q0, q0o, rtol=0, atol=1e-13); np.testing.assert_allclose(qk, qko, rtol=0, atol=1e-13)
    np.testing.assert_allclose(E, Eo, rtol=1e-12)


def test_fast_math_generic_sweep_stays_inside_its_bound_on_the_host(lib):
    """HSG_FLAG_FAST_MATH through the generic kernel, special-function unit modelled by libm: colour 0 of one heat-bath sweep is
    drawn from equal inputs, so the per-site bound applies as it stands (tests/test_variants_gpu.py does the same on the GPU)."""
    L, D, O, T = 8, 1, 2, 4
    temps = np.asarray([0.06, 0.25, 3.0, 60.0], dtype=np.float32)
    J = hsg_inputs.couplings(L, D, 91); H = hsg_inputs.gaussian_field(L, D, 0.1, 91)
    dev = Host(lib, L, D, O, temps, 91, fast=True)
    orc = oracle.Oracle(L, D, O, temps, 91, precision=32)
    for s in (dev, orc):
        s.set_disorder(J, H); s.init_spins()
    dev.sweep(2, 0); orc.sweep(2, 0)
    assert np.array_equal(dev.get_spins(), orc.get_spins())              # over-relaxation is untouched by the flag
    S1 = orc.get_spins()
    dev.sweep(0, 1); orc.sweep(0, 1)
    a_dev, a_ref = dev.get_spins(), orc.get_spins()
    dev_max = np.abs(a_dev - a_ref).max(axis=3)[0]
    h = np.broadcast_to(H[0].astype(np.float64), S1[0].shape).copy()
    for d, ax in enumerate((-1, -2, -3)):
        h += J[0, d].astype(np.float64) * np.roll(S1[0], -1, axis=ax) + np.roll(J[0, d].astype(np.float64), 1, axis=ax) * np.roll(S1[0], 1, axis=ax)
    beta = (1.0 / temps.astype(np.float64)).astype(np.float32).astype(np.float64)
    a = np.sqrt((h ** 2).sum(axis=-4)) * beta[None, :, None, None, None]
    z, y, x = np.meshgrid(np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    even = np.broadcast_to((x + y + z) % 2 == 0, dev_max.shape)
    assert (dev_max[even] <= fast_math_bound(a[even]) + 1e-7).all()
    assert 0 < dev_max.max() and np.median(dev_max) < 5e-6


def test_arithmetic_self_test_kernel_on_the_host(lib):
    counts = np.zeros(3, dtype=np.uint64)
    lib.emuk_selftest(12345, 300000, _p(counts))
    assert tuple(counts) == (0, 0, 0)


def test_overlap_of_a_lattice_wider_than_a_block_on_the_host(lib):
    """L = 258 (Lh = 129, one site per item, 258 items per row lane > 256 threads): the reductions take their items in
    several passes (q came back as zeros)."""
    L = 258
    temps = np.array([0.5], dtype=np.float32)
    dev = Host(lib, L, 1, 2, temps, 9)
    rng = np.random.default_rng(4)
    S = rng.normal(size=(1, 2, 1, 3, L, L, L)).astype(np.float32)
    S /= np.sqrt((S.astype(np.float64) ** 2).sum(axis=3, keepdims=True)).astype(np.float32)
    dev.set_disorder(np.zeros((1, 3, L, L, L), dtype=np.float32), None)
    dev.set_spins(S)
    _, _, q0, qk = dev.measure(energy=False)
    Sd = S.astype(np.float64)
    ref = np.einsum("mzyx,nzyx->mn", Sd[0, 0, 0], Sd[0, 1, 0]) / L ** 3
    np.testing.assert_allclose(q0[0, 0, 0], ref, atol=1e-12)
    ph = np.exp(2j * np.pi * np.arange(L) / L)
    refk = np.einsum("mzyx,nzyx,x->mn", Sd[0, 0, 0], Sd[0, 1, 0], ph) / L ** 3
    np.testing.assert_allclose(qk[0, 0, 0, :, :, 0], refk.real, atol=1e-12)
    np.testing.assert_allclose(qk[0, 0, 0, :, :, 1], refk.imag, atol=1e-12)
    assert np.abs(q0).max() > 0
