"""The z-marching sweep kernel (paper_1204_6192_b200/csrc/hsg_zmarch.cuh — the hot kernel, its source unmodified) executed on
the HOST, thread for thread, and compared with the oracle bit for bit.  No GPU.

The kernel is plain C++ over csrc/hsg_zmarch_ptx.cuh (PTX wrappers, CUDA built-ins) and csrc/hsg_prim.cuh (rounded
arithmetic).  tests/host_emul/ restates exactly those two headers on a small execution model (emu.h): one OS thread per CUDA
thread, CTA barriers, warp shuffles, mbarriers with transaction counts, per-thread cp.async groups, bulk copies, remote
shared-memory stores into the neighbour CTA of a thread-block cluster, the split cluster barrier.  Asynchronous copies land
either when they are issued (mode "early") or only when somebody waits for them ("late") — the two ends of the window the
hardware allows — so that a ring slot overwritten too early or a read that was never waited for gives wrong spins in one of
the two modes.  What is checked: thread-to-site ownership, neighbour indexing and the x neighbours that travel by shuffle,
ring-slot and mbarrier-phase arithmetic, the strip / halo protocol of the L = 64 cluster kernel, the heat-bath counters, the
fused energy / magnetisation reduction.  What is NOT: the PTX instructions themselves, memory-model subtleties below this
granularity, and performance — those need the GPU (-m gpu parity tests, ncu)."""
import ctypes as C
import hashlib
import re
import shutil
import subprocess
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

import numpy as np
import pytest

import hsg_inputs
import oracle

ROOT = Path(__file__).resolve().parent.parent
CSRC = ROOT / "paper_1204_6192_b200" / "csrc"
HERE = Path(__file__).resolve().parent
SOURCES = [CSRC / "hsg_zmarch.cuh", CSRC / "hsg_zmarch_launch.h", CSRC / "hsg_layout.cuh", CSRC / "hsg_math.cuh",
           HERE / "host_math" / "cuda_runtime.h", HERE / "host_math" / "hsg_prim.cuh",
           HERE / "host_emul" / "emu.h", HERE / "host_emul" / "hsg_zmarch_ptx.cuh", HERE / "host_emul" / "zmarch_driver.cpp"]
EARLY, LATE = 0, 1


def _build(d: Path, sizes, edit=None):
    """Copy the kernel source and the host restatements into d (optionally editing the KERNEL copy: seeded faults), compile
    one shared object per lattice size in parallel."""
    for p in SOURCES:
        shutil.copy(p, d / p.name)
    if edit is not None:
        k = d / "hsg_zmarch.cuh"
        text = k.read_text()
        new = edit(text)
        assert new != text, "the edit did not change the kernel source"
        k.write_text(new)
    flags = ["-O1", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-Wno-unknown-pragmas", "-shared", "-fPIC", "-pthread", "-I", str(d)]
    if oracle._cpu_has_fma():
        flags.append("-mfma")

    def one(L):
        out = d / f"libemu_l{L}.so"
        subprocess.run(["g++", *flags, f"-DEMU_L={L}", str(d / "zmarch_driver.cpp"), "-o", str(out)], check=True)
        return L, out
    with ThreadPoolExecutor(max_workers=4) as ex:
        return dict(ex.map(one, sizes))


def _entry(so: Path, L):
    lib = C.CDLL(str(so))
    f = getattr(lib, f"emu_zmarch_l{L}")
    vp, ull, i32 = C.c_void_p, C.c_ulonglong, C.c_int
    f.argtypes = [i32, i32, i32, i32, i32, vp, ull, ull, ull, i32, i32, vp, vp, vp, vp, vp, i32]
    f.restype = i32
    return f


@pytest.fixture(scope="module")
def emu(tmp_path_factory):
    tag = hashlib.sha1(b"".join(p.read_bytes() for p in SOURCES)).hexdigest()[:12]
    d = tmp_path_factory.mktemp(f"zmarch_host_{tag}")
    return {L: _entry(so, L) for L, so in _build(d, (8, 16, 32, 64)).items()}


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _run(entry, L, G, mode, D, O, T, calls, seed=5, sample_offset=0, h_r=0.1, t_lo=0.08, t_hi=0.30):
    """calls = [(n_or, n_hb), ...] made one after the other on the emulated kernel and on the oracle; returns the largest spin
    difference, with the fused E and m of the last call checked on the way."""
    temps = hsg_inputs.geometric_ladder(t_lo, t_hi, T) if T > 1 else np.array([0.5 * (t_lo + t_hi)], dtype=np.float32)
    J = hsg_inputs.couplings(L, D, seed, sample_offset)
    H = hsg_inputs.gaussian_field(L, D, h_r, seed, sample_offset) if h_r > 0 else None
    orc = oracle.Oracle(L, D, O, temps, seed, precision=32, sample_offset=sample_offset, n_threads=8)
    orc.set_disorder(J, H); orc.init_spins()
    S = np.ascontiguousarray(orc.get_spins().astype(np.float32))
    E = np.zeros(D * O * T); M = np.zeros((D * O * T, 3))
    k_hb = 0
    for n_or, n_hb in calls:
        rc = entry(G, mode, D, O, T, _p(temps), seed, sample_offset, k_hb, n_or, n_hb, _p(J), _p(H), _p(S), _p(E), _p(M), 0)
        assert rc == 0, rc
        k_hb += n_hb
        orc.sweep(n_or, n_hb)
    dev = float(np.abs(S.astype(np.float64) - orc.get_spins()).max())
    if dev == 0.0:
        Eo, Mo, _, _ = orc.measure()
        np.testing.assert_allclose(E, np.asarray(Eo).reshape(-1), rtol=1e-12)
        np.testing.assert_allclose(M, np.asarray(Mo).reshape(-1, 3), rtol=0, atol=1e-13)
    return dev


# (L, G, D, O, T, calls): every lattice size of the kernel, the smallest and the largest group size each can run with,
# several samples (J/H per sample), several temperatures per chain, warm rings across calls, OR-only / HB-only / mixed calls
CASES = [
    (8, 2, 2, 2, 3, [(2, 1), (1, 2)]),
    (8, 8, 1, 2, 4, [(1, 1)]),
    (8, 1, 1, 1, 3, [(1, 1)]),               # 16-thread CTA (O*T odd): half a warp
    (8, 4, 1, 2, 2, [(1, 1)]),               # the group size zmarch_pick_g takes for a few hundred systems
    (16, 1, 1, 1, 3, [(2, 1)]),
    (16, 8, 2, 2, 4, [(2, 0), (0, 2)]),
    (16, 4, 1, 2, 2, [(1, 1)]),
    (32, 2, 1, 2, 2, [(2, 1)]),
    (32, 1, 2, 1, 1, [(1, 1)]),              # two samples: the J/H planes of the second one
    (64, 2, 1, 2, 1, [(1, 1)]),              # thread-block cluster of four strips, two systems per CTA
    (64, 1, 1, 1, 1, [(1, 1)]),
]


@pytest.mark.parametrize("mode", [EARLY, LATE], ids=["early", "late"])
@pytest.mark.parametrize("L,G,D,O,T,calls", CASES, ids=[f"L{c[0]}-G{c[1]}" for c in CASES])
def test_sweep_kernel_on_the_host_model_reproduces_the_oracle_bit_for_bit(emu, L, G, D, O, T, calls, mode):
    assert _run(emu[L], L, G, mode, D, O, T, calls, seed=5 + L, sample_offset=3) == 0.0


def test_zero_field_and_hot_ladder_on_the_host_model(emu):
    """H = NULL packs as a zero field; a hot ladder drives the heat bath through the series branch (a < 1e-4)."""
    assert _run(emu[16], 16, 2, LATE, 1, 2, 2, [(1, 2)], h_r=0.0) == 0.0
    assert _run(emu[8], 8, 2, EARLY, 1, 2, 2, [(1, 2)], t_lo=1e2, t_hi=1e6) == 0.0


@pytest.mark.parametrize("L,G", [(8, 2), (32, 2)])
def test_fast_math_variant_of_the_sweep_kernel_on_the_host_model(emu, L, G):
    """zmarch_kernel<..., FM = true> (HSG_FLAG_FAST_MATH), special-function unit modelled by libm: over-relaxation sweeps stay
    bit-identical, and after one heat-bath sweep colour 0 (drawn from equal inputs) is inside the variant's stated bound,
    the typical deviation at the 1e-6 level (the same assertions tests/test_variants_gpu.py makes on the GPU)."""
    from tests.test_device_math_on_host import fast_math_bound
    D, O, seed = 1, 2, 91
    temps = np.asarray([0.06, 3.0], dtype=np.float32)
    T = len(temps)
    J = hsg_inputs.couplings(L, D, seed); H = hsg_inputs.gaussian_field(L, D, 0.1, seed)
    orc = oracle.Oracle(L, D, O, temps, seed, precision=32, n_threads=8)
    orc.set_disorder(J, H); orc.init_spins()
    S = np.ascontiguousarray(orc.get_spins().astype(np.float32))
    E = np.zeros(D * O * T); M = np.zeros((D * O * T, 3))
    assert emu[L](G, LATE, D, O, T, _p(temps), seed, 0, 0, 2, 0, _p(J), _p(H), _p(S), _p(E), _p(M), 1) == 0
    orc.sweep(2, 0)
    S1 = orc.get_spins()
    assert np.array_equal(S.astype(np.float64), S1)
    assert emu[L](G, EARLY, D, O, T, _p(temps), seed, 0, 0, 0, 1, _p(J), _p(H), _p(S), _p(E), _p(M), 1) == 0
    orc.sweep(0, 1)
    dev = np.abs(S.astype(np.float64) - orc.get_spins()).max(axis=3)[0]
    h = np.broadcast_to(H[0].astype(np.float64), S1[0].shape).copy()
    for d, ax in enumerate((-1, -2, -3)):
        h += J[0, d].astype(np.float64) * np.roll(S1[0], -1, axis=ax) + np.roll(J[0, d].astype(np.float64), 1, axis=ax) * np.roll(S1[0], 1, axis=ax)
    beta = (1.0 / temps.astype(np.float64)).astype(np.float32).astype(np.float64)
    a = np.sqrt((h ** 2).sum(axis=-4)) * beta[None, :, None, None, None]
    z, y, x = np.meshgrid(np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    even = np.broadcast_to((x + y + z) % 2 == 0, dev.shape)
    assert (dev[even] <= fast_math_bound(a[even]) + 1e-7).all()
    assert 0 < dev.max() and np.median(dev) < 5e-6 and np.quantile(dev, 0.99) < 2e-4
    np.testing.assert_allclose(E, orc.energy().reshape(-1), rtol=1e-4)


# Seeded faults: the model must SEE a broken protocol, each in the mode its kind of hazard belongs to.
FAULTS = {
    # the step reads its stage one cp.async group too early: a read of data nobody waited for -> visible when copies land late
    "stage_not_waited_for": (lambda s: s.replace("cp_async_wait<C::DS - 1>();", "cp_async_wait<C::DS>();", 1), LATE, EARLY),
    # the ring of old colour-1 planes one slot too small: a live plane is overwritten by the copy for a later step -> visible
    # when copies land early
    "spin_ring_too_small": (lambda s: s.replace("static constexpr int NC1 = DS + 2;", "static constexpr int NC1 = DS + 1;", 1), EARLY, LATE),
    # the J/H mbarrier is not waited for (wrong in either mode: without the wait a thread can also overtake the ISSUE of the copy)
    "jh_plane_not_waited_for": (lambda s: s.replace("    mbar_wait(bar, parity);\n", "    (void)bar; (void)parity;\n", 1), LATE, None),
}


def _no_halo_wait(s):
    return s.replace("if (HALO) { mbar_wait(sm.hfull + 8u * par, (hph >> par) & 1u); hph ^= 1u << par; }", "if (HALO) { hph ^= 1u << par; }", 1)


def _dj1(s):
    s = s.replace("template <> struct Tune<64> { static constexpr int YS = 16, V = 4, VHB = 4, GMAX = 2, DS = 2, DJ = 2; };",
                  "template <> struct Tune<64> { static constexpr int YS = 16, V = 4, VHB = 4, GMAX = 2, DS = 2, DJ = 1; };", 1)
    return re.sub(r"\n  static_assert\(!HALO \|\| DJ >= 2,[^\n]*\n", "\n", s, count=1)


@pytest.fixture(scope="module")
def edited(tmp_path_factory):
    """The edited copies of the kernel (seeded faults at L = 16, the halo fault and the DJ = 1 ring at L = 64), built side by
    side: name -> entry point."""
    jobs = {name: (16, f[0]) for name, f in FAULTS.items()}
    jobs["no_halo_wait"] = (64, _no_halo_wait)
    jobs["dj1"] = (64, _dj1)

    def one(item):
        name, (L, edit) = item
        return name, _entry(_build(tmp_path_factory.mktemp(f"zmarch_{name}"), (L,), edit)[L], L)
    with ThreadPoolExecutor(max_workers=len(jobs)) as ex:
        return dict(ex.map(one, jobs.items()))


@pytest.mark.parametrize("name", sorted(FAULTS))
def test_the_host_model_detects_seeded_protocol_faults(edited, name):
    _, bad_mode, good_mode = FAULTS[name]
    entry = edited[name]
    assert _run(entry, 16, 8, bad_mode, 1, 2, 4, [(2, 1)]) > 1e-3
    if good_mode is not None:                     # the fault is of ONE kind: the other end of the window hides it
        assert _run(entry, 16, 8, good_mode, 1, 2, 4, [(2, 1)]) == 0.0


def test_halo_fault_in_the_cluster_kernel_is_detected(edited):
    """L = 64: the colour-1 update must wait for the halo rows its neighbour strips push (st.async + mbarrier)."""
    assert _run(edited["no_halo_wait"], 64, 1, LATE, 1, 1, 1, [(1, 0)]) > 1e-3


def test_jh_ring_depth_one_in_the_cluster_kernel_passes_the_model(edited):
    """J/H ring depth DJ = 1 faulted on the GPU at L = 64, G = 1 in round 1 and is not shipped.  On the model
    that configuration reproduces the oracle in both modes: whatever faulted is not a slot-reuse or missing-wait hazard of the
    ring protocol (it is recorded as an open point, and the kernel static_asserts DJ >= 2 for strip kernels)."""
    entry = edited["dj1"]
    assert _run(entry, 64, 1, EARLY, 1, 1, 1, [(1, 0)]) == 0.0
    assert _run(entry, 64, 1, LATE, 1, 1, 1, [(0, 1)]) == 0.0
