"""ORACLE — test infrastructure, NOT part of the product path.

ctypes front end of ``oracle/hsg_oracle.cpp`` (plain serial C++ written from PAPER.md; see that
file's header).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_1204_6192_b200`` and the CUDA path imports nothing from here.

The shared object is built on first use, on the machine that uses it (``-mfma`` only when
/proc/cpuinfo lists it, so a library built on one host never runs an illegal instruction on
another; without it gcc falls back to the correctly rounded libm ``fmaf``).
"""
from __future__ import annotations

import ctypes as C
import hashlib
import os
import platform
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "hsg_oracle.cpp"
_LIB = None


def _cpu_has_fma() -> bool:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    return " fma " in (line + " ")
    except OSError:
        pass
    return False


def build(force: bool = False) -> Path:
    """Compile oracle/hsg_oracle.cpp with g++ (no CUDA, no torch) and return the .so path."""
    flags = ["-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC", "-pthread"]
    if _cpu_has_fma():
        flags.append("-mfma")
    tag = hashlib.sha1((_SRC.read_text() + " ".join(flags) + platform.machine()).encode()).hexdigest()[:12]
    out = _HERE / "build" / f"liboracle_{tag}.so"
    if out.exists() and not force:
        return out
    out.parent.mkdir(parents=True, exist_ok=True)
    tmp = out.with_suffix(f".tmp{os.getpid()}.so")
    subprocess.run(["g++", *flags, str(_SRC), "-o", str(tmp)], check=True)
    os.replace(tmp, out)
    return out


def lib() -> C.CDLL:
    global _LIB
    if _LIB is None:
        L = C.CDLL(str(build()))
        vp, i32, u32, u64, f32, f64 = C.c_void_p, C.c_int32, C.c_uint32, C.c_uint64, C.c_float, C.c_double
        L.orc_philox4x32_10.argtypes = [vp, vp, vp]
        L.orc_u01.argtypes = [u32]; L.orc_u01.restype = f64
        L.orc_u01_f32.argtypes = [u32]; L.orc_u01_f32.restype = f32
        L.orc_spec_omexp_f32.argtypes = [f32]; L.orc_spec_omexp_f32.restype = f32
        L.orc_spec_log1m_f32.argtypes = [f32]; L.orc_spec_log1m_f32.restype = f32
        L.orc_spec_sincos2pi_f32.argtypes = [f32, vp, vp]
        for n in ("orc_or_reflect_f32", "orc_or_reflect_f64"):
            getattr(L, n).argtypes = [vp, vp, vp]
        L.orc_hb_draw_f32.argtypes = [vp, f32, f32, f32, vp]
        L.orc_hb_draw_f64.argtypes = [vp, f64, f64, f64, vp]
        L.orc_hb_sample.argtypes = [C.c_int, vp, f64, u64, C.c_long, vp]
        L.orc_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, vp, u64, u64, C.c_int]
        L.orc_create.restype = vp
        L.orc_destroy.argtypes = [vp]
        L.orc_set_disorder.argtypes = [vp, vp, vp]
        L.orc_init_spins.argtypes = [vp]
        L.orc_set_spins.argtypes = [vp, vp]
        L.orc_get_spins.argtypes = [vp, vp]
        L.orc_sweep.argtypes = [vp, C.c_int, C.c_int, C.c_int]
        L.orc_energy.argtypes = [vp, vp]
        L.orc_energy_plain.argtypes = [vp, vp]
        L.orc_pt_swap.argtypes = [vp, vp]
        L.orc_measure.argtypes = [vp, vp, vp, vp, vp]
        L.orc_get_state.argtypes = [vp, vp, vp]
        L.orc_chi_field.argtypes = [vp, vp, C.c_int, C.c_int]; L.orc_chi_field.restype = C.c_int
        L.orc_measure_chiral.argtypes = [vp, vp, vp, vp]
        L.orc_xi_second_moment.argtypes = [f64, f64, C.c_int]; L.orc_xi_second_moment.restype = f64
        L.orc_pt_diag_reset.argtypes = [vp]
        L.orc_pt_diag_get.argtypes = [vp, vp, vp, vp, vp]
        L.orc_set_counters.argtypes = [vp, vp]
        _LIB = L
    return _LIB


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


# ---- unit-level functions -------------------------------------------------------------------
def philox4x32_10(ctr, key) -> np.ndarray:
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32); key = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.empty(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_p(ctr), _p(key), _p(out))
    return out


def u01(w: int) -> float:
    return lib().orc_u01(int(w))


def spec_omexp_f32(x: float) -> float:
    return lib().orc_spec_omexp_f32(float(x))


def spec_log1m_f32(y: float) -> float:
    return lib().orc_spec_log1m_f32(float(y))


def spec_sincos2pi_f32(u: float):
    s = C.c_float(); c = C.c_float()
    lib().orc_spec_sincos2pi_f32(float(u), C.addressof(s), C.addressof(c))
    return s.value, c.value


def or_reflect(s, h, precision=64) -> np.ndarray:
    dt = np.float32 if precision == 32 else np.float64
    s = np.ascontiguousarray(s, dtype=dt); h = np.ascontiguousarray(h, dtype=dt); out = np.empty(3, dtype=dt)
    getattr(lib(), f"orc_or_reflect_f{precision}")(_p(s), _p(h), _p(out))
    return out


def hb_draw(h, beta, u1, u2, precision=64) -> np.ndarray:
    dt = np.float32 if precision == 32 else np.float64
    h = np.ascontiguousarray(h, dtype=dt); out = np.empty(3, dtype=dt)
    getattr(lib(), f"orc_hb_draw_f{precision}")(_p(h), float(beta), float(u1), float(u2), _p(out))
    return out


def xi_second_moment(chi_0: float, chi_k: float, L: int) -> float:
    """Eq. (8) / Eq. (15): xi = sqrt(chi(0)/chi(k_min) - 1) / (2 sin(k_min/2)), |k_min| = 2 pi/L."""
    return lib().orc_xi_second_moment(float(chi_0), float(chi_k), int(L))


def hb_sample(h, beta, seed, n, precision=64) -> np.ndarray:
    h = np.ascontiguousarray(h, dtype=np.float64); out = np.empty((n, 3), dtype=np.float64)
    lib().orc_hb_sample(int(precision), _p(h), float(beta), int(seed), int(n), _p(out))
    return out


# ---- simulation object ----------------------------------------------------------------------
class Oracle:
    """Serial reference simulation.  precision=32 is the GPU's trajectory reference, 64 the physics truth.

    Arrays: J[D][3][L][L][L] (z,y,x order, bond site -> site+e_dir), H[D][3][L][L][L],
    spins S[D][O][T][3][L][L][L] indexed by temperature index.
    """

    def __init__(self, L, n_samples, n_replicas, temps, seed, precision=32, sample_offset=0, n_threads=1):
        self.L, self.D, self.O, self.T = int(L), int(n_samples), int(n_replicas), len(temps)
        self.N = self.L ** 3
        self.precision = precision
        self.n_threads = n_threads
        self.temps = np.ascontiguousarray(temps, dtype=np.float32)
        self._h = lib().orc_create(self.L, self.D, self.O, self.T, _p(self.temps), int(seed), int(sample_offset), precision)
        if not self._h:
            raise ValueError("orc_create: invalid arguments")

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_destroy(self._h); self._h = None

    def set_disorder(self, J, H=None):
        J = np.ascontiguousarray(J, dtype=np.float32).reshape(self.D, 3, self.N)
        Hh = None if H is None else np.ascontiguousarray(H, dtype=np.float32).reshape(self.D, 3, self.N)
        lib().orc_set_disorder(self._h, _p(J), _p(Hh))

    def init_spins(self):
        lib().orc_init_spins(self._h)

    def set_spins(self, S):
        S = np.ascontiguousarray(S, dtype=np.float64).reshape(self.D, self.O, self.T, 3, self.N)
        lib().orc_set_spins(self._h, _p(S))

    def get_spins(self) -> np.ndarray:
        S = np.empty((self.D, self.O, self.T, 3, self.L, self.L, self.L), dtype=np.float64)
        lib().orc_get_spins(self._h, _p(S))
        return S

    def sweep(self, n_or, n_hb):
        lib().orc_sweep(self._h, int(n_or), int(n_hb), int(self.n_threads))

    def energy(self) -> np.ndarray:
        E = np.empty((self.D, self.O, self.T), dtype=np.float64)
        lib().orc_energy(self._h, _p(E))
        return E

    def energy_plain(self) -> np.ndarray:
        """Eq. (1) as written: forward bonds once, every product and the sum in fp64 (the plain definition)."""
        E = np.empty((self.D, self.O, self.T), dtype=np.float64)
        lib().orc_energy_plain(self._h, _p(E))
        return E

    def pt_swap(self) -> np.ndarray:
        acc = np.empty((self.D, self.O, max(self.T - 1, 0)), dtype=np.int32)
        lib().orc_pt_swap(self._h, _p(acc))
        return acc

    def measure(self):
        P = self.O * (self.O - 1) // 2
        E = np.empty((self.D, self.O, self.T), dtype=np.float64)
        M = np.empty((self.D, self.O, self.T, 3), dtype=np.float64)
        q0 = np.empty((self.D, P, self.T, 3, 3), dtype=np.float64)
        qk = np.empty((self.D, P, self.T, 3, 3, 2), dtype=np.float64)
        lib().orc_measure(self._h, _p(E), _p(M), _p(q0), _p(qk))
        return E, M, q0, qk

    def chi_field(self, plain=False) -> np.ndarray:
        """Summands of Eq. (10) from replicas 0..3: chi[D][T][2 (k=0, k_min)][3 (chi_1, chi_2, chi_3)][2 (re, im)].
        plain=True: the O(N^2) double sum as printed; False: the factored form (identical numbers, pinned)."""
        chi = np.empty((self.D, self.T, 2, 3, 2), dtype=np.float64)
        if lib().orc_chi_field(self._h, _p(chi), int(bool(plain)), int(self.n_threads)) != 0:
            raise ValueError("chi_field needs at least four replicas")
        return chi

    def measure_chiral(self, want_kappa=False):
        """Chiral overlaps of Eqs. (12), (13): qc0[D][P][T][3], qck[D][P][T][3][2]; optionally kappa[D][O][T][3][L][L][L]."""
        P = self.O * (self.O - 1) // 2
        qc0 = np.empty((self.D, P, self.T, 3), dtype=np.float64)
        qck = np.empty((self.D, P, self.T, 3, 2), dtype=np.float64)
        kap = np.empty((self.D, self.O, self.T, 3, self.L, self.L, self.L), dtype=np.float64) if want_kappa else None
        lib().orc_measure_chiral(self._h, _p(qc0), _p(qck), _p(kap))
        return (qc0, qck, kap) if want_kappa else (qc0, qck)

    def pt_diag_reset(self):
        """Start (or restart) the parallel-tempering diagnostics of PAPER.md:197 / Fig. 3; every later pt_swap() is counted."""
        lib().orc_pt_diag_reset(self._h)

    def pt_diag_get(self):
        """(moved[D][O][T] by temperature index, traversals[D][O][T] by configuration slot, n_pass, p_diff[T])."""
        moved = np.empty((self.D, self.O, self.T), dtype=np.int64)
        trav = np.empty((self.D, self.O, self.T), dtype=np.int64)
        n = C.c_uint64(0)
        p = np.empty(self.T, dtype=np.float64)
        lib().orc_pt_diag_get(self._h, _p(moved), _p(trav), C.addressof(n), _p(p))
        return moved, trav, int(n.value), p

    def get_state(self):
        perm = np.empty((self.D, self.O, self.T), dtype=np.int32)
        cnt = np.empty(2, dtype=np.uint64)
        lib().orc_get_state(self._h, _p(perm), _p(cnt))
        return perm, cnt

    def set_counters(self, k_hb, k_pt):
        cnt = np.array([k_hb, k_pt], dtype=np.uint64)
        lib().orc_set_counters(self._h, _p(cnt))
