"""paper_1204_6192_b200 — thin Python binding of the hsg C ABI (include/hsg.h).

Argument marshalling only: every step of the hot path (sweeps, energies, parallel tempering,
measurements, layout conversion, initialisation) runs in the CUDA kernels behind ``lib/libhsg.so``.
PyTorch provides device memory and the CUDA stream, nothing else.  There is no CPU fallback: importing
works without a GPU (so the symbol table can be checked), but creating an engine without CUDA raises.

    eng = hsg_create(L, n_samples, n_replicas, temps, seed)     # -> Hsg
    eng.set_disorder(J, H); eng.init_spins()
    eng.sweep(n_or=5, n_hb=1); acc = eng.pt_swap(); E, M, q0, qk = eng.measure()
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import _build

HSG_OK, HSG_EINVAL, HSG_ESTATE, HSG_EUNSUPPORTED, HSG_ECUDA = 0, -1, -2, -3, -4
HSG_KERNEL_AUTO, HSG_KERNEL_GENERIC, HSG_KERNEL_ZMARCH = 0, 1, 2
HSG_OPT_SWEEP_KERNEL, HSG_OPT_FUSE_ENERGY = 1, 2
HSG_FLAG_FAST_MATH = 1
KERNELS = {"auto": HSG_KERNEL_AUTO, "generic": HSG_KERNEL_GENERIC, "zmarch": HSG_KERNEL_ZMARCH}

# every symbol include/hsg.h declares (tests check that the library exports each of them)
SYMBOLS = (
    "hsg_query_bytes", "hsg_create", "hsg_destroy", "hsg_set_disorder", "hsg_init_spins", "hsg_set_spins",
    "hsg_get_spins", "hsg_sweep", "hsg_energy", "hsg_pt_swap", "hsg_measure", "hsg_get_state", "hsg_set_state",
    "hsg_set_option", "hsg_launch_count", "hsg_last_sweep_kernel", "hsg_last_error", "hsg_version", "hsg_selftest_arith",
    "hsg_measure_field", "hsg_measure_chiral", "hsg_xi_second_moment", "hsg_pt_diag_reset", "hsg_pt_diag_get",
)


class hsg_desc(C.Structure):
    _fields_ = [
        ("L", C.c_int32), ("n_samples", C.c_int32), ("n_replicas", C.c_int32), ("n_temps", C.c_int32),
        ("temps_host", C.POINTER(C.c_float)), ("seed", C.c_uint64), ("sample_offset", C.c_uint64), ("flags", C.c_uint32),
    ]


class HsgError(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"hsg error {code}: {text}")
        self.code = code


_LIB = None


def lib() -> C.CDLL:
    """Load (building first if the sources are newer) the C-ABI library.  Fails loudly if it cannot be built."""
    global _LIB
    if _LIB is None:
        L = C.CDLL(str(_build.build()))
        vp, i32 = C.c_void_p, C.c_int
        L.hsg_query_bytes.argtypes = [C.POINTER(hsg_desc), C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]
        L.hsg_create.argtypes = [C.POINTER(hsg_desc), vp, C.c_size_t, vp, C.c_size_t, vp, C.POINTER(vp)]
        L.hsg_destroy.argtypes = [vp]
        L.hsg_set_disorder.argtypes = [vp, vp, vp]
        L.hsg_init_spins.argtypes = [vp]
        L.hsg_set_spins.argtypes = [vp, vp]
        L.hsg_get_spins.argtypes = [vp, vp]
        L.hsg_sweep.argtypes = [vp, i32, i32]
        L.hsg_energy.argtypes = [vp, vp]
        L.hsg_pt_swap.argtypes = [vp, vp]
        L.hsg_measure.argtypes = [vp, vp, vp, vp, vp]
        L.hsg_get_state.argtypes = [vp, vp, C.POINTER(C.c_uint64)]
        L.hsg_set_state.argtypes = [vp, vp, C.POINTER(C.c_uint64)]
        L.hsg_set_option.argtypes = [vp, i32, i32]
        L.hsg_launch_count.argtypes = [vp]; L.hsg_launch_count.restype = C.c_uint64
        L.hsg_last_sweep_kernel.argtypes = [vp]; L.hsg_last_sweep_kernel.restype = C.c_char_p
        L.hsg_last_error.argtypes = [vp]; L.hsg_last_error.restype = C.c_char_p
        L.hsg_version.argtypes = []; L.hsg_version.restype = C.c_char_p
        L.hsg_selftest_arith.argtypes = [vp, C.c_uint64, C.c_uint64, vp]
        L.hsg_measure_field.argtypes = [vp, vp]
        L.hsg_measure_chiral.argtypes = [vp, vp, vp]
        L.hsg_xi_second_moment.argtypes = [C.c_double, C.c_double, C.c_int32, C.POINTER(C.c_double)]
        L.hsg_pt_diag_reset.argtypes = [vp]
        L.hsg_pt_diag_get.argtypes = [vp, vp, vp, vp, C.POINTER(C.c_uint64)]
        _LIB = L
    return _LIB


def hsg_version() -> str:
    return lib().hsg_version().decode()


def hsg_selftest_arith(n, seed=1, exceptional=False):
    """(division mismatches, square-root mismatches) of the kernels' branch-free IEEE routines over n operand sets;
    exceptional=True: the count for divisors whose mantissa is all ones instead (counted apart by the kernel)."""
    import torch
    counts = torch.zeros(3, dtype=torch.int64, device="cuda")
    rc = lib().hsg_selftest_arith(C.c_void_p(torch.cuda.current_stream().cuda_stream), int(seed), int(n), counts.data_ptr())
    if rc != HSG_OK:
        raise HsgError(rc, "hsg_selftest_arith failed")
    c = tuple(int(x) for x in counts.cpu())
    return c[2] if exceptional else c[:2]


def hsg_xi_second_moment(chi_0, chi_kmin, L) -> float:
    """Eq. (8) / Eq. (15) of the paper through the C ABI (host arithmetic)."""
    xi = C.c_double(0.0)
    rc = lib().hsg_xi_second_moment(float(chi_0), float(chi_kmin), int(L), C.byref(xi))
    if rc != HSG_OK:
        raise HsgError(rc, "hsg_xi_second_moment: chi(0) >= chi(k_min) > 0 required")
    return xi.value


def hsg_query_bytes(L, n_samples, n_replicas, temps, seed=0, sample_offset=0, flags=0):
    temps = np.ascontiguousarray(temps, dtype=np.float32)
    d = hsg_desc(int(L), int(n_samples), int(n_replicas), len(temps), temps.ctypes.data_as(C.POINTER(C.c_float)),
                 int(seed), int(sample_offset), int(flags))
    a, b = C.c_size_t(0), C.c_size_t(0)
    rc = lib().hsg_query_bytes(C.byref(d), C.byref(a), C.byref(b))
    if rc != HSG_OK:
        raise HsgError(rc, "hsg_query_bytes: invalid descriptor")
    return a.value, b.value


def _on_device(method):
    """Run a method with the engine's device current (hsg.h: the device of hsg_create() must be current at every call),
    so that engines on several devices can be driven from one process."""
    import functools

    @functools.wraps(method)
    def wrapped(self, *a, **kw):
        with self.torch.cuda.device(self.device):
            return method(self, *a, **kw)
    return wrapped


class Hsg:
    """One hsg context over torch-owned device buffers.  Methods mirror the C calls (hsg_<name>)."""

    def __init__(self, L, n_samples, n_replicas, temps, seed, sample_offset=0, device=None, stream=None, kernel="auto", flags=0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("hsg needs a CUDA device: there is no CPU fallback")
        self.torch = torch
        self.device = torch.device(device if device is not None else f"cuda:{torch.cuda.current_device()}")
        self.L, self.D, self.O = int(L), int(n_samples), int(n_replicas)
        self.temps = np.ascontiguousarray(temps, dtype=np.float32)
        self.T = len(self.temps)
        self.N = self.L ** 3
        self.P = self.O * (self.O - 1) // 2
        self._desc = hsg_desc(self.L, self.D, self.O, self.T, self.temps.ctypes.data_as(C.POINTER(C.c_float)),
                              int(seed), int(sample_offset), int(flags))
        nb_state, nb_scratch = C.c_size_t(0), C.c_size_t(0)
        rc = lib().hsg_query_bytes(C.byref(self._desc), C.byref(nb_state), C.byref(nb_scratch))
        if rc != HSG_OK:
            raise HsgError(rc, "hsg_query_bytes: invalid descriptor")
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self._state = torch.empty(max(nb_state.value, 256), dtype=torch.uint8, device=self.device)
            self._scratch = torch.empty(max(nb_scratch.value, 256), dtype=torch.uint8, device=self.device)
            h = C.c_void_p()
            rc = lib().hsg_create(C.byref(self._desc), self._state.data_ptr(), self._state.numel(), self._scratch.data_ptr(),
                                  self._scratch.numel(), C.c_void_p(self.stream.cuda_stream), C.byref(h))
        if rc != HSG_OK:
            raise HsgError(rc, "hsg_create failed")
        self._h = h
        if kernel != "auto":
            self.set_option(HSG_OPT_SWEEP_KERNEL, KERNELS[kernel])

    # -- helpers
    def _ck(self, rc):
        if rc != HSG_OK:
            raise HsgError(rc, lib().hsg_last_error(self._h).decode())

    def _dev(self, a, dtype, shape=None):
        """torch tensor on this device (numpy arrays are uploaded on the engine's stream)."""
        torch = self.torch
        if a is None:
            return None
        if not isinstance(a, torch.Tensor):
            a = torch.from_numpy(np.ascontiguousarray(a))
        with torch.cuda.stream(self.stream):
            a = a.to(device=self.device, dtype=dtype, non_blocking=True).contiguous()
        if shape is not None and tuple(a.shape) != tuple(shape):
            a = a.reshape(shape)
        return a

    def _new(self, shape, dtype):
        with self.torch.cuda.stream(self.stream):
            return self.torch.empty(shape, dtype=dtype, device=self.device)

    def destroy(self):
        if getattr(self, "_h", None):
            lib().hsg_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # -- the C calls
    def set_option(self, option, value):
        self._ck(lib().hsg_set_option(self._h, int(option), int(value)))

    @_on_device
    def set_disorder(self, J, H=None):
        t = self.torch
        Jd = self._dev(J, t.float32, (self.D, 3, self.L, self.L, self.L))
        Hd = self._dev(H, t.float32, (self.D, 3, self.L, self.L, self.L))
        self._ck(lib().hsg_set_disorder(self._h, Jd.data_ptr(), None if Hd is None else Hd.data_ptr()))
        self._keep = (Jd, Hd)      # stay alive until the pack kernel has run; freed at the next call

    @_on_device
    def init_spins(self):
        self._ck(lib().hsg_init_spins(self._h))

    @_on_device
    def set_spins(self, S):
        Sd = self._dev(S, self.torch.float32, (self.D, self.O, self.T, 3, self.L, self.L, self.L))
        self._ck(lib().hsg_set_spins(self._h, Sd.data_ptr()))
        self._keep_s = Sd

    @_on_device
    def get_spins(self, out=None):
        S = out if out is not None else self._new((self.D, self.O, self.T, 3, self.L, self.L, self.L), self.torch.float32)
        self._ck(lib().hsg_get_spins(self._h, S.data_ptr()))
        return S

    @_on_device
    def sweep(self, n_or, n_hb):
        self._ck(lib().hsg_sweep(self._h, int(n_or), int(n_hb)))

    @_on_device
    def energy(self, out=None):
        E = out if out is not None else self._new((self.D, self.O, self.T), self.torch.float64)
        self._ck(lib().hsg_energy(self._h, E.data_ptr()))
        return E

    @_on_device
    def pt_swap(self, out=None, want_flags=True):
        acc = None
        if want_flags:
            acc = out if out is not None else self._new((self.D, self.O, max(self.T - 1, 0)), self.torch.int32)
        self._ck(lib().hsg_pt_swap(self._h, None if acc is None else acc.data_ptr()))
        return acc

    @_on_device
    def measure(self, out=None):
        t = self.torch
        if out is None:
            out = (self._new((self.D, self.O, self.T), t.float64), self._new((self.D, self.O, self.T, 3), t.float64),
                   self._new((self.D, self.P, self.T, 3, 3), t.float64), self._new((self.D, self.P, self.T, 3, 3, 2), t.float64))
        E, M, q0, qk = out
        self._ck(lib().hsg_measure(self._h, *(None if x is None else x.data_ptr() for x in (E, M, q0, qk))))
        return E, M, q0, qk

    @_on_device
    def measure_field(self, out=None):
        chi = out if out is not None else self._new((self.D, self.T, 2, 3, 2), self.torch.float64)
        self._ck(lib().hsg_measure_field(self._h, chi.data_ptr()))
        return chi

    @_on_device
    def measure_chiral(self, out=None):
        t = self.torch
        if out is None:
            out = (self._new((self.D, self.P, self.T, 3), t.float64), self._new((self.D, self.P, self.T, 3, 2), t.float64))
        qc0, qck = out
        self._ck(lib().hsg_measure_chiral(self._h, *(None if x is None else x.data_ptr() for x in (qc0, qck))))
        return qc0, qck

    @_on_device
    def pt_diag_reset(self):
        self._ck(lib().hsg_pt_diag_reset(self._h))

    @_on_device
    def pt_diag_get(self):
        """(moved[D][O][T], traversals[D][O][T], p_diff[T]) device tensors and the number of passes counted."""
        t = self.torch
        moved, trav = self._new((self.D, self.O, self.T), t.int64), self._new((self.D, self.O, self.T), t.int64)
        p_diff = self._new((self.T,), t.float64)
        n = C.c_uint64(0)
        self._ck(lib().hsg_pt_diag_get(self._h, moved.data_ptr(), trav.data_ptr(), p_diff.data_ptr(), C.byref(n)))
        return moved, trav, p_diff, int(n.value)

    @_on_device
    def get_state(self):
        perm = self._new((self.D, self.O, self.T), self.torch.int32)
        cnt = (C.c_uint64 * 2)()
        self._ck(lib().hsg_get_state(self._h, perm.data_ptr(), cnt))
        return perm, (int(cnt[0]), int(cnt[1]))

    @_on_device
    def set_state(self, perm=None, counters=None):
        p = self._dev(perm, self.torch.int32, (self.D, self.O, self.T))
        cnt = None if counters is None else (C.c_uint64 * 2)(int(counters[0]), int(counters[1]))
        self._ck(lib().hsg_set_state(self._h, None if p is None else p.data_ptr(), cnt))
        self._keep_p = p

    def launch_count(self) -> int:
        return int(lib().hsg_launch_count(self._h))

    def last_sweep_kernel(self) -> str:
        return lib().hsg_last_sweep_kernel(self._h).decode()

    def synchronize(self):
        self.stream.synchronize()


def hsg_create(L, n_samples, n_replicas, temps, seed, **kw) -> Hsg:
    return Hsg(L, n_samples, n_replicas, temps, seed, **kw)
