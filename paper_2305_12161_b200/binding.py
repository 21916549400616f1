"""Thin Python binding of the C-ABI library (include/ising3d.h) -- argument marshalling only.

Every step of the path (init, sweep, RNG, measurement reductions) runs in the CUDA kernels
of libising3d.so; nothing here computes.  PyTorch is used for device memory and streams
only (the lattice lives in a torch uint8 tensor, kernels run on torch's current stream).
There is no CPU fallback: if the library is missing or no CUDA device is present the calls
raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libising3d.so")

OK, EINVAL, ENOMEM, ECUDA = 0, -1, -2, -3
CYCLE_01, CYCLE_MIXED, CYCLE_DOUBLE_CB, CYCLE_DOUBLE_CB_MIXED = 0, 1, 2, 3
MEASURE_AUTO, MEASURE_POPCOUNT, MEASURE_TENSOR = 0, 1, 2
VARIANT_AUTO, VARIANT_GENERIC, VARIANT_FUSED, VARIANT_FUSED2, VARIANT_RESIDENT = 0, 1, 2, 3, 4
VARIANT_FUSED3 = 5
VARIANT_ACTIVE = 6

EXPORTED = [
    "ising3d_required_bytes", "ising3d_words_per_replica", "ising3d_init", "ising3d_init_batch",
    "ising3d_init_batch_with_buffer", "ising3d_reset", "ising3d_set_stream", "ising3d_set_variant", "ising3d_set_cycle", "ising3d_set_temperature", "ising3d_init_menger", "ising3d_set_measure_variant",
    "ising3d_measure_variant_name",
    "ising3d_sweep", "ising3d_measure", "ising3d_measure_static", "ising3d_measure_radial", "ising3d_radial_rounding", "ising3d_release_radial", "ising3d_get_state", "ising3d_set_state",
    "ising3d_get_state_device", "ising3d_set_state_device", "ising3d_L", "ising3d_n_rep",
    "ising3d_sweep_count", "ising3d_launch_count", "ising3d_variant_name", "ising3d_cluster_size",
    "ising3d_set_cluster_size", "ising3d_activity", "ising3d_active_stats", "ising3d_set_activity_policy", "ising3d_sync",
    "ising3d_free", "ising3d_last_error",
]


class Ising3DError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("ising3d error %d: %s" % (code, msg))
        self.code = code


class MeasT(C.Structure):
    _fields_ = [("L", C.c_int32), ("n_rep", C.c_int32), ("sweep", C.c_uint64),
                ("n_up", C.POINTER(C.c_uint64)), ("n_broken", C.POINTER(C.c_uint64)),
                ("antipar", C.POINTER(C.c_uint64)), ("C", C.POINTER(C.c_double)),
                ("ell", C.POINTER(C.c_double)), ("c_intercept", C.c_double)]


class RadialT(C.Structure):
    _fields_ = [("L", C.c_int32), ("n_rep", C.c_int32), ("sweep", C.c_uint64),
                ("corr_sum", C.POINTER(C.c_int64)), ("shell", C.POINTER(C.c_uint64)),
                ("C_rad", C.POINTER(C.c_double)), ("S_rad", C.POINTER(C.c_double)),
                ("ell", C.POINTER(C.c_double)), ("c_intercept", C.c_double)]


_lib = None


def load():
    """dlopen libising3d.so; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("libising3d.so is not built: run `python -m paper_2305_12161_b200.build` "
                          "(or __graft_entry__.build()); there is no CPU fallback")
    l = C.CDLL(LIB_PATH)
    vp, u64, u32p, u64p = C.c_void_p, C.c_uint64, C.POINTER(C.c_uint32), C.POINTER(C.c_uint64)
    sig = {
        "ising3d_required_bytes": (C.c_size_t, [C.c_int, C.c_int]),
        "ising3d_words_per_replica": (C.c_size_t, [C.c_int]),
        "ising3d_init": (C.c_int, [C.POINTER(vp), C.c_int, u64]),
        "ising3d_init_batch": (C.c_int, [C.POINTER(vp), C.c_int, C.c_int, u64p]),
        "ising3d_init_batch_with_buffer": (C.c_int, [C.POINTER(vp), C.c_int, C.c_int, u64p, vp,
                                                     C.c_size_t, vp]),
        "ising3d_reset": (C.c_int, [vp]),
        "ising3d_set_stream": (C.c_int, [vp, vp]),
        "ising3d_set_variant": (C.c_int, [vp, C.c_int]),
        "ising3d_set_cycle": (C.c_int, [vp, C.c_int]),
        "ising3d_set_temperature": (C.c_int, [vp, C.c_double]),
        "ising3d_set_measure_variant": (C.c_int, [vp, C.c_int]),
        "ising3d_measure_variant_name": (C.c_char_p, [vp]),
        "ising3d_init_menger": (C.c_int, [vp, C.c_int]),
        "ising3d_sweep": (C.c_int, [vp, u64]),
        "ising3d_measure": (C.c_int, [vp, C.POINTER(MeasT)]),
        "ising3d_measure_radial": (C.c_int, [vp, C.POINTER(RadialT)]),
        "ising3d_measure_static": (C.c_int, [vp, C.c_int, C.c_int, u64p, u64p, vp]),
        "ising3d_radial_rounding": (C.c_int, [vp, C.POINTER(C.c_double)]),
        "ising3d_release_radial": (C.c_int, [vp]),
        "ising3d_get_state": (C.c_int, [vp, vp, C.c_size_t, u64p]),
        "ising3d_set_state": (C.c_int, [vp, vp, C.c_size_t, u64]),
        "ising3d_get_state_device": (C.c_int, [vp, vp, C.c_size_t, u64p]),
        "ising3d_set_state_device": (C.c_int, [vp, vp, C.c_size_t, u64]),
        "ising3d_L": (C.c_int, [vp]),
        "ising3d_n_rep": (C.c_int, [vp]),
        "ising3d_sweep_count": (u64, [vp]),
        "ising3d_launch_count": (u64, [vp]),
        "ising3d_variant_name": (C.c_char_p, [vp]),
        "ising3d_cluster_size": (C.c_int, [vp]),
        "ising3d_set_cluster_size": (C.c_int, [vp, C.c_int]),
        "ising3d_activity": (C.c_int, [vp, u64p, C.POINTER(C.c_double)]),
        "ising3d_active_stats": (C.c_int, [vp, u64p]),
        "ising3d_set_activity_policy": (C.c_int, [vp, u64, C.c_double, C.c_double]),
        "ising3d_sync": (C.c_int, [vp]),
        "ising3d_free": (None, [vp]),
        "ising3d_last_error": (C.c_char_p, []),
    }
    for name, (res, args) in sig.items():
        fn = getattr(l, name)
        fn.restype = res
        fn.argtypes = args
    _lib = l
    return l


def last_error() -> str:
    return load().ising3d_last_error().decode()


def _check(code):
    if code != OK:
        raise Ising3DError(code, last_error())


def required_bytes(L: int, n_rep: int = 1) -> int:
    return int(load().ising3d_required_bytes(L, n_rep))


def words_per_replica(L: int) -> int:
    return int(load().ising3d_words_per_replica(L))


STATIC_MAX_COUNTS = 16384


def measure_static(dev_ptr: int, L: int, n_rep: int = 1, cuda_stream: int = 0):
    """ising3d_measure_static: N_up and A_mu(r) of a packed state already on the device, without a
    handle and without any device allocation (the counters live in an array inside libising3d.so).

    For callers that cannot allocate on the GPU where they measure: all memory belongs to somebody
    else's pool, or a cudaMalloc would stall the other streams.  `dev_ptr` is the device address of
    n_rep * L^3/32 uint32 words in the get_state format.  n_rep * (1 + 3 (L/2+1)) must not exceed
    STATIC_MAX_COUNTS.  Calls share that array: do not let two of them overlap on one GPU.
    """
    nr = L // 2 + 1
    n_up = np.zeros(max(n_rep, 0), dtype=np.uint64)
    antipar = np.zeros((max(n_rep, 0), 3, nr), dtype=np.uint64)
    _check(load().ising3d_measure_static(C.c_void_p(dev_ptr), int(L), int(n_rep),
                                         n_up.ctypes.data_as(C.POINTER(C.c_uint64)),
                                         antipar.ctypes.data_as(C.POINTER(C.c_uint64)), C.c_void_p(cuda_stream)))
    return {"n_up": n_up, "antipar": antipar}


class Ising3D:
    """One handle of the library: `n_rep` lattices of size L^3 advancing together.

    Method names follow the C ABI: sweep, measure, get_state, set_state, reset, free.
    """

    def __init__(self, L: int, seeds, variant: int = VARIANT_AUTO, torch_buffer: bool = True):
        self._l = load()
        self._h = C.c_void_p()
        if isinstance(seeds, (int, np.integer)):
            seeds = [int(seeds)]
        self.seeds = [int(s) for s in seeds]
        self.L, self.n_rep = int(L), len(self.seeds)
        arr = (C.c_uint64 * self.n_rep)(*self.seeds)
        self._buf = None
        if torch_buffer:
            import torch
            if not torch.cuda.is_available():
                raise Ising3DError(ECUDA, "no CUDA device (there is no CPU fallback)")
            nbytes = self._l.ising3d_required_bytes(self.L, self.n_rep)
            if nbytes == 0:
                raise Ising3DError(EINVAL, "L must be a multiple of 64 in [64, 4096] and n_rep >= 1")
            self._buf = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
            stream = torch.cuda.current_stream().cuda_stream
            _check(self._l.ising3d_init_batch_with_buffer(
                C.byref(self._h), self.L, self.n_rep, arr, C.c_void_p(self._buf.data_ptr()),
                nbytes, C.c_void_p(stream)))
        else:
            _check(self._l.ising3d_init_batch(C.byref(self._h), self.L, self.n_rep, arr))
        if variant != VARIANT_AUTO:
            self.set_variant(variant)

    # -- life cycle ----------------------------------------------------
    def free(self):
        if getattr(self, "_h", None) and self._h.value:
            self._l.ising3d_free(self._h)
            self._h = C.c_void_p()
            self._buf = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.free()

    # -- control -------------------------------------------------------
    def set_stream(self, cuda_stream: int):
        _check(self._l.ising3d_set_stream(self._h, C.c_void_p(cuda_stream)))

    def set_variant(self, variant: int):
        _check(self._l.ising3d_set_variant(self._h, variant))

    def set_cluster_size(self, cs: int):
        _check(self._l.ising3d_set_cluster_size(self._h, int(cs)))

    def set_activity_policy(self, probe_interval: int, on_below: float = 0.11, off_above: float = 0.14):
        _check(self._l.ising3d_set_activity_policy(self._h, int(probe_interval), float(on_below), float(off_above)))

    def activity(self):
        """(awake_groups [n_rep][2], fraction): groups holding a site with Delta E <= 0."""
        out = np.zeros((self.n_rep, 2), dtype=np.uint64)
        frac = C.c_double()
        _check(self._l.ising3d_activity(self._h, out.ctypes.data_as(C.POINTER(C.c_uint64)), C.byref(frac)))
        return out, float(frac.value)

    def active_stats(self) -> np.ndarray:
        """[n_rep][2]: groups evaluated / changed by the activity-driven kernel since the last call."""
        out = np.zeros((self.n_rep, 2), dtype=np.uint64)
        _check(self._l.ising3d_active_stats(self._h, out.ctypes.data_as(C.POINTER(C.c_uint64))))
        return out

    @property
    def last_activity(self) -> float:
        frac = C.c_double()
        _check(self._l.ising3d_activity(self._h, None, C.byref(frac)))
        return float(frac.value)

    def set_measure_variant(self, variant: int):
        _check(self._l.ising3d_set_measure_variant(self._h, variant))

    @property
    def measure_variant_name(self) -> str:
        return self._l.ising3d_measure_variant_name(self._h).decode()

    def set_temperature(self, T: float):
        _check(self._l.ising3d_set_temperature(self._h, float(T)))

    def set_cycle(self, cycle: int):
        _check(self._l.ising3d_set_cycle(self._h, cycle))

    def init_menger(self, k: int):
        _check(self._l.ising3d_init_menger(self._h, int(k)))

    def reset(self):
        _check(self._l.ising3d_reset(self._h))

    def sync(self):
        _check(self._l.ising3d_sync(self._h))

    @property
    def sweep_count(self) -> int:
        return int(self._l.ising3d_sweep_count(self._h))

    @property
    def launch_count(self) -> int:
        return int(self._l.ising3d_launch_count(self._h))

    @property
    def cluster_size(self) -> int:
        return int(self._l.ising3d_cluster_size(self._h))

    @property
    def variant_name(self) -> str:
        return self._l.ising3d_variant_name(self._h).decode()

    # -- the path ------------------------------------------------------
    def sweep(self, n_sweeps: int = 1):
        _check(self._l.ising3d_sweep(self._h, int(n_sweeps)))

    def measure(self, c_intercept: float = 0.5):
        nr = self.L // 2 + 1
        n_up = np.zeros(self.n_rep, dtype=np.uint64)
        n_broken = np.zeros(self.n_rep, dtype=np.uint64)
        antipar = np.zeros((self.n_rep, 3, nr), dtype=np.uint64)
        Cr = np.zeros((self.n_rep, nr), dtype=np.float64)
        ell = np.zeros(self.n_rep, dtype=np.float64)
        m = MeasT(self.L, self.n_rep, 0,
                  n_up.ctypes.data_as(C.POINTER(C.c_uint64)),
                  n_broken.ctypes.data_as(C.POINTER(C.c_uint64)),
                  antipar.ctypes.data_as(C.POINTER(C.c_uint64)),
                  Cr.ctypes.data_as(C.POINTER(C.c_double)),
                  ell.ctypes.data_as(C.POINTER(C.c_double)), float(c_intercept))
        _check(self._l.ising3d_measure(self._h, C.byref(m)))
        return {"sweep": int(m.sweep), "n_up": n_up, "n_broken": n_broken, "antipar": antipar,
                "C": Cr, "ell": ell}

    def measure_radial(self, c_intercept: float = 0.5):
        nb = self.L // 2 + 1
        corr = np.zeros((self.n_rep, nb), dtype=np.int64)
        shell = np.zeros(nb, dtype=np.uint64)
        Cr = np.zeros((self.n_rep, nb), dtype=np.float64)
        Sr = np.zeros((self.n_rep, nb), dtype=np.float64)
        ell = np.zeros(self.n_rep, dtype=np.float64)
        m = RadialT(self.L, self.n_rep, 0, corr.ctypes.data_as(C.POINTER(C.c_int64)),
                    shell.ctypes.data_as(C.POINTER(C.c_uint64)), Cr.ctypes.data_as(C.POINTER(C.c_double)),
                    Sr.ctypes.data_as(C.POINTER(C.c_double)), ell.ctypes.data_as(C.POINTER(C.c_double)),
                    float(c_intercept))
        _check(self._l.ising3d_measure_radial(self._h, C.byref(m)))
        return {"sweep": int(m.sweep), "corr_sum": corr, "shell": shell, "C_rad": Cr, "S_rad": Sr, "ell": ell}

    @property
    def radial_rounding(self) -> float:
        """max |v/N - round(v/N)| of the last measure_radial call (exactness margin, D12)."""
        d = C.c_double()
        _check(self._l.ising3d_radial_rounding(self._h, C.byref(d)))
        return float(d.value)

    def release_radial(self):
        _check(self._l.ising3d_release_radial(self._h))

    def get_state(self, out: np.ndarray | None = None) -> np.ndarray:
        n = self.n_rep * self.L ** 3 // 32
        if out is None:
            out = np.empty(n, dtype=np.uint32)
        assert out.dtype == np.uint32 and out.size == n and out.flags.c_contiguous
        sw = C.c_uint64()
        _check(self._l.ising3d_get_state(self._h, C.c_void_p(out.ctypes.data), n, C.byref(sw)))
        return out

    def set_state(self, words: np.ndarray, sweep: int):
        w = np.ascontiguousarray(words, dtype=np.uint32)
        _check(self._l.ising3d_set_state(self._h, C.c_void_p(w.ctypes.data), w.size, int(sweep)))

    def set_state_ptr(self, host_ptr: int, n_words: int, sweep: int):
        """set_state from a raw (e.g. pinned) host pointer."""
        _check(self._l.ising3d_set_state(self._h, C.c_void_p(host_ptr), n_words, int(sweep)))

    def get_state_device(self, dev_ptr: int, n_words: int):
        sw = C.c_uint64()
        _check(self._l.ising3d_get_state_device(self._h, C.c_void_p(dev_ptr), n_words, C.byref(sw)))
        return int(sw.value)

    def set_state_device(self, dev_ptr: int, n_words: int, sweep: int):
        _check(self._l.ising3d_set_state_device(self._h, C.c_void_p(dev_ptr), n_words, int(sweep)))
