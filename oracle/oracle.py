"""ctypes front end of the CPU oracle (oracle/ising_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / --impl reference leg may import this module.
It imports nothing from paper_2305_12161_b200 and the CUDA path imports
nothing from here.

What each call computes and which passage of the paper it follows is stated in
ising_oracle.c next to the function of the same name (eq. (6),
PAPER.md:116 sweep order, eq. (2), PAPER.md:51 ell).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ising_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")


def build(force: bool = False) -> str:
    """Compile ising_oracle.c with gcc (-O2, OpenMP over z-planes only)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    tmp = _LIB + ".tmp.%d" % os.getpid()
    cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
    subprocess.check_call(cmd)
    os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        l = C.CDLL(build())
        u32p = C.POINTER(C.c_uint32)
        u64p = C.POINTER(C.c_uint64)
        i32p = C.POINTER(C.c_int32)
        dp = C.POINTER(C.c_double)
        l.orc_philox4x32_10.argtypes = [u32p, u32p, u32p]
        l.orc_philox4x32_10.restype = None
        l.orc_create.argtypes = [C.c_int, C.c_uint64]
        l.orc_create.restype = C.c_void_p
        l.orc_free.argtypes = [C.c_void_p]
        l.orc_free.restype = None
        l.orc_spins.argtypes = [C.c_void_p]
        l.orc_spins.restype = C.POINTER(C.c_int8)
        l.orc_get_sweep.argtypes = [C.c_void_p]
        l.orc_get_sweep.restype = C.c_uint32
        l.orc_set_sweep.argtypes = [C.c_void_p, C.c_uint32]
        l.orc_set_sweep.restype = None
        l.orc_set_seed.argtypes = [C.c_void_p, C.c_uint64]
        l.orc_set_seed.restype = None
        l.orc_site_bit.argtypes = [C.c_uint64, C.c_int, C.c_int, C.c_int, C.c_int,
                                   C.c_uint32, C.c_uint32]
        l.orc_site_bit.restype = C.c_int
        l.orc_init_random.argtypes = [C.c_void_p]
        l.orc_init_random.restype = None
        l.orc_half_sweep.argtypes = [C.c_void_p, C.c_uint32, C.c_int, C.c_int, C.c_uint64]
        l.orc_half_sweep.restype = None
        l.orc_sweep.argtypes = [C.c_void_p, C.c_uint64]
        l.orc_sweep.restype = None
        l.orc_energy.argtypes = [C.c_void_p]
        l.orc_energy.restype = C.c_int64
        l.orc_half_sweep_brute.argtypes = [C.c_void_p, C.c_uint32, C.c_int]
        l.orc_half_sweep_brute.restype = None
        l.orc_sweep_brute.argtypes = [C.c_void_p, C.c_uint64]
        l.orc_sweep_brute.restype = None
        l.orc_measure.argtypes = [C.c_void_p, i32p, C.c_int, u64p, u64p]
        l.orc_measure.restype = None
        l.orc_postprocess.argtypes = [C.c_int, C.c_uint64, u64p, C.c_double, dp, dp, dp]
        l.orc_postprocess.restype = None
        l.orc_words_per_colour.argtypes = [C.c_int]
        l.orc_words_per_colour.restype = C.c_size_t
        l.orc_export.argtypes = [C.c_void_p, u32p]
        l.orc_export.restype = None
        l.orc_import.argtypes = [C.c_void_p, u32p, C.c_uint32]
        l.orc_import.restype = None
        l.orc_sites_after.argtypes = [C.c_uint64, C.c_int, i32p, C.c_int, C.c_int,
                                      C.POINTER(C.c_int8)]
        l.orc_sites_after.restype = None
        l.orc_activity.argtypes = [C.c_void_p, u64p]
        l.orc_activity.restype = None
        l.orc_first_colour.argtypes = [C.c_uint64, C.c_uint32]
        l.orc_first_colour.restype = C.c_int
        l.orc_sweep_mixed.argtypes = [C.c_void_p, C.c_uint64]
        l.orc_sweep_mixed.restype = None
        l.orc_menger_solid.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int]
        l.orc_menger_solid.restype = C.c_int
        l.orc_init_menger.argtypes = [C.c_void_p, C.c_int]
        l.orc_init_menger.restype = None
        l.orc_menger_site.argtypes = [C.c_uint64, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int]
        l.orc_menger_site.restype = C.c_int
        i64p = C.POINTER(C.c_int64)
        l.orc_radial_bin.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int]
        l.orc_radial_bin.restype = C.c_int
        l.orc_corr_direct.argtypes = [C.c_void_p, i64p]
        l.orc_corr_direct.restype = None
        l.orc_radial_sums.argtypes = [C.c_int, i64p, i64p, u64p]
        l.orc_radial_sums.restype = None
        l.orc_half_sweep_dcb.argtypes = [C.c_void_p, C.c_uint32, C.c_int, C.c_int, C.c_int]
        l.orc_half_sweep_dcb.restype = None
        l.orc_sweep_dcb.argtypes = [C.c_void_p, C.c_uint64, C.c_int]
        l.orc_sweep_dcb.restype = None
        l.orc_block_first_fine.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32]
        l.orc_block_first_fine.restype = C.c_int
        l.orc_pass_dcb_mixed.argtypes = [C.c_void_p, C.c_uint32, C.c_int, C.c_int, C.c_int]
        l.orc_pass_dcb_mixed.restype = None
        l.orc_sweep_dcb_mixed.argtypes = [C.c_void_p, C.c_uint64, C.c_int]
        l.orc_sweep_dcb_mixed.restype = None
        l.orc_glauber_thresholds.argtypes = [C.c_double, u64p]
        l.orc_glauber_thresholds.restype = None
        l.orc_site_uniform.argtypes = [C.c_uint64, C.c_int, C.c_int, C.c_int, C.c_int, C.c_uint32]
        l.orc_site_uniform.restype = C.c_uint32
        l.orc_sweep_T.argtypes = [C.c_void_p, C.c_uint64, C.c_double]
        l.orc_sweep_T.restype = None
        l.orc_half_sweep_T.argtypes = [C.c_void_p, C.c_uint32, C.c_int, u64p]
        l.orc_half_sweep_T.restype = None
        l.orc_num_threads.argtypes = []
        l.orc_num_threads.restype = C.c_int
        l.orc_set_num_threads.argtypes = [C.c_int]
        l.orc_set_num_threads.restype = None
        _lib = l
    return _lib


def _p(a, ty):
    return a.ctypes.data_as(C.POINTER(ty))


def philox4x32_10(ctr, key):
    """D5.  ctr: 4 uint32, key: 2 uint32 -> 4 uint32 (numpy)."""
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32))
    return out


def site_bit(seed, L, x, y, z, t, tag):
    return int(lib().orc_site_bit(int(seed), L, x, y, z, t, tag))


def sites_after(seed, L, xyz, n_half_sweeps):
    """Spins (+-1) of the sampled sites xyz[n][3] after n_half_sweeps half-sweeps from the
    T = infinity start of `seed`, each computed from the definition by light-cone recursion."""
    a = np.ascontiguousarray(xyz, dtype=np.int32).reshape(-1, 3)
    out = np.zeros(len(a), dtype=np.int8)
    lib().orc_sites_after(int(seed), int(L), _p(a, C.c_int32), len(a), int(n_half_sweeps),
                          _p(out, C.c_int8))
    return out


def first_colour(seed: int, t: int) -> int:
    """Mixed cycle (D10): the colour updated first in sweep t."""
    return int(lib().orc_first_colour(int(seed), int(t)))


def menger_solid(u: int, v: int, w: int, k: int) -> int:
    """1 iff (u,v,w) in [0,3^k)^3 belongs to the k-th iteration Menger sponge."""
    return int(lib().orc_menger_solid(int(u), int(v), int(w), int(k)))


def menger_site(seed: int, L: int, k: int, x: int, y: int, z: int) -> int:
    """Spin (+-1) of site (x,y,z) in the Menger start of iteration k (D11), one site at a time."""
    return int(lib().orc_menger_site(int(seed), int(L), int(k), int(x), int(y), int(z)))


def radial_bin(L: int, dx: int, dy: int, dz: int) -> int:
    """D12: bin of the displacement (dx,dy,dz) in [0,L)^3 (minimal image, nearest integer to |d|)."""
    return int(lib().orc_radial_bin(int(L), int(dx), int(dy), int(dz)))


def radial_sums(L: int, field: np.ndarray):
    """Sums of an int64 field[dz][dy][dx] over the radial bins 0..L/2 and the bin populations."""
    f = np.ascontiguousarray(field, dtype=np.int64)
    assert f.shape == (L, L, L)
    s = np.zeros(L // 2 + 1, dtype=np.int64)
    n = np.zeros(L // 2 + 1, dtype=np.uint64)
    lib().orc_radial_sums(int(L), _p(f, C.c_int64), _p(s, C.c_int64), _p(n, C.c_uint64))
    return s, n


def block_first_fine(seed: int, t: int, block_index: int) -> int:
    """D15: the fine colour a block updates first in sweep t (mixed-cycle double checkerboard)."""
    return int(lib().orc_block_first_fine(int(seed), int(t), int(block_index)))


def glauber_thresholds(T: float) -> np.ndarray:
    """D13: thr[n] = floor(2^32 / (1 + exp((12 - 4n)/T))), n = 0..6 antiparallel neighbours."""
    thr = np.zeros(7, dtype=np.uint64)
    lib().orc_glauber_thresholds(float(T), _p(thr, C.c_uint64))
    return thr


def site_uniform(seed: int, L: int, x: int, y: int, z: int, t: int) -> int:
    """D13: the site's 32-bit uniform of sweep t (Philox bit planes, tags 4..35)."""
    return int(lib().orc_site_uniform(int(seed), int(L), int(x), int(y), int(z), int(t)))


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(n: int) -> None:
    lib().orc_set_num_threads(int(n))


def postprocess(L, n_up, antipar, c_intercept=0.5):
    """D9.  antipar: uint64 [3][L/2+1].  Returns (m, C[L/2+1], ell)."""
    nr = L // 2 + 1
    a = np.ascontiguousarray(antipar, dtype=np.uint64).reshape(3, nr)
    Cr = np.zeros(nr, dtype=np.float64)
    m = C.c_double()
    ell = C.c_double()
    lib().orc_postprocess(L, int(n_up), _p(a, C.c_uint64), float(c_intercept),
                          C.byref(m), _p(Cr, C.c_double), C.byref(ell))
    return m.value, Cr, ell.value


def _bins_numpy(L: int) -> np.ndarray:
    """D12 bins of all displacements [dz][dy][dx], vectorised (same integer rule as orc_radial_bin)."""
    d = np.arange(L, dtype=np.int64)
    d = np.where(d > L // 2, d - L, d)
    n4 = 4 * (d[:, None, None] ** 2 + d[None, :, None] ** 2 + d[None, None, :] ** 2)
    b = np.floor((np.sqrt(n4.astype(np.float64)) + 1.0) / 2.0).astype(np.int64)
    b = np.where((2 * b + 1) ** 2 <= n4, b + 1, b)          # integer fix-up of the float guess
    b = np.where((b > 0) & ((2 * b - 1) ** 2 > n4), b - 1, b)
    return b


class Oracle:
    """One lattice of the CPU oracle (int8 per spin)."""

    def __init__(self, L: int, seed: int, init: bool = True):
        self._l = lib()
        self.L = int(L)
        self.seed = int(seed)
        self._h = self._l.orc_create(self.L, self.seed)
        if not self._h:
            raise ValueError("oracle: L must be even and >= 4 (D1)")
        if init:
            self._l.orc_init_random(self._h)

    def close(self):
        if getattr(self, "_h", None):
            self._l.orc_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- state ---------------------------------------------------------
    @property
    def spins(self) -> np.ndarray:
        """View [z][y][x] of the int8 spins (writable, no copy)."""
        n = self.L ** 3
        buf = (C.c_int8 * n).from_address(C.addressof(self._l.orc_spins(self._h).contents))
        buf._owner = self          # the view keeps the lattice alive
        return np.frombuffer(buf, dtype=np.int8).reshape(self.L, self.L, self.L)

    @property
    def sweep_count(self) -> int:
        return int(self._l.orc_get_sweep(self._h))

    @sweep_count.setter
    def sweep_count(self, t: int):
        self._l.orc_set_sweep(self._h, int(t))

    def set_seed(self, seed: int):
        self.seed = int(seed)
        self._l.orc_set_seed(self._h, self.seed)

    def init_random(self):
        self._l.orc_init_random(self._h)

    # -- dynamics ------------------------------------------------------
    def half_sweep(self, t: int, c: int, order: int = 0, order_seed: int = 0):
        self._l.orc_half_sweep(self._h, int(t), int(c), int(order), int(order_seed))

    def sweep(self, n: int = 1):
        self._l.orc_sweep(self._h, int(n))

    # -- the paper's estimator: full correlation matrix + radial average (8(f)-1, D12) --------
    def corr_direct(self) -> np.ndarray:
        """P(d) = sum_i s_i s_{i+d} for every d, from the definition (O(N^2): L <= 32)."""
        L = self.L
        out = np.zeros((L, L, L), dtype=np.int64)
        self._l.orc_corr_direct(self._h, _p(out, C.c_int64))
        return out

    def corr_fft(self) -> np.ndarray:
        """The same integers by eq. (7): F^-1(|F s|^2) in fp64 (numpy), rounded to
        the nearest integer (the error of the fp64 transforms is < 1e-3 for L <= 512)."""
        s = self.spins.astype(np.float64)
        p = np.fft.irfftn(np.abs(np.fft.rfftn(s)) ** 2, s=s.shape, axes=(0, 1, 2))
        return np.rint(p).astype(np.int64)

    def power_spectrum(self) -> np.ndarray:
        """|F s|^2 on the full k grid [kz][ky][kx] (fp64)."""
        return np.abs(np.fft.fftn(self.spins.astype(np.float64))) ** 2

    def measure_radial(self, c_intercept: float = 0.5, direct: bool = False):
        """D12: radially averaged C(r) (eq. (2) with the paper's estimator), shell populations,
        radially averaged structure factor S(k) = |F s|^2 / N over the same bins in index space,
        and ell from C_rad = c (D9 interpolation rule)."""
        L = self.L
        N = L ** 3
        P = self.corr_direct() if direct else self.corr_fft()
        sums, cnt = radial_sums(L, P)
        m = float(self.spins.astype(np.int64).sum()) / N
        C_rad = sums.astype(np.float64) / (float(N) * cnt.astype(np.float64)) - m * m
        ps = self.power_spectrum()
        nb = L // 2 + 1
        S_sum = np.zeros(nb)
        idx = np.arange(L)
        bins = np.array([[[radial_bin(L, int(a), int(b), int(c)) for a in idx] for b in idx] for c in idx]) \
            if L <= 16 else _bins_numpy(L)
        for b in range(nb):
            S_sum[b] = ps[bins == b].sum()
        S_rad = S_sum / (float(N) * cnt.astype(np.float64))
        ell = float("nan")
        for r in range(nb - 1):
            if C_rad[r] >= c_intercept and C_rad[r + 1] < c_intercept:
                ell = r + (C_rad[r] - c_intercept) / (C_rad[r] - C_rad[r + 1])
                break
        return {"corr_sum": sums, "shell": cnt, "C_rad": C_rad, "S_rad": S_rad, "ell": ell, "m": m}

    def sweep_dcb(self, n: int = 1, block: int = 8):
        """n sweeps of the double-checkerboard 01 cycle (Supp. I.A, D14), block edge `block`."""
        assert self.L % (2 * block) == 0 or block >= self.L
        self._l.orc_sweep_dcb(self._h, int(n), int(block))

    def half_sweep_dcb(self, t: int, coarse: int, fine: int, block: int = 8):
        self._l.orc_half_sweep_dcb(self._h, int(t), int(coarse), int(fine), int(block))

    def sweep_dcb_mixed(self, n: int = 1, block: int = 8):
        """n sweeps of the mixed-cycle double checkerboard (Supp. I.B, D15)."""
        assert self.L % (2 * block) == 0
        self._l.orc_sweep_dcb_mixed(self._h, int(n), int(block))

    def pass_dcb_mixed(self, t: int, coarse: int, pas: int, block: int = 8):
        self._l.orc_pass_dcb_mixed(self._h, int(t), int(coarse), int(pas), int(block))

    def sweep_T(self, n: int, T: float):
        """n sweeps of finite-temperature Glauber dynamics (eq. (5), D13)."""
        self._l.orc_sweep_T(self._h, int(n), float(T))

    def half_sweep_T(self, t: int, c: int, T: float):
        thr = glauber_thresholds(T)
        self._l.orc_half_sweep_T(self._h, int(t), int(c), _p(thr, C.c_uint64))

    def activity(self) -> np.ndarray:
        """[2]: groups of each colour holding a site with Delta E <= 0 (eq. (6))."""
        out = np.zeros(2, dtype=np.uint64)
        self._l.orc_activity(self._h, _p(out, C.c_uint64))
        return out

    def sweep_mixed(self, n: int = 1):
        """n sweeps of the mixed cycle (D10): the first colour is drawn per sweep."""
        self._l.orc_sweep_mixed(self._h, int(n))

    def init_menger(self, k: int):
        """Menger-sponge start of iteration k (D11); sweep counter 0."""
        self._l.orc_init_menger(self._h, int(k))

    def half_sweep_brute(self, t: int, c: int):
        self._l.orc_half_sweep_brute(self._h, int(t), int(c))

    def sweep_brute(self, n: int = 1):
        self._l.orc_sweep_brute(self._h, int(n))

    def energy(self) -> int:
        return int(self._l.orc_energy(self._h))

    # -- measurements --------------------------------------------------
    def measure(self, r_list=None):
        """D8.  Returns (n_up, antipar[3][len(r_list)]); r_list defaults to 0..L/2."""
        if r_list is None:
            r_list = np.arange(self.L // 2 + 1, dtype=np.int32)
        r = np.ascontiguousarray(r_list, dtype=np.int32)
        a = np.zeros((3, len(r)), dtype=np.uint64)
        n_up = C.c_uint64()
        self._l.orc_measure(self._h, _p(r, C.c_int32), len(r), C.byref(n_up), _p(a, C.c_uint64))
        return int(n_up.value), a

    def measure_full(self, c_intercept: float = 0.5):
        """D8 + D9 over all r: dict with n_up, n_broken, antipar, m, C, ell."""
        n_up, a = self.measure()
        m, Cr, ell = postprocess(self.L, n_up, a, c_intercept)
        return {"n_up": n_up, "n_broken": int(a[0, 1] + a[1, 1] + a[2, 1]),
                "antipar": a, "m": m, "C": Cr, "ell": ell, "sweep": self.sweep_count}

    # -- D3 packed layout ---------------------------------------------
    def words_per_colour(self) -> int:
        return int(self._l.orc_words_per_colour(self.L))

    def export_words(self) -> np.ndarray:
        w = np.zeros(2 * self.words_per_colour(), dtype=np.uint32)
        self._l.orc_export(self._h, _p(w, C.c_uint32))
        return w

    def import_words(self, words, sweep: int):
        w = np.ascontiguousarray(words, dtype=np.uint32)
        assert w.size == 2 * self.words_per_colour()
        self._l.orc_import(self._h, _p(w, C.c_uint32), int(sweep))


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
