"""Seeded synthetic inputs and workload presets.

This module holds NO arithmetic of the method (no site rule, no Philox, no
measurement): only (i) seeded numpy generators of spin configurations,
(ii) hand-built structured configurations used as test inputs, (iii) the
canonical packed format D3 (the boundary's data format, include/ising3d.h),
and (iv) the five workloads of BASELINE.json with their measurement times.
It is the one module both the CUDA-path tests and the oracle tests import.

The paper uses no dataset: every run starts from "random spin configurations
(with magnetization m ~ 0)", so the synthetic workloads ARE the
paper's workloads: iid +-1, p = 1/2.  The T = infinity start proper is drawn by
each side's own Philox (D6); the numpy generators here only serve
set_state / import tests that need an arbitrary state.
"""
from __future__ import annotations

import numpy as np

# ----------------------------------------------------------------------
# Workloads (BASELINE.json "configs")
# ----------------------------------------------------------------------


def measurement_times(n: int):
    """Log-spaced integer times T(n) = {m*10^d <= n : m in {1,2,3,4,5,6,8}} U {n}  (S12)."""
    ts = set()
    d = 1
    while d <= n:
        for m in (1, 2, 3, 4, 5, 6, 8):
            if m * d <= n:
                ts.add(m * d)
        d *= 10
    ts.add(n)
    return sorted(ts)


WORKLOADS = {
    # name: L, seeds, sweeps, measurement times
    "config1_L64": dict(L=64, seeds=[1], sweeps=100, times=[1, 2, 5, 10, 20, 50, 100]),
    "config2_L256": dict(L=256, seeds=[2], sweeps=2000, times=measurement_times(2000)),
    "config3_64xL128": dict(L=128, seeds=list(range(100, 164)), sweeps=10_000,
                            times=measurement_times(10_000)),
    "config4_L1024": dict(L=1024, seeds=[3], sweeps=100_000, times=measurement_times(100_000)),
    "config5_L2048": dict(L=2048, seeds=[4], sweeps=300_000, times=measurement_times(300_000),
                          throughput_window=1000),
}

# ----------------------------------------------------------------------
# D3: canonical packed format  (spins[z][y][x] int8 +-1  <->  uint32 words)
# ----------------------------------------------------------------------


def words_per_colour(L: int) -> int:
    return (L ** 3 // 2 + 31) // 32


def pack_spins(spins: np.ndarray) -> np.ndarray:
    """int8 spins[z][y][x] in {-1,+1} -> uint32 words (colour 0 words, then colour 1)."""
    L = spins.shape[0]
    assert spins.shape == (L, L, L) and L % 2 == 0
    z, y, x = np.meshgrid(np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    c = (x + y + z) & 1
    b = (z.astype(np.int64) * L + y) * (L // 2) + (x >> 1)
    wpc = words_per_colour(L)
    bits = np.zeros((2, wpc * 32), dtype=np.uint8)
    bits[c.ravel(), b.ravel()] = (spins.ravel() == 1).astype(np.uint8)
    # little-endian bit order inside each 32-bit word
    by = np.packbits(bits.reshape(2, wpc * 4, 8), axis=-1, bitorder="little").reshape(2, wpc, 4)
    words = (by[..., 0].astype(np.uint32) | (by[..., 1].astype(np.uint32) << 8)
             | (by[..., 2].astype(np.uint32) << 16) | (by[..., 3].astype(np.uint32) << 24))
    return np.ascontiguousarray(words.reshape(-1))


def unpack_words(words: np.ndarray, L: int) -> np.ndarray:
    """Inverse of pack_spins."""
    wpc = words_per_colour(L)
    w = np.asarray(words, dtype=np.uint32).reshape(2, wpc)
    by = np.stack([(w >> s) & 0xFF for s in (0, 8, 16, 24)], axis=-1).astype(np.uint8)
    bits = np.unpackbits(by.reshape(2, wpc * 4, 1), axis=-1, bitorder="little").reshape(2, wpc * 32)
    z, y, x = np.meshgrid(np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    c = (x + y + z) & 1
    b = (z.astype(np.int64) * L + y) * (L // 2) + (x >> 1)
    up = bits[c, b]
    return np.where(up == 1, 1, -1).astype(np.int8)


# ----------------------------------------------------------------------
# seeded random states (numpy PCG64) -- for set_state / import tests
# ----------------------------------------------------------------------


def random_spins(L: int, seed: int, p_up: float = 0.5) -> np.ndarray:
    rng = np.random.Generator(np.random.PCG64(seed))
    return np.where(rng.random((L, L, L)) < p_up, 1, -1).astype(np.int8)


def random_words(L: int, n_rep: int, seed: int) -> np.ndarray:
    """Packed iid p=1/2 state of n_rep replicas (uint32 [n_rep * L^3/32])."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = n_rep * (L ** 3 // 32)
    return rng.integers(0, 2 ** 32, size=n, dtype=np.uint64).astype(np.uint32)


def coarse_words(L: int, seed: int, block: int = 8) -> np.ndarray:
    """A domain-like state (iid signs on block^3 cubes, then 3 % of sites flipped):
    fewer ties and long runs of equal bits, as late in a quench."""
    rng = np.random.Generator(np.random.PCG64(seed))
    nb = L // block
    coarse = np.where(rng.random((nb, nb, nb)) < 0.5, 1, -1).astype(np.int8)
    s = np.kron(coarse, np.ones((block, block, block), dtype=np.int8))
    flip = rng.random((L, L, L)) < 0.03
    s = np.where(flip, -s, s).astype(np.int8)
    return pack_spins(s)


def domain_spins(L: int, seed: int, block: int = 16, p_minority: float = 0.15, noise: float = 0.0) -> np.ndarray:
    """A late-time-like state as int8 spins: a +1 background in which a fraction p_minority of
    the block^3 cubes is -1 (large uniform regions, activity only at the cube edges and
    corners), optionally with a fraction `noise` of the sites flipped."""
    rng = np.random.Generator(np.random.PCG64(seed))
    nb = L // block
    coarse = np.where(rng.random((nb, nb, nb)) < p_minority, -1, 1).astype(np.int8)
    s = np.kron(coarse, np.ones((block, block, block), dtype=np.int8))
    if noise > 0.0:
        s = np.where(rng.random((L, L, L)) < noise, -s, s).astype(np.int8)
    return s


# ----------------------------------------------------------------------
# structured configurations (closed-form test inputs)
# ----------------------------------------------------------------------


def all_up(L: int) -> np.ndarray:
    return np.ones((L, L, L), dtype=np.int8)


def neel(L: int) -> np.ndarray:
    z, y, x = np.meshgrid(np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    return np.where(((x + y + z) & 1) == 0, 1, -1).astype(np.int8)


def slab(L: int, axis: int, start: int, thickness: int) -> np.ndarray:
    """-1 everywhere except +1 for `thickness` planes from `start` (periodic) normal to
    `axis` (0 = x, 1 = y, 2 = z)."""
    s = -np.ones((L, L, L), dtype=np.int8)
    idx = [(start + i) % L for i in range(thickness)]
    if axis == 0:
        s[:, :, idx] = 1
    elif axis == 1:
        s[:, idx, :] = 1
    else:
        s[idx, :, :] = 1
    return s


def single_spin(L: int, x: int, y: int, z: int) -> np.ndarray:
    s = np.ones((L, L, L), dtype=np.int8)
    s[z % L, y % L, x % L] = -1
    return s


def cube(L: int, x0: int, y0: int, z0: int, edge: int = 2) -> np.ndarray:
    """+1 background with an edge^3 cube of -1 at (x0,y0,z0), periodic wrap."""
    s = np.ones((L, L, L), dtype=np.int8)
    for dz in range(edge):
        for dy in range(edge):
            for dx in range(edge):
                s[(z0 + dz) % L, (y0 + dy) % L, (x0 + dx) % L] = -1
    return s
