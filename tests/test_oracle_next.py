"""Pins of the oracle functions behind the SURVEY.md 8(f) rows built so far:
  f-2  mixed cycle (Supp. I.B PAPER.md:258)  -> orc_first_colour, orc_sweep_mixed
  f-3  Menger-sponge start     -> orc_menger_solid, orc_init_menger
Each pin is something the paper or the mathematics fixes, not a retyping of the oracle."""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_2305_12161_b200 import inputs
from test_oracle_pins import py_philox, MASK


# ------------------------------------------------------------------ f-2: mixed cycle
def test_first_colour_is_the_documented_philox_bit():
    """D10: bit 0 of word 0 of Philox(key = seed, counter = (0, t, 0, 2)), against the
    big-integer Python Philox (itself pinned by the known-answer vectors)."""
    for seed in (1, 4, 0xDEADBEEFCAFE1234):
        for t in list(range(40)) + [2 ** 31, 2 ** 32 - 2]:
            want = py_philox([0, t, 0, 2], [seed & MASK, seed >> 32])[0] & 1
            assert orc.first_colour(seed, t) == want


def test_mixed_cycle_neel_closed_form():
    """From the Neel state s = (-1)^(x+y+z) the colour updated first flips completely (n = 6)
    and the lattice orders with the OTHER colour's value (pinned for the
    fixed order in test_oracle_pins): black first -> all -1, white first -> all +1.  So one
    mixed sweep from the Neel state reads out the order the oracle really used."""
    L, seed = 8, 11
    seen = set()
    for t in range(48):
        o = orc.Oracle(L, seed, init=False)
        o.spins[...] = inputs.neel(L)
        o.sweep_count = t
        o.sweep_mixed(1)
        first = py_philox([0, t, 0, 2], [seed & MASK, seed >> 32])[0] & 1
        assert np.all(o.spins == (1 if first else -1)), "sweep %d" % t
        assert o.sweep_count == t + 1
        seen.add(first)
    assert seen == {0, 1}


def test_mixed_cycle_order_is_fair_and_seed_dependent():
    n = 4000
    f1 = np.array([orc.first_colour(5, t) for t in range(n)])
    f2 = np.array([orc.first_colour(6, t) for t in range(n)])
    assert abs(f1.sum() - n / 2) < 4 * np.sqrt(n) / 2          # binomial 4 sigma
    assert abs((f1 != f2).sum() - n / 2) < 4 * np.sqrt(n) / 2  # independent streams


def test_mixed_cycle_every_site_proposed_once_and_energy_monotone():
    """PAPER.md:258 "still every spin is proposed to flip exactly once per sweep": a mixed
    sweep equals the two half-sweeps of the drawn order, the interface energy never increases
    (each half-sweep only accepts Delta E <= 0), and a sweep whose drawn order is (0, 1) equals
    the 01-cycle sweep."""
    L, seed = 12, 3
    a = orc.Oracle(L, seed)
    b = orc.Oracle(L, seed)
    c = orc.Oracle(L, seed)
    e_prev = a.measure([1])[1].sum()
    for t in range(12):
        first = orc.first_colour(seed, t)
        state_before = a.spins.copy()
        a.sweep_mixed(1)
        b.half_sweep(t, first)
        b.half_sweep(t, 1 - first)
        assert np.array_equal(a.spins, b.spins)
        e = a.measure([1])[1].sum()
        assert e <= e_prev
        e_prev = e
        c.spins[...] = state_before
        c.sweep_count = t
        c.sweep(1)
        if first == 0:
            assert np.array_equal(c.spins, a.spins)


def test_mixed_cycle_fixed_points():
    L = 8
    for s0 in (inputs.all_up(L), -inputs.all_up(L), inputs.slab(L, 2, 1, 4)):
        o = orc.Oracle(L, 9, init=False)
        o.spins[...] = s0
        o.sweep_mixed(5)
        assert np.array_equal(o.spins, s0)


# ------------------------------------------------------------------ f-3: Menger sponge
def test_menger_solid_counts_and_first_iteration():
    """A k-th iteration Menger sponge keeps 20 of 27 sub-cubes per level: 20^k sites of 27^k.
    k = 1 written out: of the 27 cells the 6 face centres and the body centre are removed."""
    for k in range(0, 4):
        n = 3 ** k
        cnt = sum(orc.menger_solid(u, v, w, k) for u in range(n) for v in range(n) for w in range(n))
        assert cnt == 20 ** k
    removed = {(1, 1, 0), (1, 1, 2), (1, 0, 1), (1, 2, 1), (0, 1, 1), (2, 1, 1), (1, 1, 1)}
    for u in range(3):
        for v in range(3):
            for w in range(3):
                assert orc.menger_solid(u, v, w, 1) == (0 if (u, v, w) in removed else 1)


def test_menger_solid_self_similarity_and_symmetry():
    """Iteration k+1 = 20 copies of iteration k placed on the iteration-1 pattern; the sponge is
    invariant under permutations and reflections of the axes."""
    k = 2
    n = 3 ** k
    for u in range(3 * n):
        for v in range(0, 3 * n, 2):
            for w in range(0, 3 * n, 3):
                want = orc.menger_solid(u // n, v // n, w // n, 1) and orc.menger_solid(u % n, v % n, w % n, k)
                assert orc.menger_solid(u, v, w, k + 1) == int(bool(want))
    m = 27
    for (u, v, w) in [(1, 4, 13), (0, 0, 0), (13, 13, 2), (26, 1, 1), (9, 10, 12), (4, 22, 16)]:
        ref = orc.menger_solid(u, v, w, 3)
        assert orc.menger_solid(v, w, u, 3) == ref and orc.menger_solid(w, v, u, 3) == ref
        assert orc.menger_solid(m - 1 - u, v, w, 3) == ref and orc.menger_solid(u, m - 1 - v, m - 1 - w, 3) == ref


@pytest.mark.parametrize("L,k", [(54, 3), (32, 2), (20, 1)])
def test_init_menger_structure(L, k):
    """Every (possibly cut) tile is one sponge pattern or its negative, the pattern
    is the restated Menger rule, and the sign is the documented Philox bit (D11)."""
    size = 3 ** k
    seed = 77
    o = orc.Oracle(L, seed, init=False)
    o.init_menger(k)
    s = o.spins                                           # [z][y][x]
    nT = -(-L // size)
    u = np.arange(size)
    U, V, W = np.meshgrid(u, u, u, indexing="ij")         # as [z][y][x] local coordinates
    solid = np.ones((size, size, size), dtype=bool)
    a, b, c = U.copy(), V.copy(), W.copy()
    for _ in range(k):
        ones = (a % 3 == 1).astype(int) + (b % 3 == 1) + (c % 3 == 1)
        solid &= ones < 2
        a //= 3; b //= 3; c //= 3
    pattern = np.where(solid, 1, -1).astype(np.int8)
    signs = []
    for Z in range(nT):
        for Y in range(nT):
            for X in range(nT):
                blk = s[Z * size:(Z + 1) * size, Y * size:(Y + 1) * size, X * size:(X + 1) * size]
                pat = pattern[:blk.shape[0], :blk.shape[1], :blk.shape[2]]
                T = (Z * nT + Y) * nT + X
                bit = (py_philox([T >> 7, k, 0, 3], [seed & MASK, seed >> 32])[(T >> 5) & 3] >> (T & 31)) & 1
                assert np.array_equal(blk, pat if bit else -pat), (X, Y, Z)
                signs.append(bit)
    assert o.sweep_count == 0
    if len(signs) >= 8:
        assert 0 < sum(signs) < len(signs)


def test_init_menger_k0_is_an_iid_start():
    """k = 0: one site per sponge, i.e. an iid p = 1/2 configuration."""
    L = 32
    o = orc.Oracle(L, 5, init=False)
    o.init_menger(0)
    N = L ** 3
    n_up, a = o.measure([1, 2, 5])
    assert abs(n_up - N / 2) < 4 * np.sqrt(N) / 2
    assert np.all(np.abs(a.astype(float) - N / 2) < 4 * np.sqrt(N) / 2)


def test_init_menger_tile_signs_fair():
    L, k = 96, 1                                           # 32^3 tiles
    o = orc.Oracle(L, 123, init=False)
    o.init_menger(k)
    corner = o.spins[::3, ::3, ::3]                        # (0,0,0) of every tile is solid
    n = corner.size
    assert abs((corner == 1).sum() - n / 2) < 4 * np.sqrt(n) / 2
    # magnetisation of a sponge start: |m| per tile = (20 - 7)/27
    tiles = o.spins.reshape(32, 3, 32, 3, 32, 3).sum(axis=(1, 3, 5))
    assert set(np.unique(tiles)) <= {13, -13}


def test_menger_site_equals_the_array_form_and_the_documented_bit_beyond_2_to_32():
    """orc_menger_site (one site of D11) against orc_init_menger site by site on small lattices,
    and, where the tile index T passes 2^32 (L = 2048, k = 0: T = (z*L + y)*L + x up to 2^33),
    against the rule written out with the big-integer Python Philox: sign bit = bit T & 31 of
    word (T >> 5) & 3 of Philox(counter (T >> 7 mod 2^32, k, 0, 3)) (D11)."""
    for L, k, seed in [(20, 1, 9), (18, 2, 10), (12, 0, 11)]:
        o = orc.Oracle(L, seed, init=False)
        o.init_menger(k)
        s = o.spins
        for z in range(L):
            for y in range(L):
                for x in range(0, L, 1 if L < 16 else 3):
                    assert orc.menger_site(seed, L, k, x, y, z) == int(s[z, y, x])
    L, seed = 2048, 4
    key = [seed & MASK, seed >> 32]
    seen_high = 0
    for (x, y, z) in [(0, 0, 0), (5, 0, 1023), (7, 1, 1024), (2047, 2047, 2047), (100, 900, 1500),
                      (100, 900, 476), (1, 2, 2046), (64, 0, 1024), (64, 0, 0)]:
        T = (z * L + y) * L + x
        seen_high += T >= 2 ** 32
        word = py_philox([(T >> 7) & MASK, 0, 0, 3], key)[(T >> 5) & 3]
        want = 1 if (word >> (T & 31)) & 1 else -1
        assert orc.menger_site(seed, L, 0, x, y, z) == want, (x, y, z)
    assert seen_high >= 4
    # a 32-bit tile index would alias planes z and z + 1024 at L = 2048: the rule does not
    a = [orc.menger_site(seed, L, 0, x, 3, 10) for x in range(256)]
    b = [orc.menger_site(seed, L, 0, x, 3, 10 + 1024) for x in range(256)]
    assert a != b


# ------------------------------------------------------------------ f-1: FFT correlation + radial average
def _exact_bin(L, dx, dy, dz):
    """D12 restated with exact rationals: nearest integer to |d| of the minimal image."""
    from fractions import Fraction
    f = lambda v: v - L if v > L // 2 else v
    n = f(dx) ** 2 + f(dy) ** 2 + f(dz) ** 2
    b = 0
    while Fraction(2 * b + 1, 2) ** 2 <= n:
        b += 1
    return b


def test_radial_bins_and_shell_counts():
    L = 12
    seen = {}
    for dz in range(L):
        for dy in range(L):
            for dx in range(L):
                b = orc.radial_bin(L, dx, dy, dz)
                assert b == _exact_bin(L, dx, dy, dz)
                seen[b] = seen.get(b, 0) + 1
    assert orc.radial_bin(L, 0, 0, 0) == 0 and seen[0] == 1
    assert seen[1] == 6 + 12                      # |d| = 1 (6) and sqrt(2) = 1.41 (12); sqrt(3) -> 2
    assert orc.radial_bin(L, L - 1, 0, 0) == 1 and orc.radial_bin(L, L // 2, 0, 0) == L // 2
    _, cnt = orc.radial_sums(L, np.ones((L, L, L), dtype=np.int64))
    assert [int(c) for c in cnt] == [seen.get(b, 0) for b in range(L // 2 + 1)]
    # vectorised bins used by the FFT route == the C rule
    from oracle.oracle import _bins_numpy
    bn = _bins_numpy(L)
    assert all(bn[z, y, x] == orc.radial_bin(L, x, y, z) for x in range(L) for y in range(L) for z in range(L))


def test_correlation_matrix_identities():
    """P(d) = sum_i s_i s_{i+d} from the definition: P(0) = N; sum_d P(d) = M^2; P(-d) = P(d);
    along the axes P(r e_mu) = N - 2 A_mu(r) with A_mu from the (separately pinned) pair counts;
    and the FFT route of eq. (7) gives the same integers."""
    L = 8
    o = orc.Oracle(L, 21)
    o.sweep(3)
    P = o.corr_direct()
    N = L ** 3
    M = int(o.spins.astype(np.int64).sum())
    assert P[0, 0, 0] == N and P.sum() == M * M
    assert np.array_equal(P, P[(-np.arange(L)) % L][:, (-np.arange(L)) % L][:, :, (-np.arange(L)) % L])
    n_up, a = o.measure()
    for r in range(L // 2 + 1):
        assert P[0, 0, r] == N - 2 * int(a[0][r]) and P[0, r, 0] == N - 2 * int(a[1][r]) \
            and P[r, 0, 0] == N - 2 * int(a[2][r])
    assert np.array_equal(o.corr_fft(), P)
    o16 = orc.Oracle(16, 5)
    o16.sweep(2)
    assert np.array_equal(o16.corr_fft(), o16.corr_direct())


def test_correlation_closed_forms():
    """All up: P = N everywhere, C_rad = 0.  Slab of thickness L/2 along z: P(d) depends on dz
    only, P = N (1 - 4|dz|/L) for the folded dz (triangle wave)."""
    L = 8
    N = L ** 3
    o = orc.Oracle(L, 1, init=False)
    o.spins[...] = 1
    r = o.measure_radial(direct=True)
    assert np.all(r["corr_sum"] == N * r["shell"].astype(np.int64)) and np.allclose(r["C_rad"], 0.0)
    o.spins[...] = inputs.slab(L, 2, 1, L // 2)
    P = o.corr_direct()
    for dz in range(L):
        f = dz if dz <= L // 2 else L - dz
        assert np.all(P[dz] == N - 4 * f * L * L)
    assert o.measure_radial(direct=True)["m"] == 0.0


def test_structure_factor_identities():
    """S(k) = |F s|^2 / N: Parseval sum_k |F s|^2 = N * sum_i s_i^2 = N^2; the k = 0 bin is N m^2;
    a plane wave s = sign(cos) along x puts all weight on kx = +-1 (odd harmonics), none on ky, kz != 0."""
    L = 16
    N = L ** 3
    o = orc.Oracle(L, 8)
    o.sweep(4)
    ps = o.power_spectrum()
    assert abs(ps.sum() - float(N) ** 2) < 1e-6 * N ** 2
    r = o.measure_radial()
    assert abs(r["S_rad"][0] - N * r["m"] ** 2) < 1e-9 * max(1.0, N * r["m"] ** 2)
    o.spins[...] = inputs.slab(L, 0, 0, L // 2)           # +1 for x < L/2: a square wave along x
    ps = o.power_spectrum()
    assert np.all(ps[1:, :, :] < 1e-9) and np.all(ps[:, 1:, :] < 1e-9)
    assert ps[0, 0, 1] > 0.3 * N ** 2 and abs(ps[0, 0, 2]) < 1e-9


def test_radial_measure_fft_equals_direct_and_ell():
    L = 16
    o = orc.Oracle(L, 13)
    o.sweep(6)
    a = o.measure_radial(direct=True)
    b = o.measure_radial(direct=False)
    assert np.array_equal(a["corr_sum"], b["corr_sum"]) and np.array_equal(a["shell"], b["shell"])
    assert a["C_rad"][0] == pytest.approx(1.0 - a["m"] ** 2, abs=1e-15)     # P(0) = N
    # ell: first crossing of C_rad with c, linear interpolation (D9 rule)
    C = a["C_rad"]
    r0 = next(r for r in range(L // 2) if C[r] >= 0.5 > C[r + 1])
    assert a["ell"] == pytest.approx(r0 + (C[r0] - 0.5) / (C[r0] - C[r0 + 1]), rel=1e-15)


# ------------------------------------------------------------------ f-4: finite-temperature Glauber
def test_glauber_thresholds():
    """eq. (5) PAPER.md:101 with Delta E = 12 - 4n: p(3) = 1/2 exactly, p(6-n) = 1 - p(n), hand
    values at T = 4 (p(0) = 1/(1+e^3) = 0.0474258731...), limits T -> 0 (eq. (6)) and T -> inf."""
    import math
    thr = orc.glauber_thresholds(4.0)
    assert int(thr[3]) == 2 ** 31
    for n in range(7):
        assert abs(int(thr[n]) + int(thr[6 - n]) - 2 ** 32) <= 1
        want = 1.0 / (1.0 + math.exp((12 - 4 * n) / 4.0))
        assert abs(int(thr[n]) / 2.0 ** 32 - want) < 2.0 ** -31
    assert abs(int(thr[0]) / 2.0 ** 32 - 0.04742587317756678) < 1e-9
    cold = orc.glauber_thresholds(0.05)
    assert [int(v) for v in cold] == [0, 0, 0, 2 ** 31, 2 ** 32, 2 ** 32, 2 ** 32]     # eq. (6)
    hot = orc.glauber_thresholds(1e12)
    assert all(abs(int(v) - 2 ** 31) <= 1 for v in hot)


def test_site_uniform_is_the_documented_bit_planes():
    """D13: u = sum_j b_j 2^(31-j), b_j the site's bit of Philox(counter (q, t, c, 4 + j))."""
    from test_oracle_pins import py_site_bit
    L, seed = 8, 0x1234567899
    for (x, y, z, t) in [(0, 0, 0, 0), (7, 3, 5, 2), (2, 6, 1, 1000)]:
        want = 0
        for j in range(32):
            want |= py_site_bit(seed, L, x, y, z, t, 4 + j) << (31 - j)
        assert orc.site_uniform(seed, L, x, y, z, t) == want
    us = np.array([orc.site_uniform(3, 8, x, y, z, 0) for x in range(8) for y in range(8) for z in range(8)],
                  dtype=np.float64) / 2.0 ** 32
    assert abs(us.mean() - 0.5) < 4 * (1 / 12 ** 0.5) / 512 ** 0.5


def test_glauber_acceptance_frequencies():
    """States where every site has the same n: all up (n = 0) flips a fraction p(0) of the first
    colour, the Neel state (n = 6) a fraction p(6) = 1 - p(0); binomial 4 sigma."""
    import math
    L, T = 32, 4.0
    half = L ** 3 // 2
    p0 = 1.0 / (1.0 + math.exp(12 / T))
    o = orc.Oracle(L, 17, init=False)
    o.spins[...] = 1
    o.half_sweep_T(0, 0, T)
    flipped = int((o.spins == -1).sum())
    assert abs(flipped - half * p0) < 4 * math.sqrt(half * p0 * (1 - p0))
    z, y, x = np.meshgrid(np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    assert np.all(o.spins[((x + y + z) & 1) == 1] == 1)          # the other colour was not proposed
    o.spins[...] = inputs.neel(L)
    o.half_sweep_T(3, 0, T)
    kept = int((o.spins[((x + y + z) & 1) == 0] == 1).sum())     # black sites that did NOT flip
    assert abs(kept - half * p0) < 4 * math.sqrt(half * p0 * (1 - p0))


def test_glauber_hot_limit_closed_form():
    """T -> infinity: thr = 2^31 for every n, so a site flips iff the top bit of u (Philox tag 4)
    is 0, whatever its neighbours."""
    from test_oracle_pins import py_site_bit
    L, seed = 6, 5
    o = orc.Oracle(L, seed)
    before = o.spins.copy()
    o.half_sweep_T(0, 0, 1e12)
    for z in range(L):
        for y in range(L):
            for x in range(L):
                if (x + y + z) & 1:
                    assert o.spins[z, y, x] == before[z, y, x]
                else:
                    flip = py_site_bit(seed, L, x, y, z, 0, 4) == 0
                    assert o.spins[z, y, x] == (-before[z, y, x] if flip else before[z, y, x])


def test_glauber_cold_limit_and_relaxation():
    """T -> 0: the deterministic moves of eq. (6) (n >= 4 flips, n <= 2 stays) are reproduced;
    at T = 1.5 the energy of a quench relaxes far below the random start and stays above the
    ground state; sweep_T(n) == n x (half_sweep_T colour 0, colour 1)."""
    L = 16
    a = orc.Oracle(L, 9)
    b = orc.Oracle(L, 9)
    s0 = a.spins.copy()
    a.half_sweep_T(0, 0, 0.05)
    b.half_sweep(0, 0)                                           # T = 0 rule: same except at ties
    z, y, x = np.meshgrid(np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    nbr = sum(np.roll(s0, sh, axis=ax) for ax in (0, 1, 2) for sh in (1, -1))
    n_anti = (6 - s0 * nbr) // 2
    det = (((x + y + z) & 1) == 0) & (n_anti != 3)
    assert np.array_equal(a.spins[det], b.spins[det])
    c = orc.Oracle(L, 4)
    d = orc.Oracle(L, 4)
    e0 = c.measure([1])[1].sum()
    c.sweep_T(12, 1.5)
    for t in range(12):
        d.half_sweep_T(t, 0, 1.5)
        d.half_sweep_T(t, 1, 1.5)
    assert np.array_equal(c.spins, d.spins) and c.sweep_count == 12
    e1 = c.measure([1])[1].sum()
    assert 0 < e1 < 0.45 * e0


# ------------------------------------------------------------------ f-2: double checkerboard
def test_double_checkerboard_reduces_to_plain_sweep():
    """One block (B >= L): the coarse colour is 0 everywhere, the sweep is (fine 0, fine 1) and
    nothing else: the plain 01 sweep."""
    L = 12
    a = orc.Oracle(L, 6)
    b = orc.Oracle(L, 6)
    a.sweep_dcb(5, block=L)
    b.sweep(5)
    assert np.array_equal(a.spins, b.spins) and a.sweep_count == 5


def test_double_checkerboard_python_restatement():
    """Pure-Python statement of Supp. I.A on L = 8, B = 4: red blocks (dark, then light), then
    blue blocks, sites visited one by one with the Delta-E rule and the site's Philox bit."""
    from test_oracle_pins import py_site_bit
    L, B, seed = 8, 4, 31
    o = orc.Oracle(L, seed)
    s = o.spins.copy().astype(int)                       # [z][y][x]
    for t in range(3):
        for coarse in (0, 1):
            for fine in (0, 1):
                for z in range(L):
                    for y in range(L):
                        for x in range(L):
                            if (x + y + z) % 2 != fine or (x // B + y // B + z // B) % 2 != coarse:
                                continue
                            h = (s[z][y][(x + 1) % L] + s[z][y][(x - 1) % L] + s[z][(y + 1) % L][x]
                                 + s[z][(y - 1) % L][x] + s[(z + 1) % L][y][x] + s[(z - 1) % L][y][x])
                            dE = 2 * s[z][y][x] * h
                            if dE < 0 or (dE == 0 and py_site_bit(seed, L, x, y, z, t, 0)):
                                s[z][y][x] = -s[z][y][x]
    o.sweep_dcb(3, block=B)
    assert np.array_equal(o.spins, s.astype(np.int8))


def test_double_checkerboard_order_readout_and_invariants():
    """From the Neel state the first phase (red blocks, dark sites) flips exactly the dark sites
    of the red blocks (n = 6) and nothing else; the dark sites of the blue blocks bordering a red
    block have then lost antiparallel neighbours.  Every phase only lowers the energy; all-up and
    slab states are fixed points."""
    L, B = 16, 4
    z, y, x = np.meshgrid(np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    fine = (x + y + z) & 1
    coarse = (x // B + y // B + z // B) & 1
    o = orc.Oracle(L, 2, init=False)
    o.spins[...] = inputs.neel(L)
    o.half_sweep_dcb(0, 0, 0, B)
    want = inputs.neel(L).copy()
    want[(fine == 0) & (coarse == 0)] *= -1
    assert np.array_equal(o.spins, want)
    o = orc.Oracle(L, 3)
    e = o.measure([1])[1].sum()
    for t in range(4):
        for c in (0, 1):
            for f in (0, 1):
                o.half_sweep_dcb(t, c, f, B)
                e2 = o.measure([1])[1].sum()
                assert e2 <= e
                e = e2
    for s0 in (inputs.all_up(L), inputs.slab(L, 1, 2, L // 2)):
        o.spins[...] = s0
        o.sweep_dcb(3, block=B)
        assert np.array_equal(o.spins, s0)


# ------------------------------------------------------------------ f-2: double checkerboard, mixed cycle
def test_dcb_mixed_bits_and_neel_readout():
    """D15: block bits are the documented Philox bits; from the Neel state the first pass of a
    sweep flips, in every block of the coarse colour drawn first, exactly the sites of that
    block's first fine colour (n = 6) and nothing else: the state reads out both random choices."""
    L, B, seed = 16, 4, 21
    nB = L // B
    for Bi in (0, 1, 17, 63):
        for t in (0, 3):
            want = (py_philox([Bi >> 7, t, 0, 36], [seed & MASK, seed >> 32])[(Bi >> 5) & 3] >> (Bi & 31)) & 1
            assert orc.block_first_fine(seed, t, Bi) == want
    z, y, x = np.meshgrid(np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    fine = (x + y + z) & 1
    coarse = (x // B + y // B + z // B) & 1
    Bi = ((z // B) * nB + (y // B)) * nB + (x // B)
    seen_first, seen_ff = set(), set()
    for t in range(6):
        o = orc.Oracle(L, seed, init=False)
        o.spins[...] = inputs.neel(L)
        first = orc.first_colour(seed, t)
        ff = np.vectorize(lambda b: orc.block_first_fine(seed, t, int(b)))(Bi)
        o.pass_dcb_mixed(t, first, 0, B)
        want = inputs.neel(L).copy()
        want[(coarse == first) & (fine == ff)] *= -1
        assert np.array_equal(o.spins, want)
        seen_first.add(first)
        seen_ff |= set(np.unique(ff[coarse == first]))
    assert seen_first == {0, 1} and seen_ff == {0, 1}


def test_dcb_mixed_python_restatement_and_invariants():
    from test_oracle_pins import py_site_bit
    L, B, seed = 8, 4, 5
    nB = L // B
    o = orc.Oracle(L, seed)
    s = o.spins.copy().astype(int)
    for t in range(3):
        first = py_philox([0, t, 0, 2], [seed & MASK, seed >> 32])[0] & 1
        for coarse in (first, 1 - first):
            for pas in (0, 1):
                for z in range(L):
                    for y in range(L):
                        for x in range(L):
                            if (x // B + y // B + z // B) % 2 != coarse:
                                continue
                            bi = ((z // B) * nB + (y // B)) * nB + (x // B)
                            ff = (py_philox([bi >> 7, t, 0, 36], [seed & MASK, seed >> 32])[(bi >> 5) & 3] >> (bi & 31)) & 1
                            if (x + y + z) % 2 != (ff ^ pas):
                                continue
                            h = (s[z][y][(x + 1) % L] + s[z][y][(x - 1) % L] + s[z][(y + 1) % L][x]
                                 + s[z][(y - 1) % L][x] + s[(z + 1) % L][y][x] + s[(z - 1) % L][y][x])
                            dE = 2 * s[z][y][x] * h
                            if dE < 0 or (dE == 0 and py_site_bit(seed, L, x, y, z, t, 0)):
                                s[z][y][x] = -s[z][y][x]
    o.sweep_dcb_mixed(3, block=B)
    assert np.array_equal(o.spins, s.astype(np.int8)) and o.sweep_count == 3
    # energy never increases pass by pass; fixed points stay
    L = 16
    a = orc.Oracle(L, 9)
    e = a.measure([1])[1].sum()
    for t in range(3):
        first = orc.first_colour(9, t)
        for coarse in (first, 1 - first):
            for pas in (0, 1):
                a.pass_dcb_mixed(t, coarse, pas, 4)
                e2 = a.measure([1])[1].sum()
                assert e2 <= e
                e = e2
    a.spins[...] = inputs.slab(L, 2, 3, L // 2)
    keep = a.spins.copy()
    a.sweep_dcb_mixed(3, block=4)
    assert np.array_equal(a.spins, keep)


# ------------------------------------------------------------------ activity (ising3d_activity)
def _groups_changed(before: np.ndarray, after: np.ndarray) -> np.ndarray:
    """[2][groups] bool: 128-spin groups (4 packed words, D3) whose words differ."""
    d = (before != after).reshape(2, -1, 4).any(axis=2)
    return d


def test_activity_closed_forms():
    """eq. (6): only sites with Delta E <= 0 can change.  All up: none.  Neel
    state: every site has Delta E = -12, so every group counts.  One reversed spin in an ordered
    lattice: that site has Delta E = -12, its six neighbours Delta E = +8: exactly one group, of
    the reversed site's colour."""
    L = 16
    G = L ** 3 // 2 // 128
    o = orc.Oracle(L, 1, init=False)
    o.spins[...] = 1
    assert list(o.activity()) == [0, 0]
    o.spins[...] = inputs.neel(L)
    assert list(o.activity()) == [G, G]
    for (x, y, z) in [(0, 0, 0), (5, 2, 8), (15, 15, 15), (3, 0, 15)]:
        o.spins[...] = -1
        o.spins[z, y, x] = 1
        want = [0, 0]
        want[(x + y + z) & 1] = 1
        assert list(o.activity()) == want


@pytest.mark.parametrize("L,kind,sweeps", [(16, "random", 0), (32, "random", 6), (64, "domains", 0),
                                           (64, "domains", 4), (64, "noisy", 0), (64, "noisy", 1)])
def test_activity_is_exactly_the_groups_a_half_sweep_can_change(L, kind, sweeps):
    """Operational pin through the separately pinned orc_half_sweep: from one configuration, the
    union over many seeds (= tie-bit assignments) of the groups a colour-c half-sweep changes is
    exactly the set of groups holding a site with Delta E <= 0 -- a site with Delta E < 0 flips
    for every seed, a tie for about half of them -- and the count is non-trivial (neither 0 nor
    all groups) on the domain states."""
    base = orc.Oracle(L, 77)
    if kind == "domains":
        base.spins[...] = inputs.domain_spins(L, 5, block=16, p_minority=0.15)
    elif kind == "noisy":
        base.spins[...] = inputs.domain_spins(L, 6, block=16, p_minority=0.3, noise=0.002)
    base.sweep(sweeps)
    words0 = base.export_words()
    spins0 = base.spins.copy()
    want = base.activity()
    G = L ** 3 // 2 // 128
    union = np.zeros((2, G), dtype=bool)
    for seed in range(200, 248):                       # 48 tie-bit assignments: a miss has p = 2^-48
        for c in (0, 1):
            o = orc.Oracle(L, seed, init=False)
            o.spins[...] = spins0
            o.half_sweep(sweeps, c)
            union[c] |= _groups_changed(words0, o.export_words())[c]
    assert [int(union[0].sum()), int(union[1].sum())] == [int(want[0]), int(want[1])]
    if kind != "random":
        assert 0 < want[0] < G and 0 < want[1] < G
