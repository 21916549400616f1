"""GPU parity of the SURVEY.md 8(f) rows built so far, through the C ABI, against the oracle:
mixed cycle (f-2, Supp. I.B PAPER.md:258, D10) and Menger-sponge start (f-3, D11).
Bit-exact states and counts; C(r), ell within 1e-12 relative."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2305_12161_b200 import inputs  # noqa: E402
from test_gpu_parity import check_measure, VARIANTS, _sample_sites, _bits_at  # noqa: E402


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2305_12161_b200 import build, binding
    build.build()
    return binding


@pytest.fixture(scope="module")
def orc():
    from oracle import oracle
    oracle.build()
    return oracle


# ------------------------------------------------------------------ f-2: mixed cycle
@pytest.mark.parametrize("L,seed,variant,cps", [
    (64, 1, "resident", [1, 2, 5, 20]), (64, 5, "generic", [1, 7]), (128, 7, "resident", [3, 12]),
    (192, 8, "generic", [1, 4]), (256, 2, "resident", [2, 9]), (256, 2, "generic", [3]),
    (512, 11, "fused2", [1, 2, 6]), (1024, 3, "fused2", [1, 3])])
def test_mixed_cycle_against_oracle(B, orc, L, seed, variant, cps):
    sim = B.Ising3D(L, [seed], variant=VARIANTS(B)[variant])
    sim.set_cycle(B.CYCLE_MIXED)
    assert sim.variant_name == variant
    ref = orc.Oracle(L, seed)
    t = 0
    for cp in cps:
        sim.sweep(cp - t)
        ref.sweep_mixed(cp - t)
        t = cp
        assert np.array_equal(sim.get_state(), ref.export_words()), "state differs at sweep %d" % cp
    if L <= 512:
        check_measure(sim.measure(), ref.measure_full())
    # the orders drawn so far contained both colours (else the test proves nothing)
    assert {orc.first_colour(seed, s) for s in range(cps[-1])} == {0, 1} or cps[-1] < 3
    sim.free()


def test_mixed_cycle_batch_draws_an_order_per_replica(B, orc):
    L, seeds = 128, [100, 101, 102, 103, 131, 163]
    batch = B.Ising3D(L, seeds)
    batch.set_cycle(B.CYCLE_MIXED)
    assert batch.variant_name == "resident"
    refs = [orc.Oracle(L, s) for s in seeds]
    assert len({tuple(orc.first_colour(s, t) for t in range(6)) for s in seeds}) > 1
    for n in (1, 5):
        batch.sweep(n)
        st = batch.get_state().reshape(len(seeds), -1)
        for i, ref in enumerate(refs):
            ref.sweep_mixed(n)
            assert np.array_equal(st[i], ref.export_words())
    batch.free()


def test_mixed_cycle_neel_closed_form_on_gpu(B, orc):
    """One mixed sweep from the Neel state orders the lattice with the value of the colour
    updated second (closed form, see tests/test_oracle_next.py): reads out the order used."""
    for L, variant in ((64, "resident"), (512, "fused2"), (192, "generic")):
        sim = B.Ising3D(L, [11], variant=VARIANTS(B)[variant])
        sim.set_cycle(B.CYCLE_MIXED)
        words = inputs.pack_spins(inputs.neel(L))
        for t in range(6):
            sim.set_state(words, t)
            sim.sweep(1)
            first = orc.first_colour(11, t)
            want = np.full(L ** 3 // 32, 0xFFFFFFFF if first else 0, dtype=np.uint32)
            assert np.array_equal(sim.get_state(), want)
        sim.free()


def test_mixed_cycle_full_size_sampled(B, orc):
    """L = 2048 in the bench launch configuration, mixed cycle: fused2 == generic word for word
    over sweeps whose drawn orders differ."""
    L, seed = 2048, 4
    a = B.Ising3D(L, [seed])
    b = B.Ising3D(L, [seed], variant=B.VARIANT_GENERIC)
    a.set_cycle(B.CYCLE_MIXED)
    b.set_cycle(B.CYCLE_MIXED)
    assert a.variant_name == "fused2"
    assert {orc.first_colour(seed, t) for t in range(4)} == {0, 1}
    for n in (1, 3):
        a.sweep(n)
        b.sweep(n)
        assert np.array_equal(a.get_state(), b.get_state())
    a.free()
    b.free()


def test_cycle_errors(B):
    sim = B.Ising3D(256, [1], variant=B.VARIANT_FUSED)
    with pytest.raises(B.Ising3DError):
        sim.set_cycle(B.CYCLE_MIXED)
    with pytest.raises(B.Ising3DError):
        sim.set_cycle(7)
    sim.free()


# ------------------------------------------------------------------ f-3: Menger sponge
@pytest.mark.parametrize("L,k,seed", [(64, 0, 3), (64, 1, 3), (64, 2, 4), (64, 3, 5), (128, 3, 6),
                                      (192, 2, 7), (256, 4, 8)])
def test_menger_start_and_quench(B, orc, L, k, seed):
    sim = B.Ising3D(L, [seed])
    sim.sweep(2)
    sim.init_menger(k)
    assert sim.sweep_count == 0
    ref = orc.Oracle(L, seed, init=False)
    ref.init_menger(k)
    assert np.array_equal(sim.get_state(), ref.export_words()), "Menger start differs"
    for n in (1, 4):
        sim.sweep(n)
        ref.sweep(n)
        assert np.array_equal(sim.get_state(), ref.export_words())
    check_measure(sim.measure(), ref.measure_full())
    sim.free()


def test_menger_batch_and_errors(B, orc):
    L, seeds = 128, [100, 101, 163]
    batch = B.Ising3D(L, seeds)
    batch.init_menger(2)
    st = batch.get_state().reshape(3, -1)
    for i, s in enumerate(seeds):
        ref = orc.Oracle(L, s, init=False)
        ref.init_menger(2)
        assert np.array_equal(st[i], ref.export_words())
    assert not np.array_equal(st[0], st[1])
    with pytest.raises(B.Ising3DError):
        batch.init_menger(5)          # 3^5 = 243 > L
    with pytest.raises(B.Ising3DError):
        batch.init_menger(-1)
    batch.free()


def test_menger_full_size_structure(B, orc):
    """L = 512, k = 3 (the paper's Fig. 4(c) size): sampled sites against the oracle's
    menger_solid and tile signs read off the solid corner site of each tile."""
    L, k, seed = 512, 3, 9
    sim = B.Ising3D(L, [seed])
    sim.init_menger(k)
    words = sim.get_state()
    rng = np.random.Generator(np.random.PCG64(1))
    xyz = rng.integers(0, L, size=(4000, 3)).astype(np.int32)
    got = _bits_at(words, L, xyz)
    corner = (xyz // 27) * 27
    sign = _bits_at(words, L, corner.astype(np.int32))      # local (0,0,0) is always solid
    solid = np.array([orc.menger_solid(int(x % 27), int(y % 27), int(z % 27), k) for x, y, z in xyz])
    assert np.array_equal(got, np.where(solid == 1, sign, -sign))
    m = sim.measure()
    assert 0 < int(m["n_up"][0]) < L ** 3
    sim.free()


def test_menger_k0_at_L2048_tile_index_beyond_32_bits(B, orc):
    """k = 0 at L = 2048: one tile per site, tile index T = (z*L + y)*L + x up to 2^33 (D11).
    Sampled sites (both halves in z, so that a tile index truncated to 32 bits would alias
    planes z and z + 1024) against the oracle's single-site form of the rule."""
    L, seed = 2048, 4
    sim = B.Ising3D(L, [seed])
    sim.init_menger(0)
    buf = np.empty(L ** 3 // 32, dtype=np.uint32)
    words = sim.get_state(buf)
    rng = np.random.Generator(np.random.PCG64(5))
    xyz = rng.integers(0, L, size=(3000, 3)).astype(np.int32)
    mirror = xyz.copy()
    mirror[:, 2] = (mirror[:, 2] + L // 2) % L
    xyz = np.concatenate([xyz, mirror, [[0, 0, 0], [L - 1, L - 1, L - 1], [0, 0, L // 2]]]).astype(np.int32)
    got = _bits_at(words, L, xyz)
    want = np.array([orc.menger_site(seed, L, 0, int(x), int(y), int(z)) for x, y, z in xyz], dtype=np.int8)
    assert np.array_equal(got, want)
    assert (xyz[:, 2] >= L // 2).sum() > 1000        # tile indices >= 2^32 are covered
    sim.free()


# ------------------------------------------------------------------ f-4 (part): L = 4096 on one GPU
def test_L4096_one_gpu(B, orc):
    """The size the paper hopes for next ("L=4096, in the near future"): 6.9e10 spins,
    8 GiB packed (16 GiB with the ping-pong buffer).  fused2 == generic word for word, sampled
    sites against the oracle's single-site evaluation, tensor == popcount measurement."""
    L, seed = 4096, 12
    a = B.Ising3D(L, [seed])
    assert a.variant_name == "fused2" and a.measure_variant_name == "tensor"
    xyz = _sample_sites(L, 3000, 23, RPT=60)
    buf = np.empty(L ** 3 // 32, dtype=np.uint32)
    got0 = _bits_at(a.get_state(buf), L, xyz)
    assert np.array_equal(got0, orc.sites_after(seed, L, xyz, 0))
    a.sweep(1)
    got1 = _bits_at(a.get_state(buf), L, xyz)
    assert np.array_equal(got1, orc.sites_after(seed, L, xyz, 2))
    b = B.Ising3D(L, [seed], variant=B.VARIANT_GENERIC)
    b.sweep(1)
    buf_b = np.empty(L ** 3 // 32, dtype=np.uint32)
    assert np.array_equal(b.get_state(buf_b), buf)
    b.free()
    del buf_b
    m_t = a.measure()
    a.set_measure_variant(B.MEASURE_POPCOUNT)
    m_p = a.measure()
    assert np.array_equal(m_t["antipar"], m_p["antipar"]) and np.array_equal(m_t["n_up"], m_p["n_up"])
    assert int(m_t["n_broken"][0]) == int(m_t["antipar"][0][:, 1].sum())
    a.free()


# ------------------------------------------------------------------ f-1: FFT correlation + radial average
def _check_radial(got, want, rep=0):
    assert np.array_equal(got["corr_sum"][rep], want["corr_sum"])          # exact integers
    assert np.array_equal(got["shell"], want["shell"])
    assert np.all(np.abs(got["C_rad"][rep] - want["C_rad"]) <= 1e-12 * np.maximum(1.0, np.abs(want["C_rad"])))
    # S(k): fp64 sums in a different order; D12 tolerance 1e-9 of the largest bin
    scale = np.abs(want["S_rad"]).max()
    assert np.all(np.abs(got["S_rad"][rep] - want["S_rad"]) <= 1e-9 * scale)
    if np.isnan(want["ell"]):
        assert np.isnan(got["ell"][rep])
    else:
        assert abs(got["ell"][rep] - want["ell"]) <= 1e-12 * abs(want["ell"])


@pytest.mark.parametrize("L,seed,sweeps", [(64, 1, 0), (64, 1, 12), (128, 7, 5), (192, 8, 3), (256, 2, 20),
                                           (384, 11, 6)])
def test_radial_estimator_against_oracle(B, orc, L, seed, sweeps):
    sim = B.Ising3D(L, [seed])
    ref = orc.Oracle(L, seed)
    assert sim.radial_rounding == -1.0
    sim.sweep(sweeps)
    ref.sweep(sweeps)
    _check_radial(sim.measure_radial(), ref.measure_radial())
    assert 0.0 <= sim.radial_rounding < 1e-3            # exactness margin of the llrint (D12)
    # measuring does not disturb the state or the other measurement
    assert np.array_equal(sim.get_state(), ref.export_words())
    check_measure(sim.measure(), ref.measure_full())
    sim.free()


def test_radial_estimator_batch_and_structured(B, orc):
    L, seeds = 64, [100, 101, 102]
    batch = B.Ising3D(L, seeds)
    batch.sweep(4)
    got = batch.measure_radial(c_intercept=0.3)
    for i, s in enumerate(seeds):
        ref = orc.Oracle(L, s)
        ref.sweep(4)
        _check_radial(got, ref.measure_radial(c_intercept=0.3), rep=i)
    batch.free()
    sim = B.Ising3D(L, [1])
    ref = orc.Oracle(L, 1, init=False)
    for s0 in (inputs.all_up(L), inputs.slab(L, 2, 5, L // 2), inputs.neel(L)):
        w = inputs.pack_spins(s0)
        sim.set_state(w, 0)
        ref.import_words(w, 0)
        _check_radial(sim.measure_radial(), ref.measure_radial())
    sim.free()


def test_radial_estimator_large_identities(B):
    """L = 1024 (8.6 GB field): what holds at any size -- P(0) = N in bin 0, S(k = 0) = N m^2,
    Parseval through the bins that are complete, C_rad(0) = 1 - m^2."""
    L = 1024
    sim = B.Ising3D(L, [3])
    sim.sweep(10)
    r = sim.measure_radial()
    m = sim.measure()
    N = L ** 3
    mag = (2.0 * float(m["n_up"][0]) - N) / N
    assert int(r["corr_sum"][0][0]) == N and int(r["shell"][0]) == 1 and int(r["shell"][1]) == 18
    assert abs(r["C_rad"][0][0] - (1.0 - mag * mag)) < 1e-12
    assert abs(r["S_rad"][0][0] - N * mag * mag) <= 1e-9 * max(1.0, N * mag * mag)
    # the radial C and the axis-averaged C agree to a few per cent at short distance
    assert abs(r["C_rad"][0][1] - m["C"][0][1]) < 0.1
    assert abs(r["ell"][0] - m["ell"][0]) < 0.25 * m["ell"][0]
    import torch
    free0 = torch.cuda.mem_get_info()[0]
    sim.release_radial()                               # 8.6 GB field + work area go back
    assert torch.cuda.mem_get_info()[0] > free0 + 8 * 2 ** 30
    r2 = sim.measure_radial()                          # and are re-created on demand
    assert np.array_equal(r2["corr_sum"], r["corr_sum"])
    assert 0.0 < sim.radial_rounding < 1e-2
    print("radial rounding margin at L=%d: %.3e" % (L, sim.radial_rounding))
    sim.free()


@pytest.mark.slow
def test_radial_estimator_L2048_rounding_margin(B):
    """D12 claims the inverse transform of +-1 data at L = 2048 is within 1e-3 of an integer multiple of
    N, so llrint recovers P(d) exactly: measured here (64 GiB field + cuFFT work area), together with
    the identities that hold at any size."""
    import gc
    import torch
    gc.collect()
    torch.cuda.empty_cache()          # 128 GiB are needed: give back what torch cached for earlier tests
    L = 2048
    sim = B.Ising3D(L, [4])
    sim.sweep(20)
    r = sim.measure_radial()
    N = L ** 3
    assert int(r["corr_sum"][0][0]) == N and int(r["shell"][0]) == 1 and int(r["shell"][1]) == 18
    dev = sim.radial_rounding
    print("radial rounding margin at L=2048: %.3e" % dev)
    assert 0.0 < dev < 1e-2
    sim.free()


# ------------------------------------------------------------------ f-4: finite-temperature Glauber
@pytest.mark.parametrize("L,seed,T,cps", [(64, 1, 4.0, [1, 2, 5]), (64, 2, 1.5, [1, 4]), (64, 3, 0.3, [2]),
                                          (128, 7, 4.51, [1, 3]), (192, 8, 2.0, [2]), (64, 9, 1e9, [1, 3]),
                                          # L % 256 == 0: the kernel's 128-bit branch (kernels_generic.cuh, WPR % 4 == 0);
                                          # L = 256 has one 128-spin group per row (previous = next = itself), L = 512 two;
                                          # T = 0.3 makes p(n = 6) round to 1, i.e. the threshold 2^32 (bit 32 of D13's table)
                                          (256, 11, 0.3, [1, 3]), (256, 12, 4.51, [1, 2]),
                                          (512, 13, 0.5, [1, 2]), (512, 14, 3.0, [1, 2])])
def test_glauber_against_oracle(B, orc, L, seed, T, cps):
    sim = B.Ising3D(L, [seed])
    sim.set_temperature(T)
    assert sim.variant_name == "glauber"
    ref = orc.Oracle(L, seed)
    t = 0
    for cp in cps:
        sim.sweep(cp - t)
        ref.sweep_T(cp - t, T)
        t = cp
        assert np.array_equal(sim.get_state(), ref.export_words()), "state differs at sweep %d" % cp
    check_measure(sim.measure(), ref.measure_full())
    # back to T = 0: the quench continues with the paper's rule
    sim.set_temperature(0.0)
    assert sim.variant_name != "glauber"
    sim.sweep(2)
    ref.sweep(2)
    assert np.array_equal(sim.get_state(), ref.export_words())
    sim.free()


@pytest.mark.parametrize("L,T", [(256, 0.5), (256, 4.0), (512, 1.5)])
def test_glauber_vector_branch_from_coarse_state_and_batch(B, orc, L, T):
    """The 128-bit branch of the Glauber kernel (L % 256 == 0) on a domain-like state entered through
    set_state at a late sweep index, every word against orc_sweep_T (eq. (5)); at L = 256
    also as a batch, whose replicas must equal single lattices."""
    words = inputs.coarse_words(L, 21, block=16)
    sim = B.Ising3D(L, [77])
    sim.set_temperature(T)
    sim.set_state(words, 12_345)
    assert sim.variant_name == "glauber"
    ref = orc.Oracle(L, 77, init=False)
    ref.import_words(words, 12_345)
    sim.sweep(2)
    ref.sweep_T(2, T)
    assert np.array_equal(sim.get_state(), ref.export_words())
    check_measure(sim.measure(), ref.measure_full())
    sim.free()
    if L == 256:
        seeds = [5, 6]
        batch = B.Ising3D(L, seeds)
        batch.set_temperature(T)
        batch.sweep(2)
        st = batch.get_state().reshape(2, -1)
        for i, sd in enumerate(seeds):
            r = orc.Oracle(L, sd)
            r.sweep_T(2, T)
            assert np.array_equal(st[i], r.export_words())
        batch.free()


def test_glauber_batch_and_errors(B, orc):
    L, seeds, T = 64, [100, 101, 163], 3.0
    batch = B.Ising3D(L, seeds)
    batch.set_temperature(T)
    batch.sweep(3)
    st = batch.get_state().reshape(3, -1)
    for i, s in enumerate(seeds):
        ref = orc.Oracle(L, s)
        ref.sweep_T(3, T)
        assert np.array_equal(st[i], ref.export_words())
    with pytest.raises(B.Ising3DError):
        batch.set_temperature(-1.0)
    with pytest.raises(B.Ising3DError):
        batch.set_temperature(float("nan"))
    with pytest.raises(B.Ising3DError):
        batch.set_cycle(B.CYCLE_MIXED)            # T > 0 runs the 01 cycle only
    batch.free()


def test_glauber_full_size_properties(B):
    """L = 1024 at T = 2: properties that hold at any size -- first half-sweep from the all-up
    state flips a fraction p(0) of colour 0 and leaves colour 1 alone (closed form, binomial)."""
    import math
    L, T = 1024, 2.0
    sim = B.Ising3D(L, [5], variant=B.VARIANT_GENERIC)
    sim.set_temperature(T)
    words = np.full(L ** 3 // 32, 0xFFFFFFFF, dtype=np.uint32)
    sim.set_state(words, 0)
    sim.sweep(1)
    m = sim.measure()
    N = L ** 3
    p0 = 1.0 / (1.0 + math.exp(12.0 / T))
    # after one full sweep from all-up nearly all flips are isolated (p0 = 2.5e-3): the number of
    # down spins is N p0 up to corrections of relative order 6 p0 and binomial noise
    n_down = N - int(m["n_up"][0])
    assert abs(n_down - N * p0) < 0.05 * N * p0
    sim.free()


# ------------------------------------------------------------------ f-2: double checkerboard
@pytest.mark.parametrize("L,seed,variant,cps", [(64, 1, "auto", [1, 2, 6]), (128, 7, "auto", [1, 5]),
                                                (256, 2, "auto", [2, 4]), (192, 8, "auto", [1, 3]),
                                                (64, 3, "generic", [1, 4]), (512, 11, "auto", [1, 2, 5]),
                                                (512, 12, "generic", [1, 2]), (512, 13, "fused2", [3])])
def test_double_checkerboard_against_oracle(B, orc, L, seed, variant, cps):
    sim = B.Ising3D(L, [seed], variant=VARIANTS(B)[variant])
    sim.set_cycle(B.CYCLE_DOUBLE_CB)
    want = {"generic": "generic", "fused2": "fused2"}.get(variant, "fused2" if L in (512, 1024, 2048, 4096) else
                                                          "resident" if L <= 256 and L != 192 else "generic")
    assert sim.variant_name == want
    ref = orc.Oracle(L, seed)
    t = 0
    for cp in cps:
        sim.sweep(cp - t)
        ref.sweep_dcb(cp - t, block=8)
        t = cp
        assert np.array_equal(sim.get_state(), ref.export_words()), "state differs at sweep %d" % cp
    if L <= 256:
        check_measure(sim.measure(), ref.measure_full())
    sim.set_cycle(B.CYCLE_01)                      # and back to the main-text cycle
    sim.sweep(1)
    ref.sweep(1)
    assert np.array_equal(sim.get_state(), ref.export_words())
    sim.free()


def test_double_checkerboard_batch_neel_and_errors(B, orc):
    L = 128
    batch = B.Ising3D(L, [100, 163])
    batch.set_cycle(B.CYCLE_DOUBLE_CB)
    batch.sweep(3)
    st = batch.get_state().reshape(2, -1)
    for i, s in enumerate((100, 163)):
        ref = orc.Oracle(L, s)
        ref.sweep_dcb(3, block=8)
        assert np.array_equal(st[i], ref.export_words())
    batch.free()
    sim = B.Ising3D(1024, [1])
    sim.set_cycle(B.CYCLE_DOUBLE_CB)
    with pytest.raises(B.Ising3DError):
        sim.set_variant(B.VARIANT_FUSED3)
    with pytest.raises(B.Ising3DError):
        sim.set_variant(B.VARIANT_ACTIVE)
    with pytest.raises(B.Ising3DError):
        sim.set_temperature(2.0)
    sim.free()


@pytest.mark.parametrize("L,seed,mixed", [(1024, 21, 0), (2048, 22, 0), (1024, 23, 1), (2048, 24, 1)])
def test_double_checkerboard_fused2_full_size(B, orc, L, seed, mixed):
    """The masked fused2 launches (01 cycle: one per coarse colour; mixed cycle: one per coarse colour
    and drawn fine order) against the masked generic kernel word for word, and at L = 1024 against
    the whole-lattice oracle from the iid start and from a late-time-like state."""
    cyc = B.CYCLE_DOUBLE_CB_MIXED if mixed else B.CYCLE_DOUBLE_CB
    a = B.Ising3D(L, [seed])
    a.set_cycle(cyc)
    b = B.Ising3D(L, [seed], variant=B.VARIANT_GENERIC)
    b.set_cycle(cyc)
    assert a.variant_name == "fused2" and b.variant_name == "generic"
    a.sweep(2)
    b.sweep(2)
    assert np.array_equal(a.get_state(), b.get_state())
    if L == 1024:
        ref = orc.Oracle(L, seed)
        step = (lambda n: ref.sweep_dcb_mixed(n, block=8)) if mixed else (lambda n: ref.sweep_dcb(n, block=8))
        step(2)
        assert np.array_equal(a.get_state(), ref.export_words())
        words = inputs.coarse_words(L, 5, block=16)
        a.set_state(words, 700)
        ref.import_words(words, 700)
        a.sweep(1)
        step(1)
        assert np.array_equal(a.get_state(), ref.export_words())
    a.free()
    b.free()


@pytest.mark.parametrize("L,seed,variant,cps", [(64, 1, "auto", [1, 2, 6]), (128, 7, "auto", [1, 4]), (192, 8, "auto", [2]),
                                                (512, 11, "auto", [1, 2, 5]), (512, 12, "generic", [1, 3])])
def test_double_checkerboard_mixed_against_oracle(B, orc, L, seed, variant, cps):
    sim = B.Ising3D(L, [seed], variant=VARIANTS(B)[variant])
    sim.set_cycle(B.CYCLE_DOUBLE_CB_MIXED)
    assert sim.variant_name == ("fused2" if (L >= 512 and variant == "auto") else "generic")
    ref = orc.Oracle(L, seed)
    t = 0
    for cp in cps:
        sim.sweep(cp - t)
        ref.sweep_dcb_mixed(cp - t, block=8)
        t = cp
        assert np.array_equal(sim.get_state(), ref.export_words()), "state differs at sweep %d" % cp
    if L <= 192:
        check_measure(sim.measure(), ref.measure_full())
    sim.set_cycle(B.CYCLE_01)
    sim.sweep(1)
    ref.sweep(1)
    assert np.array_equal(sim.get_state(), ref.export_words())
    sim.free()


def test_double_checkerboard_mixed_batch_and_errors(B, orc):
    L, seeds = 64, [100, 101, 163]
    batch = B.Ising3D(L, seeds)
    batch.set_cycle(B.CYCLE_DOUBLE_CB_MIXED)
    batch.sweep(4)
    st = batch.get_state().reshape(3, -1)
    for i, s in enumerate(seeds):
        ref = orc.Oracle(L, s)
        ref.sweep_dcb_mixed(4, block=8)
        assert np.array_equal(st[i], ref.export_words())
    with pytest.raises(B.Ising3DError):
        batch.set_variant(B.VARIANT_RESIDENT)
    batch.free()
