"""GPU parity of the activity-driven sweep (kernels_active.cuh, ISING3D_VARIANT_ACTIVE and the
AUTO policy) and of ising3d_activity, against the CPU oracle: the trajectory must be the dense
kernels' bit for bit (eq. (6) PAPER.md:105-108 leaves a group without a Delta E <= 0 site
unchanged whatever its random bits are), and the activity count is an exact integer."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2305_12161_b200 import inputs  # noqa: E402


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


def _states(L):
    """(name, packed words): an iid start, late-time-like domain states, structured states."""
    return [
        ("domains16", inputs.pack_spins(inputs.domain_spins(L, 5, block=16, p_minority=0.15))),
        ("domains32_noise", inputs.pack_spins(inputs.domain_spins(L, 6, block=32, p_minority=0.3, noise=0.002))),
        ("coarse8", inputs.coarse_words(L, 3)),
        ("cube", inputs.pack_spins(inputs.cube(L, L - 1, L - 1, L - 1, 2))),      # across all three wraps
        ("slab", inputs.pack_spins(inputs.slab(L, 0, L - 3, 7))),                 # flat interfaces normal to x
        ("all_up", inputs.pack_spins(inputs.all_up(L))),
    ]


def test_activity_counts_equal_oracle(B, orc):
    """ising3d_activity == orc_activity (groups holding a Delta E <= 0 site, per colour)."""
    L = 256
    G = L ** 3 // 256
    sim = B.Ising3D(L, [2])
    ref = orc.Oracle(L, 2)
    for t in (0, 3, 20):
        sim.sweep(t - sim.sweep_count)
        ref.sweep(t - ref.sweep_count)
        got, frac = sim.activity()
        want = ref.activity()
        assert list(got[0]) == list(want), "t=%d" % t
        assert abs(frac - (int(want[0]) + int(want[1])) / (2.0 * G)) < 1e-15
        assert np.array_equal(sim.get_state(), ref.export_words())       # counting changes nothing
    seen = []
    for name, words in _states(L):
        sim.set_state(words, 100)
        ref.import_words(words, 100)
        got, _ = sim.activity()
        want = ref.activity()
        assert list(got[0]) == list(want), name
        seen.append(int(want[0]) + int(want[1]))
    assert seen[-1] == 0 and min(seen[:-2]) > 0 and max(seen) < 2 * G      # non-trivial counts
    sim.free()


@pytest.mark.parametrize("cycle", ["01", "mixed"])
def test_active_sweep_against_oracle_L256(B, orc, cycle):
    """The activity-driven kernel from the T = infinity start (every group awake) and from
    late-time-like states (few groups awake), every checkpoint against the oracle."""
    L = 256
    sim = B.Ising3D(L, [9], variant=B.VARIANT_ACTIVE)
    assert sim.variant_name == "active"
    if cycle == "mixed":
        sim.set_cycle(B.CYCLE_MIXED)
    ref = orc.Oracle(L, 9)
    step = ref.sweep if cycle == "01" else ref.sweep_mixed
    for cp in (1, 2, 5, 12):
        sim.sweep(cp - sim.sweep_count)
        step(cp - ref.sweep_count)
        assert np.array_equal(sim.get_state(), ref.export_words()), "random start, sweep %d" % cp
    for name, words in _states(L):
        sim.set_state(words, 1000)
        ref.import_words(words, 1000)
        for cp in (1001, 1002, 1005, 1012, 1030):
            sim.sweep(cp - sim.sweep_count)
            step(cp - ref.sweep_count)
            assert np.array_equal(sim.get_state(), ref.export_words()), "%s, sweep %d" % (name, cp)
    got, want = sim.measure(), ref.measure_full()
    assert int(got["n_up"][0]) == want["n_up"] and np.array_equal(got["antipar"][0], want["antipar"])
    sim.free()


def test_active_sweep_against_oracle_L512_batch(B, orc):
    """Rows of two groups (x-edge wake-ups cross groups), two replicas in one handle."""
    L = 512
    seeds = [31, 32]
    sim = B.Ising3D(L, seeds, variant=B.VARIANT_ACTIVE)
    w0 = inputs.pack_spins(inputs.domain_spins(L, 7, block=32, p_minority=0.2, noise=0.001))
    w1 = inputs.coarse_words(L, 8, block=16)
    sim.set_state(np.concatenate([w0, w1]), 500)
    refs = [orc.Oracle(L, s, init=False) for s in seeds]
    refs[0].import_words(w0, 500)
    refs[1].import_words(w1, 500)
    for cp in (501, 503, 508):
        sim.sweep(cp - sim.sweep_count)
        got = sim.get_state().reshape(2, -1)
        for r in range(2):
            refs[r].sweep(cp - refs[r].sweep_count)
            assert np.array_equal(got[r], refs[r].export_words()), "replica %d, sweep %d" % (r, cp)
    cnt, _ = sim.activity()
    for r in range(2):
        assert list(cnt[r]) == list(refs[r].activity())
    sim.free()


def test_auto_policy_switches_and_keeps_the_trajectory(B, orc):
    """AUTO at L = 512 with a short probe interval: a late-time-like state switches to the
    activity-driven kernel, an iid state stays on fused2, and either way the states equal the
    oracle's; interleaving dense and activity-driven sweeps (flags rebuilt) changes nothing.
    The probes do not block the host: a switch shows once the probe has landed, i.e. for certain
    after a call that waits for the stream (sync, get_state); whether the sweeps queued in between
    ran dense or activity-driven is a matter of timing and must not show in the state."""
    L = 512
    sim = B.Ising3D(L, [41])
    sim.set_activity_policy(4, 0.5, 0.9)
    assert sim.variant_name == "fused2" and sim.last_activity == -1.0
    ref = orc.Oracle(L, 41)
    sim.sweep(9)                                   # iid start: probes at 4 and 8 see every group awake
    ref.sweep(9)
    sim.sync()
    assert sim.variant_name == "fused2" and sim.last_activity > 0.9
    assert np.array_equal(sim.get_state(), ref.export_words())
    words = inputs.pack_spins(inputs.domain_spins(L, 11, block=32, p_minority=0.2, noise=0.0005))
    sim.set_state(words, 200)
    ref.import_words(words, 200)
    assert sim.variant_name == "fused2"            # set_state voids the history
    sim.sweep(3)
    sim.sync()
    assert sim.variant_name == "fused2"            # no probe yet
    sim.sweep(1)                                   # the probe after sweep 4 ...
    sim.sync()                                     # ... has landed now
    assert sim.variant_name == "active" and 0.0 < sim.last_activity < 0.5
    sim.sweep(2)
    ref.sweep(6)
    assert np.array_equal(sim.get_state(), ref.export_words())
    sim.sweep(11)                                  # tallies read after 4 and 8 active sweeps: still few groups
    ref.sweep(11)
    assert np.array_equal(sim.get_state(), ref.export_words())
    assert sim.variant_name == "active" and 0.0 < sim.last_activity < 0.5
    # forced dense, then AUTO again (the flags are rebuilt at the next probe)
    sim.set_variant(B.VARIANT_FUSED2)
    sim.sweep(2)
    sim.set_variant(B.VARIANT_AUTO)
    assert sim.variant_name == "fused2"
    sim.sweep(7)
    ref.sweep(9)
    assert np.array_equal(sim.get_state(), ref.export_words())
    assert sim.variant_name == "active"
    got, want = sim.measure(), ref.measure_full()
    assert int(got["n_up"][0]) == want["n_up"] and np.array_equal(got["antipar"][0], want["antipar"])
    # handing back: an iid state set into an active handle goes dense again
    sim.set_state(inputs.random_words(L, 1, 5), 0)
    sim.sweep(4)
    sim.sync()
    assert sim.variant_name == "fused2"
    sim.free()


def test_auto_hands_back_when_activity_grows(B, orc):
    """The way back, active -> fused2, taken by the policy itself (no set_state, no set_variant in
    between): a 64^3 cube of up spins in a down sea starts with 8 groups that can change (its corners,
    Delta E = 0) and erodes into ever more kinks -- 5e-5 of the groups after 4 sweeps, 1e-4 after 12,
    3e-4 after 36 (counted with the oracle).  With on_below = 7e-5 and off_above = 2e-4 the handle
    goes activity-driven at the first probe and must come back to fused2 by itself once the kernel's
    own tally passes off_above; the trajectory is the oracle's throughout (eq. (6))."""
    L = 512
    words = inputs.pack_spins(inputs.cube(L, 100, 100, 100, 64))
    sim = B.Ising3D(L, [9])
    sim.set_activity_policy(4, 7e-5, 2e-4)
    sim.set_state(words, 0)
    seen, fracs, t = [], [], 0
    for _ in range(24):
        sim.sweep(4)
        sim.sync()                     # the probe queued after these 4 sweeps has landed
        t += 4
        seen.append(sim.variant_name)
        fracs.append(sim.last_activity)
        if "active" in seen and seen[-2:] == ["fused2", "fused2"]:
            break
    assert seen[0] == "active", (seen, fracs)
    first_back = seen.index("fused2")
    assert first_back >= 2 and set(seen[:first_back]) == {"active"} and set(seen[first_back:]) == {"fused2"}, (seen, fracs)
    assert fracs[first_back] > 2e-4 and all(0.0 < f <= 2e-4 for f in fracs[:first_back]), fracs
    ev = sim.active_stats()[0]
    assert ev[0] > 0 and ev[1] > 0      # the activity-driven kernel did run and did change groups
    ref = orc.Oracle(L, 9, init=False)
    ref.import_words(words, 0)
    ref.sweep(t)
    assert np.array_equal(sim.get_state(), ref.export_words())
    assert list(sim.activity()[0][0]) == list(ref.activity())
    sim.free()


def test_auto_long_call_hands_over_on_its_own(B):
    """One ising3d_sweep(5000) call under the default policy on a late-time state (config 4 at
    t = 50 000, where under 11 % of the groups can change): nothing in the call waits for the GPU,
    the probe result is picked up between launches, so the hand-over happens inside the call -- seen
    in the launch count (two launches per activity-driven sweep, one per fused2 sweep) -- and the
    state equals that of the same 5000 sweeps on fused2 alone."""
    import torch
    L, seed, t0, n = 1024, 3, 50_000, 5000
    b = B.Ising3D(L, [seed], variant=B.VARIANT_FUSED2)
    b.sweep(t0)
    nw = L ** 3 // 32
    buf = torch.empty(nw, dtype=torch.int32, device="cuda")
    b.get_state_device(buf.data_ptr(), nw)
    a = B.Ising3D(L, [seed])
    a.set_state_device(buf.data_ptr(), nw, t0)
    assert a.variant_name == "fused2"
    before = a.launch_count
    a.sweep(n)
    launches = a.launch_count - before
    b.sweep(n)
    assert launches > n + 1000, "the hand-over did not happen inside the call (%d launches)" % launches
    assert np.array_equal(a.get_state(), b.get_state())
    assert a.variant_name == "active" and 0.0 < a.last_activity < 0.11
    a.free()
    b.free()


def test_default_handle_sweeps_can_be_stream_captured(B):
    """ising3d_sweep under the default (AUTO) policy makes no synchronising call, so it can be
    recorded into a CUDA graph: capture sweep(4) at sweep index t0 on a side stream, replay the graph
    once, and the state equals that of a live sweep(4) from the same state and index (the sweep
    index is a launch argument, so one replay is exactly sweeps t0 .. t0+3; an even count leaves the
    ping-pong buffers where the handle believes them)."""
    import torch
    L, t0 = 512, 700
    words = inputs.coarse_words(L, 31, block=16)
    live = B.Ising3D(L, [77])
    live.set_state(words, t0)
    live.sweep(4)
    want = live.get_state()
    live.free()
    side = torch.cuda.Stream()
    sim = B.Ising3D(L, [77])
    sim.set_activity_policy(2, 0.11, 0.14)      # a probe would fall inside the captured call
    sim.sweep(2)                                # first use of the kernels (function attributes) outside the capture
    sim.sync()
    sim.set_stream(side.cuda_stream)
    sim.set_state(words, t0)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side, capture_error_mode="thread_local"):
        sim.sweep(4)
    assert sim.sweep_count == t0 + 4
    assert np.array_equal(sim.get_state(), words)      # recorded, not run
    g.replay()
    torch.cuda.synchronize()
    assert np.array_equal(sim.get_state(), want)
    sim.sweep(3)                                # and the handle goes on live, probes included
    sim.sync()
    sim.free()


def test_auto_policy_disabled_and_bad_arguments(B):
    sim = B.Ising3D(512, [1])
    sim.set_activity_policy(0)
    sim.set_state(inputs.pack_spins(inputs.all_up(512)), 0)
    sim.sweep(5)
    assert sim.variant_name == "fused2"
    with pytest.raises(B.Ising3DError):
        sim.set_activity_policy(4, 0.5, 0.4)
    with pytest.raises(B.Ising3DError):
        sim.set_activity_policy(4, -0.1, 0.4)
    sim.free()
    small = B.Ising3D(128, [1])
    with pytest.raises(B.Ising3DError):
        small.set_variant(B.VARIANT_ACTIVE)
    with pytest.raises(B.Ising3DError):
        small.activity()
    small.free()


@pytest.mark.slow
def test_active_equals_fused2_at_full_size_late_time(B, orc):
    """Config 5 (L = 2048, seed 4) taken to t = 10^4 on fused2, then 24 sweeps on the
    activity-driven kernel against 24 more fused2 sweeps: every word equal; then two sweeps from
    the t0 state against the whole-lattice oracle, and the activity count."""
    import torch
    L, seed, t0, n = 2048, 4, 10000, 24
    a = B.Ising3D(L, [seed], variant=B.VARIANT_FUSED2)
    a.sweep(t0)
    nw = L ** 3 // 32
    buf = torch.empty(nw, dtype=torch.int32, device="cuda")
    a.get_state_device(buf.data_ptr(), nw)
    b = B.Ising3D(L, [seed], variant=B.VARIANT_ACTIVE)
    b.set_state_device(buf.data_ptr(), nw, t0)
    cnt, frac = b.activity()
    assert 0.05 < frac < 0.6
    a.sweep(n)
    b.sweep(n)
    wa, wb = a.get_state(), b.get_state()
    assert np.array_equal(wa, wb)
    del wa, wb
    # two sweeps from the t0 state against the whole-lattice oracle (8.6 GB of int8 spins)
    ref = orc.Oracle(L, seed, init=False)
    ref.import_words(buf.cpu().numpy().view(np.uint32), t0)
    ref.sweep(2)
    b.set_state_device(buf.data_ptr(), nw, t0)
    b.sweep(2)
    assert np.array_equal(b.get_state(), ref.export_words())
    assert list(b.activity()[0][0]) == list(ref.activity())
    a.free()
    b.free()


@pytest.mark.slow
def test_auto_run_equals_fused2_run_config4(B):
    """Config 4 (L = 1024, seed 3, 10^5 sweeps) run twice: under the AUTO policy (fused2, probes every
    1024 sweeps, hand-over to the activity-driven kernel when under 11 % of the groups can change)
    and on fused2 alone.  Every word of the final states and all counts must agree, and AUTO must
    have handed over on the way."""
    L, seed, n = 1024, 3, 100_000
    a = B.Ising3D(L, [seed])
    b = B.Ising3D(L, [seed], variant=B.VARIANT_FUSED2)
    a.sweep(n)
    b.sweep(n)
    a.sync()
    assert a.variant_name == "active" and b.variant_name == "fused2"
    assert 0.0 < a.last_activity < 0.11
    ev = a.active_stats()[0]
    assert ev[0] > 0 and ev[1] > 0
    assert np.array_equal(a.get_state(), b.get_state())
    ma, mb = a.measure(), b.measure()
    assert int(ma["n_up"][0]) == int(mb["n_up"][0]) and np.array_equal(ma["antipar"], mb["antipar"])
    a.free()
    b.free()


def test_auto_policy_batch_of_two(B, orc):
    """Two replicas in one handle at L = 512 under AUTO: the hand-over follows the mean awake
    fraction, each replica keeps its own trajectory (seed) and equals the oracle."""
    L, seeds = 512, [51, 52]
    sim = B.Ising3D(L, seeds)
    sim.set_activity_policy(3, 0.6, 0.95)
    w = [inputs.pack_spins(inputs.domain_spins(L, 21, block=32, p_minority=0.25, noise=0.0005)),
         inputs.coarse_words(L, 22, block=16)]
    sim.set_state(np.concatenate(w), 40)
    refs = [orc.Oracle(L, s, init=False) for s in seeds]
    for r, ww in zip(refs, w):
        r.import_words(ww, 40)
    sim.sweep(8)
    got = sim.get_state().reshape(2, -1)
    assert sim.variant_name == "active"
    for i, r in enumerate(refs):
        r.sweep(8)
        assert np.array_equal(got[i], r.export_words()), "replica %d" % i
    cnt, frac = sim.activity()
    for i, r in enumerate(refs):
        assert list(cnt[i]) == list(r.activity())
    assert 0.0 < frac < 0.6
    sim.free()


def test_active_equals_fused2_L4096(B):
    """The largest size (6.9e10 spins, rows of 16 groups, group indices up to 2^28): the activity-driven
    kernel against fused2 word for word, from a state 30 sweeps into the quench (most groups awake)
    and from the all-up state with a handful of reversed words (a few groups awake)."""
    import torch
    L = 4096
    nw = L ** 3 // 32
    a = B.Ising3D(L, [8], variant=B.VARIANT_FUSED2)
    b = B.Ising3D(L, [8], variant=B.VARIANT_ACTIVE)
    a.sweep(30)
    buf = torch.empty(nw, dtype=torch.int32, device="cuda")
    a.get_state_device(buf.data_ptr(), nw)
    b.set_state_device(buf.data_ptr(), nw, 30)
    a.sweep(2)
    b.sweep(2)
    a.get_state_device(buf.data_ptr(), nw)
    ref = buf.clone()
    b.get_state_device(buf.data_ptr(), nw)
    b.sync()
    assert torch.equal(ref, buf)
    # sparse: all up, then reversed words at the first and last group of each colour and in the middle
    buf.fill_(-1)
    idx = torch.tensor([0, 5, nw // 2 - 1, nw // 2, nw // 2 + 7, nw - 1, nw // 3, 3 * (nw // 4) + 2], device="cuda")
    buf[idx] = 0x0F0F1234
    a.set_state_device(buf.data_ptr(), nw, 100)
    b.set_state_device(buf.data_ptr(), nw, 100)
    cnt, frac = b.activity()
    assert 0 < int(cnt.sum()) < 200
    a.sweep(5)
    b.sweep(5)
    a.get_state_device(buf.data_ptr(), nw)
    ref = buf.clone()
    b.get_state_device(buf.data_ptr(), nw)
    b.sync()
    assert torch.equal(ref, buf)
    a.free()
    b.free()
