"""ising3d_measure_static: the measurement for callers that must not allocate on the GPU.

Some users of the library want N_up and A_mu(r) at a point where device memory is not theirs to
take: every byte of the GPU already belongs to a pool they do not control (a framework's caching
allocator, a scheduler's per-tenant budget), or they sit on a path where the device-wide stall of a
cudaMalloc / cudaFree would hold up every other stream (an analysis hook between sweeps of a running
job).  The entry point keeps the kernels' 64-bit accumulators in an array that is part of
libising3d.so itself; the caller passes the spins (device) and the result arrays (host), nothing more.

What is checked here, on two calls in a row so that whatever the first call left in the shared
array cannot leak into the second: the integers equal those of the handle-based ising3d_measure
(the tests' tolerance for integer counts is equality), for a batch and then for a single lattice of
another size; a repeat of a call gives the same answer; the GPU's free memory does not move across
a call; a request beyond ISING3D_STATIC_MAX_COUNTS is refused with a message that says so.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure of this
optional entry point must not hide the parity tests of the main path.
"""
import ctypes as C

import numpy as np
import pytest


@pytest.fixture(scope="module")
def B():
    from paper_2305_12161_b200 import build, binding
    build.build()
    return binding


def _device_copy(sim):
    """The handle's packed state in a torch tensor (the allocation is the test's, not the library's)."""
    import torch
    n_words = sim.n_rep * sim.L ** 3 // 32
    t = torch.empty(n_words, dtype=torch.int32, device="cuda")
    sim.get_state_device(t.data_ptr(), n_words)
    sim.sync()
    return t


@pytest.mark.gpu
def test_static_measure_equals_handle_measure_twice_in_a_row(B):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    stream = torch.cuda.current_stream().cuda_stream

    # first call: a batch of three L=128 lattices, 20 sweeps into the quench
    a = B.Ising3D(128, [100, 101, 102])
    a.sweep(20)
    want_a = a.measure()
    words_a = _device_copy(a)
    got_a = B.measure_static(words_a.data_ptr(), 128, 3, stream)
    assert np.array_equal(got_a["n_up"], want_a["n_up"])
    assert np.array_equal(got_a["antipar"], want_a["antipar"])
    assert np.all(got_a["antipar"][:, :, 0] == 0)

    # second call, right after it: one L=192 lattice (another shape, so the counters of the first
    # call sit under and beyond the ones this call uses) -- through the popcount handle path too
    b = B.Ising3D(192, [7])
    b.sweep(3)
    b.set_measure_variant(B.MEASURE_POPCOUNT)
    want_b = b.measure()
    words_b = _device_copy(b)
    got_b = B.measure_static(words_b.data_ptr(), 192, 1, stream)
    assert np.array_equal(got_b["n_up"], want_b["n_up"])
    assert np.array_equal(got_b["antipar"], want_b["antipar"])
    n_broken = got_b["antipar"][0, :, 1].sum()
    assert int(n_broken) == int(want_b["n_broken"][0])

    # the first input again: same answer as before, and the device's free memory does not move
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    again = B.measure_static(words_a.data_ptr(), 128, 3, stream)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert np.array_equal(again["n_up"], want_a["n_up"])
    assert np.array_equal(again["antipar"], want_a["antipar"])
    assert free_after == free_before, "ising3d_measure_static changed the device's free memory"

    # a tensor-core-shaped lattice (L = 512: the handle takes the Gram path) gives the same counts
    c = B.Ising3D(512, [3])
    c.sweep(2)
    want_c = c.measure()
    assert c.measure_variant_name == "tensor"
    words_c = _device_copy(c)
    got_c = B.measure_static(words_c.data_ptr(), 512, 1, stream)
    assert np.array_equal(got_c["n_up"], want_c["n_up"])
    assert np.array_equal(got_c["antipar"], want_c["antipar"])
    for h in (a, b, c):
        h.free()


def test_static_measure_refuses_what_does_not_fit(B):
    """Argument checks come before any CUDA call, so they run without a GPU."""
    lib = B.load()
    fake = C.c_void_p(0x10000)                  # never dereferenced: the call must fail first
    n_up = (C.c_uint64 * 64)()
    ap = (C.c_uint64 * 8)()
    # 64 x L=256 needs 64 * 388 = 24 832 counters > 16 384
    assert 64 * (1 + 3 * 129) > B.STATIC_MAX_COUNTS
    assert lib.ising3d_measure_static(fake, 256, 64, n_up, ap, None) == B.EINVAL
    msg = lib.ising3d_last_error().decode()
    assert "24832" in msg and str(B.STATIC_MAX_COUNTS) in msg and "static scratch" in msg
    # every supported single lattice and the 64 x L=128 batch of config 3 fit
    assert 1 + 3 * (4096 // 2 + 1) <= B.STATIC_MAX_COUNTS
    assert 64 * (1 + 3 * 65) <= B.STATIC_MAX_COUNTS
    assert lib.ising3d_measure_static(fake, 100, 1, n_up, ap, None) == B.EINVAL      # bad L
    assert lib.ising3d_measure_static(fake, 64, 0, n_up, ap, None) == B.EINVAL       # bad n_rep
    assert lib.ising3d_measure_static(None, 64, 1, n_up, ap, None) == B.EINVAL
    assert lib.ising3d_measure_static(fake, 64, 1, None, ap, None) == B.EINVAL
    assert lib.ising3d_measure_static(C.c_void_p(0x10004), 64, 1, n_up, ap, None) == B.EINVAL
    assert b"16-byte" in lib.ising3d_last_error()
