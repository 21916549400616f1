"""CPU-side checks of the C-ABI boundary: the library builds for sm_100a, loads, exports
every symbol include/ising3d.h declares, and its host logic (argument validation, sizes)
behaves as the header says.  No compute call succeeds without a GPU -- and must fail loudly."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2305_12161_b200 import build, binding
    build.build()
    return binding.load()


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "ising3d.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ising3d_[a-z_A-Z0-9]+)\s*\(", src)))


def test_header_symbols_are_exported(lib):
    from paper_2305_12161_b200 import binding
    names = _declared_functions()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), "libising3d.so does not export %s" % n
    assert sorted(binding.EXPORTED) == names


def test_binding_constants_match_the_header():
    """Every ISING3D_* integer constant of the header has the same value in the binding."""
    from paper_2305_12161_b200 import binding
    src = open(os.path.join(ROOT, "include", "ising3d.h")).read()
    defs = dict(re.findall(r"#define\s+ISING3D_([A-Z0-9_]+)\s+\(?(-?\d+)\)?", src))
    assert len(defs) >= 17
    for name, val in defs.items():
        assert getattr(binding, name) == int(val), name


def test_library_is_sm100a_and_uses_bulk_async_copies():
    import shutil
    import subprocess
    from paper_2305_12161_b200 import binding
    if shutil.which("cuobjdump") is None:
        pytest.skip("cuobjdump not on PATH")
    out = subprocess.run(["cuobjdump", "-lelf", binding.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    sass = subprocess.run(["cuobjdump", "-sass", binding.LIB_PATH], capture_output=True, text=True).stdout
    assert "UBLKCP" in sass          # cp.async.bulk (TMA engine) feeds the fused sweep kernel
    assert "LOP3" in sass and "IMAD.WIDE.U32" in sass


def test_sizes_and_validation(lib):
    for L in (64, 128, 192, 256, 1024, 2048, 4096):
        assert lib.ising3d_words_per_replica(L) == L ** 3 // 32
        nb = lib.ising3d_required_bytes(L, 1)
        assert nb >= 2 * (L ** 3 // 8) and nb % 256 == 0
    assert lib.ising3d_required_bytes(128, 64) >= 64 * 2 * (128 ** 3 // 8)
    for L, n in [(0, 1), (32, 1), (100, 1), (4160, 1), (8192, 1), (64, 0), (64, -3), (-64, 1)]:
        assert lib.ising3d_required_bytes(L, n) == 0
    assert lib.ising3d_words_per_replica(100) == 0


def test_bad_arguments_return_einval(lib):
    from paper_2305_12161_b200 import binding
    h = C.c_void_p()
    assert lib.ising3d_init(C.byref(h), 100, 1) == binding.EINVAL
    assert h.value is None                      # *h untouched on failure
    assert b"multiple of 64" in lib.ising3d_last_error()
    assert lib.ising3d_init(None, 64, 1) == binding.EINVAL
    seeds = (C.c_uint64 * 2)(1, 2)
    assert lib.ising3d_init_batch(C.byref(h), 64, 0, seeds) == binding.EINVAL
    assert lib.ising3d_init_batch(C.byref(h), 64, 2, None) == binding.EINVAL
    assert lib.ising3d_init_batch_with_buffer(C.byref(h), 64, 2, seeds, None, 0, None) == binding.EINVAL
    assert lib.ising3d_sweep(None, 1) == binding.EINVAL
    assert lib.ising3d_measure(None, None) == binding.EINVAL
    assert lib.ising3d_get_state(None, None, 0, None) == binding.EINVAL
    assert lib.ising3d_set_variant(None, 0) == binding.EINVAL
    lib.ising3d_free(None)                      # no-op
    assert lib.ising3d_L(None) == 0 and lib.ising3d_sweep_count(None) == 0
    assert lib.ising3d_last_error() is not None


def test_concurrent_callers_keep_their_own_errors(lib):
    """include/ising3d.h: distinct handles are independent, ising3d_last_error is thread-local.
    Eight host threads validate / try to create handles at the same time (no process-wide launch
    plan or attribute cache is left to race on): every thread sees its own error text, *h stays
    untouched, nothing crashes."""
    import threading
    from paper_2305_12161_b200 import binding
    bad = [(100, b"multiple of 64"), (32, b"multiple of 64"), (8192, b"multiple of 64")]
    errors, gate = [], threading.Barrier(8)

    def worker(i):
        try:
            gate.wait()
            for rep in range(200):
                L, text = bad[(i + rep) % len(bad)]
                h = C.c_void_p()
                if (i + rep) % 2:
                    rc = lib.ising3d_init(C.byref(h), L, i)
                    assert rc == binding.EINVAL and h.value is None
                    assert text in lib.ising3d_last_error()
                else:
                    rc = lib.ising3d_sweep(None, 1)
                    assert rc == binding.EINVAL and b"null handle" in lib.ising3d_last_error()
                assert lib.ising3d_required_bytes(64 * (1 + i), 1 + rep % 3) > 0
        except BaseException as e:   # noqa: BLE001
            errors.append((i, repr(e)))

    threads = [threading.Thread(target=worker, args=(i,)) for i in range(8)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors


def test_no_process_wide_launch_state_in_the_library():
    """The launch plans and function-attribute flags live in the handle (struct ising3d), not in
    function-local statics two handles could race on."""
    csrc = os.path.join(ROOT, "paper_2305_12161_b200", "csrc")
    for f in sorted(os.listdir(csrc)):
        txt = re.sub(r"//.*", "", open(os.path.join(csrc, f)).read())
        for m in re.finditer(r"^\s+static\s+(?!constexpr|const\b|_assert|assert)[^;(]*;", txt, flags=re.M):
            raise AssertionError("%s: mutable function-local static: %s" % (f, m.group(0).strip()))
        assert "getenv" not in txt, f


def test_no_cpu_fallback(lib):
    """Without a CUDA device the library must refuse to compute (ECUDA/ENOMEM), never emulate."""
    import torch
    from paper_2305_12161_b200 import binding
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    h = C.c_void_p()
    rc = lib.ising3d_init(C.byref(h), 64, 1)
    assert rc in (binding.ECUDA, binding.ENOMEM) and h.value is None
    assert len(lib.ising3d_last_error()) > 0
    with pytest.raises(binding.Ising3DError):
        binding.Ising3D(64, [1])
    with pytest.raises(binding.Ising3DError):
        binding.Ising3D(64, [1], torch_buffer=False)


def test_product_does_not_import_oracle():
    """The product path never routes through the oracle (and the oracle never imports the product)."""
    pkg = os.path.join(ROOT, "paper_2305_12161_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                for pat in (r"^\s*(from|import)\s+oracle\b", r"liboracle", r"ising_oracle", r"\borc_\w+",
                            r"import_module\([\"']oracle"):
                    assert not re.search(pat, txt, flags=re.M), (f, pat)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2305_12161_b200", txt, flags=re.M), f
            assert "libising3d" not in txt and "ising3d.h" not in txt and "csrc/" not in txt.replace(
                "paper_2305_12161_b200/csrc (", ""), f


def test_measurement_times_and_workloads():
    from paper_2305_12161_b200 import inputs
    assert inputs.measurement_times(100) == [1, 2, 3, 4, 5, 6, 8, 10, 20, 30, 40, 50, 60, 80, 100]
    assert [len(inputs.measurement_times(n)) for n in (2000, 10_000, 100_000, 300_000)] == [23, 29, 36, 38]
    assert len(inputs.WORKLOADS) == 5
    assert inputs.WORKLOADS["config3_64xL128"]["seeds"] == list(range(100, 164))
    w = inputs.random_words(64, 2, 5)
    assert w.dtype == np.uint32 and w.size == 2 * 64 ** 3 // 32
    s = inputs.random_spins(8, 3)
    assert np.array_equal(inputs.unpack_words(inputs.pack_spins(s), 8), s)
