"""B200-native zero-temperature checkerboard sweep of the d=3 Ising model (arXiv 2305.12161).

The product is the C-ABI library libising3d.so (include/ising3d.h, csrc/); `binding` is its
thin ctypes front end, `inputs` the seeded synthetic workloads, `build` the nvcc build step.
"""
from . import inputs  # noqa: F401  (pure numpy, importable without the CUDA library)


def __getattr__(name):
    # the binding (and with it libising3d.so) is loaded on first use and fails loudly if absent
    if name in ("binding", "Ising3D"):
        import importlib
        b = importlib.import_module(".binding", __name__)
        return b if name == "binding" else b.Ising3D
    raise AttributeError(name)
