"""paper_2205_00095_b200 -- B200-native (sm_100a, fp64) hot path of the DG relativistic-hydro
method of arxiv 2205.00095: one SSP-RK stage behind the C-ABI of ``include/dgrhd.h``.

``inputs``   seeded synthetic workloads (primitives only; serves oracle and CUDA path alike)
``binding``  thin ctypes binding over ``libdgrhd.so`` (argument marshalling only)

The CUDA library is loaded lazily on first use and its absence is a hard error: there is no CPU
fallback anywhere in this package.
"""
from . import inputs  # noqa: F401

__all__ = ["inputs", "binding"]


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
