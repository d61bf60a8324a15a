"""B200-native (sm_100a) explicit finite-volume time step of the 5-/14-moment maximum-entropy
systems with the interpolative closure (arXiv 2401.15233).

`paper_2401_15233_b200.mm` is the thin ctypes binding of the C-ABI in include/mm.h; the work is
done by the CUDA kernels in csrc/ (built in-tree into libmm.so by `build_ext.build()`).
There is no CPU path: importing works anywhere, creating a solver needs a CUDA device.
"""
from . import build_ext  # noqa: F401

__all__ = ["build_ext", "mm"]


def __getattr__(name):
    if name == "mm":
        import importlib
        return importlib.import_module(".mm", __name__)
    raise AttributeError(name)
