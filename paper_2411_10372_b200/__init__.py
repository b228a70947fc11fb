"""B200-native MacCormack-TVD step of arXiv 2411.10372.

`inputs` is plain numpy (seeded synthetic states).  `binding` is the thin ctypes layer over the
C-ABI library `libmc_tvd.so` (include/mc_tvd.h); it is imported lazily so that importing the
package never needs the CUDA extension, and it raises loudly if the extension is missing.
"""
from . import inputs  # noqa: F401

__all__ = ["inputs", "binding", "MCTVD", "load_library"]


def __getattr__(name):
    if name in ("binding", "MCTVD", "load_library"):
        import importlib
        mod = importlib.import_module(".binding", __name__)
        return mod if name == "binding" else getattr(mod, name)
    raise AttributeError(name)
