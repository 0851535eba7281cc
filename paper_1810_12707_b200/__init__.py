"""B200-native hot path of the pseudo-spectral compressible MHD solver of arXiv 1810.12707 (G-MHD3D).

`inputs`  — seeded synthetic initial conditions (no method arithmetic; shared with the test oracle).
`binding` — thin ctypes binding of the C-ABI library `libmhd.so` (include/mhd.h); argument marshalling
            only, every step of the path runs in the CUDA kernels under `csrc/`.

The binding is imported lazily so that `inputs` stays usable on a box where the CUDA library has not
been built; any attempt to *use* the product path without `libmhd.so` raises (there is no CPU fallback).
"""
from . import inputs  # noqa: F401

__all__ = ["inputs", "binding", "MHD"]


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    if name == "MHD":
        from .binding import MHD
        return MHD
    raise AttributeError(name)
