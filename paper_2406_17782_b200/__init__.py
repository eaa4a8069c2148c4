"""nbsdf -- B200-native (sm_100a) neural woven-fabric BSDF decoder (arXiv 2406.17782 hot path).

The product is ``libnbsdf.so`` (C ABI in ``include/nbsdf.h``); :mod:`.api` is a thin ctypes binding
with the same call names, :mod:`.synth` the seeded synthetic inputs.  Imports are lazy so that the
input generators can be used without torch or the CUDA library.
"""
import importlib

_LAZY = {"api", "synth", "buildlib"}


def __getattr__(name):
    if name in _LAZY:
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
