"""B200-native fp64 GRMHD substep library (arXiv 2406.11669 hot path).

`workloads` (seeded input generators) imports without torch/CUDA; everything else is the
ctypes binding of the CUDA library (`binding`), loaded lazily.  There is no CPU fallback.
"""
__all__ = ["Solver", "make_opts", "prim2con_batch", "con2prim_batch", "dfma_peak",
           "maxspeed_noalloc", "lib"]


def __getattr__(name):
    if name in __all__ or name in ("binding",):
        import importlib
        b = importlib.import_module(".binding", __name__)
        return b if name == "binding" else getattr(b, name)
    raise AttributeError(name)
