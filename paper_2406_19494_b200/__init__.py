"""paper_2406_19494_b200 — B200-native (sm_100a) finite-volume compressible Navier-Stokes hot
path after arxiv/paper_2406_19494: halo fill, WENO5-JS + HLLC, 4th-order viscous/heat flux,
flux divergence, SSP-RK3, CFL reduction, as hand-written CUDA behind the C ABI of include/jf.h.

`binding` (the ctypes layer over libjf.so) is imported lazily so that `cases` (pure numpy input
generators) can be used without the CUDA library.
"""

__all__ = ["cases", "binding"]


def __getattr__(name):
    if name in ("binding", "cases", "build"):
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
