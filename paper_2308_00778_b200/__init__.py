"""B200-native (sm_100a) LSQR hot path of the Gaia AVU-GSR solver (arXiv 2308.00778).

``paper_2308_00778_b200.gsr``   -- ctypes binding of the C-ABI library (include/gsr.h)
``paper_2308_00778_b200.synth`` -- seeded synthetic Gaia-shaped inputs (no method arithmetic)

The binding is imported lazily so that the input generator can be used without the CUDA
library (e.g. by the CPU oracle's tests); any use of the solver without the built
``libgsr.so`` fails loudly -- there is no CPU fallback.
"""

__all__ = ["synth", "gsr"]


def __getattr__(name):
    if name in __all__:
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
