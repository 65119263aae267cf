"""paper_2205_06649_b200 -- B200-native hot path of the space-time decomposed 4D-Var (DD-4DVar)
of arXiv 2205.06649: hand-written sm_100a CUDA behind a small C-ABI (include/dd4dvar.h), with a
thin ctypes binding.  `synth` holds the seeded input generators (no method arithmetic)."""
from . import synth  # noqa: F401


def __getattr__(name):
    if name in ("DD4DVar", "load_library", "DD4DVarError"):
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)
