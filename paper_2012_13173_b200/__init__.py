"""B200-native HCGrid hot path (arXiv 2012.13173): HEALPix-ring pre-ordering and
gather-style Gaussian convolution gridding as sm_100a CUDA behind a C-ABI library.

`HCGrid` (binding.py) is the thin Python binding over include/hcgrid.h;
`workloads` holds the seeded synthetic input generators.  Importing the package is
cheap; the CUDA library is loaded on first use and its absence is a hard error.
"""
__all__ = ["HCGrid", "HCGridError", "load_library", "workloads"]


def __getattr__(name):
    if name in ("HCGrid", "HCGridError", "load_library"):
        from . import binding
        return getattr(binding, name)
    if name == "workloads":
        import importlib
        return importlib.import_module(".workloads", __name__)
    raise AttributeError(name)
