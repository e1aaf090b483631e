"""B200-native delta-SPH right-hand side and adjoint (diffSPH hot path, arXiv 2507.21684).

The product is the C-ABI shared library built from ``csrc/`` (``include/sph.h``); this package is
the thin Python binding (argument marshalling only) plus the seeded input generators.
Importing the package does not load the CUDA library; the first use of the binding does, and it
fails loudly if the library is missing -- there is no CPU fallback.
"""
__all__ = ["workloads"]


def __getattr__(name):
    if name in ("sph", "Sph", "load_library"):
        from . import binding
        return getattr(binding, {"sph": "Sph", "Sph": "Sph", "load_library": "load_library"}[name])
    raise AttributeError(name)
