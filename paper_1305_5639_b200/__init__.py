"""paper_1305_5639_b200 -- a B200-native (sm_100a) X-engine for FX software correlators.

The product is the C-ABI library ``libcorr.so`` (``include/corr.h``); this package is the thin
Python binding (argument marshalling only) plus the seeded input generators.
"""
__all__ = ["inputs"]


def __getattr__(name):
    # lazy: importing the package (e.g. for ``inputs``) must not require the CUDA library
    if name in ("Correlator", "CorrError", "lib", "binding"):
        import importlib
        binding = importlib.import_module(__name__ + ".binding")
        return binding if name == "binding" else getattr(binding, name)
    raise AttributeError(name)
