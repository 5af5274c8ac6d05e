"""B200-native conjugate-gradient fermion solver of arXiv 1311.2719 (staggered and
Wilson Dslash, M^+M, fused CG) behind the C-ABI of include/lqcd.h.

`synth` (input generators) imports without the CUDA library; everything else is
the binding in `lqcd.py`, loaded on first use, which raises if the library has
not been built (there is no CPU fallback).
"""
_BINDING = ("Lattice", "LqcdError", "library_path", "load_library", "STAGGERED", "WILSON", "EVEN", "ODD",
            "exported_symbols")


def __getattr__(name):
    if name in _BINDING or name == "lqcd":
        import importlib
        mod = importlib.import_module(__name__ + ".lqcd")
        return mod if name == "lqcd" else getattr(mod, name)
    raise AttributeError(name)
