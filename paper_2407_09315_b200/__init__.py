"""B200-native random batch Ewald (RBE) k-space force: Eq. (2.9) + Eq. (2.12) of arxiv 2407.09315.

``rbe`` (the ctypes binding of csrc/librbe.so) is imported lazily so that ``inputs`` -- the
seeded synthetic generators, numpy only -- can be used on a box without the CUDA library.
"""
__all__ = ["inputs", "rbe"]


def __getattr__(name):
    if name in __all__:
        import importlib

        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
