"""sp2-b200: B200-native (sm_100a) SP2 / DNN-SP2 density-matrix solver (arXiv 2107.02737).

``from paper_2107_02737_b200 import sp2`` loads the C-ABI CUDA library (and
fails loudly if it is not built); ``inputs`` only draws synthetic Hamiltonians
and can be imported anywhere.  There is no CPU fallback.
"""
__all__ = ["inputs", "sp2"]


def __getattr__(name):
    if name in __all__:
        import importlib

        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
