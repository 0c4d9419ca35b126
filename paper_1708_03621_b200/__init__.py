"""paper_1708_03621_b200: B200-native (sm_100a) H.psi hot path of plane-wave DFT (JDFTx, arXiv 1708.03621).

The product is the C-ABI library libjdft_b200.so (include/jdft.h, csrc/); this package is its build step
(`python -m paper_1708_03621_b200.build`) and a ctypes binding with the same function names (binding.py),
loaded on first attribute access.  No CPU fallback exists: without the built library the binding raises.
"""


import importlib


def __getattr__(name):
    if name.startswith("__"):
        raise AttributeError(name)
    if name in ("build", "binding", "sharding"):  # submodules: `from paper_1708_03621_b200 import build` must not load the .so
        return importlib.import_module(__name__ + "." + name)
    binding = importlib.import_module(__name__ + ".binding")
    try:
        return getattr(binding, name)
    except AttributeError:
        raise AttributeError("module %r has no attribute %r" % (__name__, name)) from None
