"""B200-native exact-exchange apply (arxiv 2501.16572 hot path): thin Python binding over libexx.so.

``import paper_2501_16572_b200`` never loads the CUDA library (so ``workloads`` is usable
anywhere); the first call into the binding does, and fails loudly if it is missing.
"""
from . import workloads  # noqa: F401


def __getattr__(name):
    if name in ("exx", "Plan", "lib_path", "load_library", "ExxError"):
        from . import exx as _exx
        return _exx if name == "exx" else getattr(_exx, name)
    raise AttributeError(name)
