"""B200-native exact-exchange apply (arxiv 2501.16572 hot path): thin Python binding over libexx.so.

    from paper_2501_16572_b200 import exx, workloads

Importing the package (or ``exx``) never loads the CUDA library, so ``workloads`` is usable anywhere;
the first call into the binding does, and fails loudly if libexx.so is missing (no CPU fallback).
"""
