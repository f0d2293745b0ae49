"""B200-native hot path of ODISSEO's direct N-body solver (arxiv 2511.22468).

``workloads`` (seeded input generators) imports no native code; the CUDA library is
loaded on first use of ``binding`` and fails loudly when it is missing.
"""
__all__ = ["workloads", "binding", "sharded", "autograd"]
