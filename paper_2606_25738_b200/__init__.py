"""pairhmm-b200: B200-native PairHMM forward (arxiv/paper_2606_25738, "Endeavor").

``paper_2606_25738_b200.binding`` is the thin ctypes layer over the C-ABI library
(include/pairhmm_b200.h); ``paper_2606_25738_b200.workloads`` holds the seeded input generators.
Importing the package does not load the CUDA library; the binding does, and fails loudly
when it is missing (there is no CPU fallback).
"""
__all__ = ["binding", "workloads", "replicas"]
