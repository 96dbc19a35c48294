"""nsgpu: B200-native (sm_100a) batched likelihood + nested slice sampling (arXiv 2509.13307 hot path).

`paper_2509_13307_b200.nsgpu` is the thin Python binding over the C-ABI library (include/nsgpu.h);
`paper_2509_13307_b200.workloads` holds the seeded synthetic inputs.  Importing this package does not
load the CUDA library; `nsgpu.lib()` does, and fails loudly if it is missing.
"""
__all__ = ["workloads", "nsgpu"]
