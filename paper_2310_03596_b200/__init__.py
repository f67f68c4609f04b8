"""B200-native (sm_100a) SPH hot path of arxiv 2310.03596 -- see DESIGN.md.

`workloads` is importable without a GPU; the CUDA binding (`paper_2310_03596_b200.sph`) loads
the C-ABI library lazily and fails loudly if it is missing.
"""
__all__ = ["workloads", "sph"]
