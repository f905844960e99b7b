"""B200-native Generalized Source Method hot path (arxiv 1501.01752): C-ABI CUDA library + thin binding.

`from paper_1501_01752_b200 import gsm` loads the CUDA library (and fails loudly if it is not built);
`paper_1501_01752_b200.workloads` holds only seeded input generators.
"""
__all__ = ["gsm", "workloads", "build"]
