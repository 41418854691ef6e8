"""B200-native NEP-ZBL hot path (arXiv 2305.08140): C-ABI CUDA library + thin Python binding.

`from paper_2305_08140_b200 import binding` loads csrc/libnepzbl.so (fails loudly if it is
missing); `workloads` holds only the seeded synthetic input generators.
"""
__all__ = ["binding", "workloads"]
