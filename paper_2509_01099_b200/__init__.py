"""B200-native ISLBM hot path (arXiv 2509.01099): C-ABI library + thin binding.

`paper_2509_01099_b200.inputs` (synthetic input generators) is importable on its
own; the binding in `paper_2509_01099_b200.islbm` loads the CUDA library and
fails loudly if it has not been built.
"""
__all__ = ["inputs", "islbm"]
