"""B200-native adjoint particle-mesh hot path (arxiv 2211.09815): C-ABI CUDA library + thin binding.

Importing the package does not load the CUDA library; `paper_2211_09815_b200.binding` does,
and fails loudly if it is missing.  There is no CPU fallback.
"""
