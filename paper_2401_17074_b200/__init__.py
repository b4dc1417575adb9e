"""B200-native fused TSLB sweep (arXiv 2401.17074): C-ABI library libtslb.so + thin Python binding.

Importing the package is cheap and never loads the CUDA library; `paper_2401_17074_b200.binding`
does that on first use and fails loudly if the library is missing (there is no CPU fallback).
"""
__all__ = ["workloads", "binding", "build"]
