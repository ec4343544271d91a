"""B200-native BioEM hot path (arXiv:1609.06634): thin Python binding over the C-ABI library
``libbioem_b200.so`` (hand-written sm_100a CUDA; see include/bioem.h and DESIGN.md).

Argument marshalling only -- every step of the path runs in the CUDA kernels.  There is no CPU fallback:
importing works without a GPU (so the symbol table can be checked), creating a context does not.
"""
from .binding import (BioEM, BioEMError, ctf_from_defocus, lib, library_path, EXPORTED_SYMBOLS, TOPK)

__all__ = ["BioEM", "BioEMError", "ctf_from_defocus", "lib", "library_path", "EXPORTED_SYMBOLS", "TOPK"]
