"""paper_2103_05034_b200 -- B200-native domain-wall fermion operator hot path (arxiv 2103.05034).

Thin Python binding over the C-ABI CUDA library libdwf.so (include/dwf.h).  Argument marshalling
only: every step of the path runs in the library's kernels.  There is no CPU fallback: importing
this package without the built library raises.
"""
from .dwf import (Dwf, DwfError, DWF_F32, DWF_F64, DWF_DHOP, DWF_DDW, DWF_HDW, DWF_DPV, DWF_SCHUR_EO,
                  DWF_MEE, DWF_MOOINV, DWF_MPVDAG_M, DWF_SCHUR_EO_ALT, DWF_DAGGER, lib_path, exported_symbols)

__all__ = ["Dwf", "DwfError", "DWF_F32", "DWF_F64", "DWF_DHOP", "DWF_DDW", "DWF_HDW", "DWF_DPV",
           "DWF_SCHUR_EO", "DWF_MEE", "DWF_MOOINV", "DWF_MPVDAG_M", "DWF_SCHUR_EO_ALT", "DWF_DAGGER", "lib_path", "exported_symbols"]
