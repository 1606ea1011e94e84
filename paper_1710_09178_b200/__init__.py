"""B200-native staggered Dslash / M^dag M / multishift CG (arXiv:1710.09178 hot path).

The product is the C-ABI library `libqcd_b200.so` (include/qcd.h, csrc/*.cu);
this package is its thin ctypes binding: argument marshalling only.  There is no
CPU fallback: importing works anywhere, but every call needs the built library
and an sm_100 device, and fails loudly otherwise.
"""
from .binding import (QCD_EVEN, QCD_ODD, QCD_OPT_PDL, QCD_OPT_CG_GRAPH, QCD_OPT_CG_BATCH, QCD_OPT_LINK_ROWS, QCD_OPT_TGROUP, QCD_OPT_L2_PERSIST_MB, QCD_OPT_Y_ONLY, QCD_OPT_DSLASH_KERNEL, QCD_OPT_DSLASH_PERSIST, QCD_OPT_MIXED, QCD_OPT_MIXED_SWITCH_EXP, QCD_OPT_OPERATOR_LINKS32, QCD_OPT_SWEEP_ALTERNATE, QCD_OPT_CG_DEFER, QCD_OPT_SWEEP_KEEP_MB, QCD_OPT_CG_FUSE, QcdError, Context, library_path, load_library,  # noqa: F401
                      exported_symbols, inv_sqrt_coeffs, pow_coeffs)

__all__ = ["QCD_EVEN", "QCD_ODD", "QCD_OPT_PDL", "QCD_OPT_CG_GRAPH", "QCD_OPT_CG_BATCH", "QCD_OPT_LINK_ROWS", "QCD_OPT_TGROUP", "QCD_OPT_L2_PERSIST_MB", "QCD_OPT_Y_ONLY", "QCD_OPT_DSLASH_KERNEL", "QCD_OPT_DSLASH_PERSIST", "QCD_OPT_MIXED", "QCD_OPT_MIXED_SWITCH_EXP", "QCD_OPT_OPERATOR_LINKS32", "QCD_OPT_SWEEP_ALTERNATE", "QCD_OPT_CG_DEFER", "QCD_OPT_SWEEP_KEEP_MB", "QCD_OPT_CG_FUSE", "QcdError", "Context", "library_path", "load_library",
           "exported_symbols", "inv_sqrt_coeffs", "pow_coeffs"]
