"""B200-native MDWF hot path: Python binding of libmdwf.so (hand-written CUDA for sm_100a).

Build with `python -m paper_1810_01609_b200.build`; the C ABI is include/mdwf.h.
"""
from .binding import (mdwf_selftest_host, Context, Field, MdwfError, SolveResult, lib, LIB_PATH, EXPORTS, OK, NOT_CONVERGED, BREAKDOWN,
                      OP_HOP, OP_M4PRE, OP_M5, OP_M5INV, OP_DHAT_ASYM, OP_DHAT_SYM, OP_NORMAL_ASYM, OP_NORMAL_SYM,
                      OP_FULL)

__all__ = ["mdwf_selftest_host", "Context", "Field", "MdwfError", "SolveResult", "lib", "LIB_PATH", "EXPORTS", "OK", "NOT_CONVERGED",
           "BREAKDOWN", "OP_HOP", "OP_M4PRE", "OP_M5", "OP_M5INV", "OP_DHAT_ASYM", "OP_DHAT_SYM", "OP_NORMAL_ASYM",
           "OP_NORMAL_SYM", "OP_FULL"]
