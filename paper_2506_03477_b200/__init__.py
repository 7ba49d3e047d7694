"""B200-native chi0(q, i*omega) build for QSGW (arxiv 2506.03477): thin Python binding over the
C-ABI library libqsgw.so (hand-written CUDA for sm_100a).  Argument marshalling only."""
from .binding import (PREC_FP64, PREC_MIXED, Chi0Context, QsgwError, chi0_run_host, lib,
                      library_path, version)

__all__ = ["PREC_FP64", "PREC_MIXED", "Chi0Context", "QsgwError", "chi0_run_host", "lib",
           "library_path", "version"]
