"""B200-native chi0(q, i*omega) build for QSGW (arxiv 2506.03477): thin Python binding over the
C-ABI library libqsgw.so (hand-written CUDA for sm_100a).  Argument marshalling only."""
from .binding import (PEAK_FP64_MMA, PEAK_TF32_MMA, probe_peak, PREC_FP64, PREC_MIXED, PREC_MIXED_TF32X1, PREC_MIXED_TF32X3, PEAK_F16_MMA, STAGE_CHI0, STAGE_FINALIZE, STAGE_WEIGHTS, STAGE_ZMEL, Chi0Context, QsgwError, chi0_run_host, wc_from_chi0, chi0_to_coulomb_basis, lib,
                      library_path, version)

__all__ = ["PEAK_FP64_MMA", "PEAK_TF32_MMA", "probe_peak", "PREC_FP64", "PREC_MIXED", "PREC_MIXED_TF32X1", "PREC_MIXED_TF32X3", "PEAK_F16_MMA", "STAGE_ZMEL", "STAGE_WEIGHTS", "STAGE_CHI0", "STAGE_FINALIZE", "Chi0Context", "QsgwError", "chi0_run_host", "wc_from_chi0", "chi0_to_coulomb_basis", "lib",
           "library_path", "version"]
