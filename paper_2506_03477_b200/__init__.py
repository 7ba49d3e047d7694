"""B200-native chi0(q, i*omega) build for QSGW (arxiv 2506.03477): thin Python binding over the
C-ABI library libqsgw.so (hand-written CUDA for sm_100a).  Argument marshalling only."""
from .binding import (PEAK_F16_MMA, PEAK_FP64_MMA, PEAK_TF32_MMA, PREC_FP64, PREC_MIXED, STAGE_CHI0,
                      STAGE_FINALIZE, STAGE_WEIGHTS, STAGE_ZMEL, Chi0Context, QsgwError,
                      chi0_run_host, chi0_to_coulomb_basis, chi0_to_coulomb_basis_static, hilbert_to_imag_axis, hilbert_to_real_axis, zmel_ipw_build, coulomb_eigenbasis, lib, library_path, probe_peak,
                      set_global_option, version, wc_from_chi0)

__all__ = ["PEAK_FP64_MMA", "PEAK_TF32_MMA", "PEAK_F16_MMA", "probe_peak", "PREC_FP64", "PREC_MIXED",
           "STAGE_ZMEL", "STAGE_WEIGHTS", "STAGE_CHI0", "STAGE_FINALIZE", "Chi0Context", "QsgwError",
           "chi0_run_host", "wc_from_chi0", "hilbert_to_imag_axis", "hilbert_to_real_axis", "zmel_ipw_build", "coulomb_eigenbasis", "chi0_to_coulomb_basis", "chi0_to_coulomb_basis_static", "set_global_option", "lib",
           "library_path", "version"]
