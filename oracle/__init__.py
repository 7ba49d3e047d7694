"""ORACLE package — test infrastructure only (see chi0_oracle.py header)."""
from .chi0_oracle import (chi0_accumulate_ref, chi0_entries_ref, chi0_ref, chi0_ref_naive,
                          chi0_sketch_ref, hermitian_finalize_ref, pair_weights, zmel_ref)

from .wc_oracle import dielectric_ref, rotate_to_coulomb_basis_ref, wc_ref
from .realaxis_oracle import hilbert_imag_ref, hilbert_matrix_imag, hilbert_matrix_real, hilbert_real_ref, imchi_accumulate_ref, imchi_naive, imchi_ref
from .eigen_oracle import coulomb_eigenbasis_ref, coulomb_from_eigenbasis_ref
from .ipw_oracle import ipw_product_tensor, zmel_ipw_naive, zmel_ipw_ref
from .sigc_oracle import imag_axis_weights, sigc_imag_naive, sigc_imag_ref, sigc_zw_ref

__all__ = ["coulomb_eigenbasis_ref", "coulomb_from_eigenbasis_ref", "ipw_product_tensor", "zmel_ipw_naive", "zmel_ipw_ref", "hilbert_matrix_real", "hilbert_real_ref", "hilbert_imag_ref", "hilbert_matrix_imag", "imchi_accumulate_ref", "imchi_naive", "imchi_ref", "imag_axis_weights", "sigc_imag_naive", "sigc_imag_ref", "sigc_zw_ref", "dielectric_ref", "rotate_to_coulomb_basis_ref", "wc_ref", "chi0_accumulate_ref", "chi0_entries_ref", "chi0_ref", "chi0_ref_naive",
           "chi0_sketch_ref", "hermitian_finalize_ref", "pair_weights", "zmel_ref"]
