"""ORACLE package — test infrastructure only (see chi0_oracle.py header)."""
from .chi0_oracle import (chi0_accumulate_ref, chi0_entries_ref, chi0_ref, chi0_ref_naive,
                          chi0_sketch_ref, hermitian_finalize_ref, pair_weights, zmel_ref)

from .wc_oracle import dielectric_ref, rotate_to_coulomb_basis_ref, wc_ref

__all__ = ["dielectric_ref", "rotate_to_coulomb_basis_ref", "wc_ref", "chi0_accumulate_ref", "chi0_entries_ref", "chi0_ref", "chi0_ref_naive",
           "chi0_sketch_ref", "hermitian_finalize_ref", "pair_weights", "zmel_ref"]
