"""The five workload configurations of BASELINE.json:configs (shapes only).

Stand-ins shaped like the paper's systems (small semiconductor cells, a magnetic
Heusler-like metal ~ Ni2MnGa with n_spin = 2, a superlattice ~ (InAs)n(GaSb)n with
n_BZ = 16; Table 2).  The paper's real eigenvectors and
product-basis integrals are not available; DESIGN.md states the recipe.
"""
from __future__ import annotations

import dataclasses
from dataclasses import dataclass
from typing import Tuple

BASE_SEED = 250603477


@dataclass(frozen=True)
class WorkloadConfig:
    name: str
    index: int                 # position in BASELINE.json:configs (seed = BASE_SEED + index)
    orb_per_site: Tuple[int, ...]   # b_s
    pb_per_site: Tuple[int, ...]    # m_s
    n_k: int
    n_spin: int
    n_o: int                   # |O|: "occupied side" bands taken from C_k
    n_u: int                   # |U|: "unoccupied side" bands taken from C_{k+q}
    n_freq: int
    kind: str                  # "insulator" | "metal"
    eps_occ: Tuple[float, float] = (0.0, 0.0)     # insulator: U[lo, hi] for O
    eps_unocc: Tuple[float, float] = (0.0, 0.0)   # insulator: U[lo, hi] for U
    eps_all: Tuple[float, float] = (0.0, 0.0)     # metal: U[lo, hi] for all N_b bands
    o_first: int = 0           # metal: rank of the first band in O (sorted energies)
    u_first: int = 0           # metal: rank of the first band in U
    kT: float = 0.0            # metal: Fermi-Dirac temperature (Ha), E_F = 0
    omega_1: float = 0.01      # first non-zero imaginary frequency (Ha)
    omega_max: float = 20.0    # last imaginary frequency (Ha)
    precision: str = "fp64"    # "fp64" | "mixed"
    occ_tol: float = 1e-12

    @property
    def n_sites(self) -> int:
        return len(self.orb_per_site)

    @property
    def n_b(self) -> int:
        return sum(self.orb_per_site)

    @property
    def n_m(self) -> int:
        return sum(self.pb_per_site)

    def stage_a_cmac(self) -> int:
        """Two-step count of stage (a) complex multiply-adds per k."""
        return sum(m * b * self.n_o * (b + self.n_u)
                   for b, m in zip(self.orb_per_site, self.pb_per_site))

    def stage_b_cmac_per_pair(self) -> int:
        """Upper-triangle complex multiply-adds per kept pair, all frequencies."""
        return self.n_freq * self.n_m * (self.n_m + 1) // 2


def _uniform(name, index, s, b, m, **kw):
    return WorkloadConfig(name=name, index=index, orb_per_site=(b,) * s,
                          pb_per_site=(m,) * s, **kw)


CONFIGS = (
    _uniform("cfg0_tiny_insulator", 0, 2, 18, 40, n_k=8, n_spin=1, n_o=8, n_u=28,
             n_freq=8, kind="insulator", eps_occ=(-0.45, 0.0), eps_unocc=(0.02, 1.1)),
    _uniform("cfg1_si_like", 1, 2, 25, 120, n_k=64, n_spin=1, n_o=4, n_u=46,
             n_freq=16, kind="insulator", eps_occ=(-0.45, 0.0), eps_unocc=(0.04, 1.1)),
    _uniform("cfg2_heusler_metal_fp64", 2, 4, 25, 150, n_k=216, n_spin=2, n_o=30, n_u=70,
             n_freq=16, kind="metal", eps_all=(-0.4, 0.8), o_first=8, u_first=28, kT=1e-3),
    _uniform("cfg3_heusler_metal_mixed", 3, 4, 25, 150, n_k=216, n_spin=2, n_o=30, n_u=70,
             n_freq=16, kind="metal", eps_all=(-0.4, 0.8), o_first=8, u_first=28, kT=1e-3,
             precision="mixed"),
    _uniform("cfg4_superlattice", 4, 16, 25, 150, n_k=16, n_spin=1, n_o=64, n_u=336,
             n_freq=16, kind="insulator", eps_occ=(-0.5, 0.0), eps_unocc=(0.01, 1.5)),
)


def get_config(index_or_name) -> WorkloadConfig:
    for c in CONFIGS:
        if c.index == index_or_name or c.name == index_or_name:
            return c
    raise KeyError(index_or_name)


def scaled_config(cfg: WorkloadConfig, **overrides) -> WorkloadConfig:
    """A copy of `cfg` with some extents replaced (reduced-size test cases)."""
    return dataclasses.replace(cfg, **overrides)
