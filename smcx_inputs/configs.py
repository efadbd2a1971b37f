"""The five BASELINE.json workloads as concrete, seeded, synthetic inputs.

The paper's own workloads are FCC Fe29Co29Ni28Al7Ti7 at 1e6, 1.07e9 and 1.6e10 sites
(PAPER.md:141, 163-173); its fitted interactions are not printed, so these configurations
reproduce the shapes and sizes with seeded interactions.
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import numpy as np

from .tables import make_epi, make_accept_table, anneal_kT_units

BCC = 0
FCC = 1


@dataclass(frozen=True)
class Config:
    name: str
    lattice: int            # 0 = BCC, 1 = FCC
    dims: tuple             # conventional cells (Lx, Ly, Lz)
    n_species: int
    n_shells: int
    amplitude: int          # EPI drawn uniform in [-A, A] (0.1 meV)
    link_cell: int          # w
    kT_units: int           # 0.1 meV; for the anneal this is the starting value
    n_sweeps: int
    seed: int
    anneal: bool = False
    sro_every: int = 0

    @property
    def basis(self) -> int:
        return 2 if self.lattice == BCC else 4

    @property
    def n_sites(self) -> int:
        return self.dims[0] * self.dims[1] * self.dims[2] * self.basis

    def epi(self) -> np.ndarray:
        return make_epi(self.n_shells, self.n_species, self.amplitude, self.seed)

    def kT_at(self, t: int) -> int:
        return anneal_kT_units(t, self.n_sweeps) if self.anneal else self.kT_units

    def accept_table(self, t: int = 0) -> np.ndarray:
        return make_accept_table(self.kT_at(t))


CONFIGS = {
    1: Config("bcc16_4sp", BCC, (16, 16, 16), 4, 2, 300, 4, 860, 100, 1001),
    2: Config("bcc64_4sp_anneal", BCC, (64, 64, 64), 4, 2, 300, 4, 1720, 2000, 1002,
              anneal=True, sro_every=100),
    3: Config("fcc128_5sp", FCC, (128, 128, 128), 5, 3, 400, 4, 690, 1000, 1003),
    4: Config("bcc800_4sp", BCC, (800, 800, 800), 4, 2, 300, 4, 600, 10000, 1004,
              sro_every=1000),
    5: Config("bcc2000_4sp", BCC, (2000, 2000, 2000), 4, 2, 300, 4, 600, 100, 1005),
}


def get_config(k: int) -> Config:
    return CONFIGS[k]


def scaled_config(k: int, dims, n_sweeps=None) -> Config:
    """Config k with a different lattice size (same species, EPI seed, kT, w)."""
    c = CONFIGS[k]
    return replace(c, name=f"{c.name}@{dims[0]}x{dims[1]}x{dims[2]}", dims=tuple(dims),
                   n_sweeps=c.n_sweeps if n_sweeps is None else n_sweeps)
