"""Seeded synthetic input generators shared by the oracle tests, the GPU tests and bench.py.

This module is *input data only*: it produces the EPI tables V_s(a,b), the integer
acceptance-threshold tables and the five workload configurations of BASELINE.json.
It holds none of the method's arithmetic (no lattice geometry, no energy, no Metropolis
step, no SRO) and imports neither ``oracle`` nor ``paper_2509_20949_b200``.

Recipes:
  * EPI: V_s(a,b)=V_s(b,a) = -A + mulhi32(philox(ctr=(a,b,s,TAG_EPI), key=seed)[0], 2A+1)
    for a <= b, i.e. uniform integers in [-A, A] in 0.1 meV units.  The paper prints no EPI
    values, so these stand in for the fitted Fe29Co29Ni28Al7Ti7 interactions.
  * nonlinear local-energy model (reading S12): make_local_weights, uniform integer weights drawn the same way.
  * threshold table: T[d] = min(floor(exp(-d/kT_units) * 2^32), 2^32-1),
    len = floor(32 ln2 kT_units) + 2 (last entry is exactly 0).  Eq. 3, PAPER.md:60-63,
    in the integer form BASELINE.json's north_star fixes ("a 32-bit Philox draw compared
    with a host-precomputed threshold table indexed by integer dE, passed in as input data").
"""
from .tables import (  # noqa: F401
    TAG_EPI,
    philox4x32_10,
    make_epi,
    make_local_weights,
    make_accept_table,
    accept_table_len,
    anneal_kT_units,
    replica_ladder,
    composition_counts,
    cooling_stages,
)
from .configs import Config, CONFIGS, get_config, scaled_config  # noqa: F401
