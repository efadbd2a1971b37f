"""The seeded input generators (smcx_inputs): ranges, symmetry, table properties (pin P8)."""
import math
import os

import numpy as np

from smcx_inputs import (CONFIGS, accept_table_len, anneal_kT_units, make_accept_table, make_epi,
                         philox4x32_10)

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _kat():
    rows = []
    for line in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        v = [int(t, 16) for t in line.split()]
        rows.append((v[0:4], v[4:6], tuple(v[6:10])))
    return rows


def test_inputs_philox_known_answers():
    for ctr, key, out in _kat():
        assert philox4x32_10(ctr, key) == out


def test_epi_symmetric_in_range_and_seeded():
    for k, cfg in CONFIGS.items():
        v = cfg.epi()
        assert v.dtype == np.int32 and v.shape == (cfg.n_shells, cfg.n_species, cfg.n_species)
        assert (v == v.transpose(0, 2, 1)).all()
        assert v.min() >= -cfg.amplitude and v.max() <= cfg.amplitude
        assert (v != make_epi(cfg.n_shells, cfg.n_species, cfg.amplitude, cfg.seed + 1)).any()
        assert (v == make_epi(cfg.n_shells, cfg.n_species, cfg.amplitude, cfg.seed)).all()


def test_accept_table_shape_and_monotone():
    for kT in (430, 600, 690, 860, 1720):
        t = make_accept_table(kT)
        assert t.dtype == np.uint32 and t.size == accept_table_len(kT)
        assert t[0] == 0xFFFFFFFF and t[-1] == 0
        assert (np.diff(t.astype(np.int64)) <= 0).all()
        # truncation never changes a decision: everything past the table would be 0 too
        assert math.exp(-t.size / kT) * 2.0 ** 32 < 1.0
        # Eq. 3: T[d]/2^32 = exp(-d/kT) to within one unit of 2^-32
        d = np.arange(1, t.size)
        assert np.abs(t[1:] / 2.0 ** 32 - np.exp(-d / kT)).max() < 2.0 ** -31


def test_accept_probability_matches_boltzmann_factor():
    """Empirical rate of u < T[d] over Philox draws is exp(-d/kT) within binomial error."""
    kT = 600
    t = make_accept_table(kT)
    n = 20000
    u = np.array([philox4x32_10((i, 7, 0, 99), (5, 6))[1] for i in range(n)], dtype=np.uint64)
    for d in (1, 150, 600, 1800):
        p = math.exp(-d / kT)
        rate = float((u < int(t[d])).mean())
        assert abs(rate - p) < 5.0 * math.sqrt(p * (1 - p) / n) + 1e-9


def test_anneal_schedule_endpoints():
    assert anneal_kT_units(0) == 1720 and anneal_kT_units(1999) == 430
    ks = [anneal_kT_units(t) for t in range(2000)]
    assert all(a >= b for a, b in zip(ks, ks[1:]))
