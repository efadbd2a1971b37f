"""Pins of the oracle's replica exchange (S9; Eq. 5-7): Delta against exact rational
arithmetic, the acceptance frequency against min(1, exp(Delta)), Boltzmann stationarity of every
temperature slot on the exactly enumerable 16-site lattice, and the 1/sqrt(N) spacing rule."""
import math
from fractions import Fraction

import numpy as np

import oracle
from smcx_inputs import make_accept_table, make_epi, replica_ladder, scaled_config
from pygeom import PyLattice
from test_oracle_statistics import _check_hist, _exact_energy_distribution


def test_delta_matches_rational_arithmetic_and_is_symmetric():
    rng = np.random.default_rng(5)
    for _ in range(200):
        Ei, Ej = (int(v) for v in rng.integers(-10 ** 12, 10 ** 12, 2))
        Ti, Tj = (int(v) for v in rng.integers(50, 5000, 2))
        exact = (Fraction(1, Ti) - Fraction(1, Tj)) * (Ei - Ej)
        got = oracle.exchange_delta(Ei, Ej, Ti, Tj)
        assert abs(got - float(exact)) <= 1e-14 * max(1.0, abs(float(exact)))
        assert got == oracle.exchange_delta(Ej, Ei, Tj, Ti)          # relabelling the pair changes nothing
    # the colder replica holding the higher energy always hands it over
    assert oracle.exchange_delta(-100, -900, 500, 800) > 0
    assert all(oracle.exchange_accept(-100, -900, 500, 800, u) for u in (0, 1, 2 ** 31, 2 ** 32 - 1))
    assert oracle.exchange_accept(7, 7, 500, 800, 2 ** 32 - 1) and oracle.exchange_accept(3, 9, 600, 600, 2 ** 32 - 1)


def test_acceptance_frequency_is_exp_delta():
    for (Ei, Ej, Ti, Tj) in [(-5000, -4000, 600, 700), (-5000, -1000, 600, 650), (-90000, -40000, 430, 440)]:
        delta = (1.0 / Ti - 1.0 / Tj) * (Ei - Ej)
        assert delta < 0
        n = 200_000
        acc = sum(oracle.exchange_accept(Ei, Ej, Ti, Tj, oracle.exchange_draw(99, r, 3)) for r in range(n))
        p = math.exp(delta)
        assert abs(acc / n - p) < 5.0 * math.sqrt(p * (1 - p) / n) + 1e-9, (acc / n, p)
    # threshold edges: u = 0 is accepted whenever exp(Delta) 2^32 >= 1, the largest u never for Delta < 0
    assert oracle.exchange_accept(-5000, -4000, 600, 700, 0)
    assert not oracle.exchange_accept(-5000, -4000, 600, 700, 2 ** 32 - 1)
    assert not oracle.exchange_accept(0, 10 ** 9, 100, 5000, 0)      # exp(Delta) 2^32 < 1: never


def test_every_slot_stays_boltzmann_under_exchange():
    """Three replicas of the 16-site two-species BCC cell, one sequential sweep each, then an
    exchange round (alternating parity): the energy histogram of every temperature slot must be the
    exact Boltzmann one of that slot's temperature.  A wrong sign or a wrong pairing of E and T fails."""
    kTs = [150, 400, 1100]
    epi = make_epi(2, 2, 300, 8)
    pl = PyLattice(0, (2, 2, 2), 2)
    tables = [make_accept_table(k) for k in kTs]
    reps = [oracle.Oracle(0, (2, 2, 2), 2, 2, epi, 1, tables[r], 4000 + r) for r in range(3)]
    burn, n = 2000, 60000
    E = np.zeros((3, n), dtype=np.int64)
    n_acc = np.zeros(2, dtype=np.int64)
    for t in range(burn + n):
        for o in reps:
            o.sweep_sequential(1)
        n_acc += np.array(oracle.replica_exchange(reps, kTs, tables, t & 1, 777, t))
        if t >= burn:
            for r in range(3):
                E[r, t - burn] = reps[r].running_energy()
    for r in range(3):
        assert reps[r].running_energy() == reps[r].energy()
        exact, _ = _exact_energy_distribution(pl, epi, kTs[r])
        vals, cnt = np.unique(E[r], return_counts=True)
        _check_hist(dict(zip(vals.tolist(), (cnt / n).tolist())), exact, n, tau=12.0)
    attempts = (burn + n) / 2
    assert (n_acc > 0.1 * attempts).all() and n_acc.min() < 0.9 * attempts   # both outcomes occur


def _exchange_rate(dims, kT_lo, dkT, sweeps=160, burn=60, seed=50):
    cfg = scaled_config(1, dims)
    kTs = [kT_lo, kT_lo + dkT]
    tables = [make_accept_table(k) for k in kTs]
    reps = [oracle.Oracle.from_config(cfg, seed=seed + r, accept=tables[r]) for r in range(2)]
    acc = 0
    for t in range(burn + sweeps):
        for o in reps:
            o.sweep(1)
        f = oracle.replica_exchange(reps, kTs, tables, 0, 31, t)
        if t >= burn:
            acc += f[0]
    return acc / sweeps


def test_spacing_rule_eq7():
    """Eq. 7: the exchange rate stays about the same when N grows fourfold and the temperature step
    halves, and collapses when the step is kept (Gaussian energy distributions whose width grows as
    sqrt(N) while their distance grows as N dT)."""
    n1, n2 = 8 * 8 * 8 * 2, 16 * 16 * 8 * 2
    step1 = replica_ladder(860, 2, n1, 60.0 * math.sqrt(n1))
    step2 = replica_ladder(860, 2, n2, 60.0 * math.sqrt(n1))
    assert step1[1] - step1[0] == 60 and step2[1] - step2[0] == 30
    r_small = _exchange_rate((8, 8, 8), 860, 60)
    r_big_scaled = _exchange_rate((16, 16, 8), 860, 30)
    r_big_same = _exchange_rate((16, 16, 8), 860, 60)
    assert 0.1 < r_small < 0.95
    assert abs(r_big_scaled - r_small) < 0.2
    assert r_big_same < r_small - 0.1
