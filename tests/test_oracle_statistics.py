"""Pins P9 (exact Boltzmann stationarity), P10 (LC schedule samples the same ensemble),
P11 (BCC Ising antiferromagnet special case), P12 (Warren-Cowley values and identities)."""
import itertools
import math

import numpy as np

import oracle
from smcx_inputs import make_accept_table, make_epi, scaled_config
from pygeom import PyLattice


def _exact_energy_distribution(pl, epi, kT):
    """All C(16,8) two-species states of the 16-site BCC 2x2x2 cell: P(E) ~ g(E) exp(-E/kT)."""
    weights = {}
    for occ in itertools.combinations(range(16), 8):
        s = np.ones(16, dtype=np.int64)
        s[list(occ)] = 0
        E = pl.energy(s, epi)
        weights[E] = weights.get(E, 0) + 1
    Emin = min(weights)
    Z = sum(g * math.exp(-(E - Emin) / kT) for E, g in weights.items())
    return {E: g * math.exp(-(E - Emin) / kT) / Z for E, g in weights.items()}, weights


def _sample_energy_histogram(o, n_sweeps, burn=2000):
    o.sweep_sequential(burn)
    o.sweep_sequential(n_sweeps)
    tr = o.energy_trace(burn, n_sweeps)
    vals, cnt = np.unique(tr, return_counts=True)
    return dict(zip(vals.tolist(), (cnt / n_sweeps).tolist())), tr


def _check_hist(hist, exact, n, tau=6.0):
    assert set(hist) <= set(exact)
    for E, p in exact.items():
        got = hist.get(E, 0.0)
        assert abs(got - p) < 5.0 * math.sqrt(p * (1 - p) * tau / n) + 2.0 / n, (E, got, p)


def test_p9_nn_only_closed_form_degeneracies():
    """NN only on BCC 2x2x2: with m = number of A on the corner sublattice, g(m) = C(8,m)^2 and
    E(m) = (V_AA+V_BB) m(8-m) + V_AB (m^2 + (8-m)^2)."""
    epi = make_epi(1, 2, 300, 7)
    pl = PyLattice(0, (2, 2, 2), 1)
    _, g = _exact_energy_distribution(pl, epi, 100.0)
    vaa, vbb, vab = int(epi[0, 0, 0]), int(epi[0, 1, 1]), int(epi[0, 0, 1])
    expect = {}
    for m in range(9):
        E = (vaa + vbb) * m * (8 - m) + vab * (m * m + (8 - m) ** 2)
        expect[E] = expect.get(E, 0) + math.comb(8, m) ** 2
    assert g == expect


def test_p9_boltzmann_histogram_nn_only():
    kT = 150
    epi = make_epi(1, 2, 300, 7)
    pl = PyLattice(0, (2, 2, 2), 1)
    exact, _ = _exact_energy_distribution(pl, epi, kT)
    o = oracle.Oracle(0, (2, 2, 2), 2, 1, epi, 1, make_accept_table(kT), 2024)
    n = 150000
    hist, tr = _sample_energy_histogram(o, n)
    _check_hist(hist, exact, n)
    mean = sum(E * p for E, p in exact.items())
    var = sum((E - mean) ** 2 * p for E, p in exact.items())
    assert abs(tr.mean() - mean) < 5.0 * math.sqrt(var * 6.0 / n)


def test_p9_boltzmann_histogram_two_shells():
    """Second shell included: every 2NN bond appears twice on the 2x2x2 cell (48 bonds, 24
    distinct), which the multiset-of-offsets rule of S0 must reproduce."""
    kT = 200
    epi = make_epi(2, 2, 300, 8)
    pl = PyLattice(0, (2, 2, 2), 2)
    assert pl.half[1].sum() * 16 == 48
    exact, _ = _exact_energy_distribution(pl, epi, kT)
    o = oracle.Oracle(0, (2, 2, 2), 2, 2, epi, 1, make_accept_table(kT), 2025)
    n = 150000
    hist, _ = _sample_energy_histogram(o, n)
    _check_hist(hist, exact, n)


def test_p10_link_cell_schedule_samples_the_same_ensemble():
    """<E> and <alpha_1^{01}> from LC sweeps and from sequential sweeps on BCC 16^3 agree within 5 sigma
    (block-averaged errors)."""
    cfg = scaled_config(1, (16, 16, 16))
    burn, n, nblk = 60, 240, 8

    def run(lc, seed):
        o = oracle.Oracle.from_config(cfg, seed=seed)
        E, A = [], []
        for t in range(burn + n):
            o.sweep(1) if lc else o.sweep_sequential(1)
            if t >= burn:
                E.append(o.running_energy())
                if t % 10 == 0:
                    A.append(o.sro()[0][0, 0, 1])
        E = np.array(E, dtype=float).reshape(nblk, -1).mean(axis=1)
        return E.mean(), E.std(ddof=1) / math.sqrt(nblk), float(np.mean(A)), float(np.std(A, ddof=1) / math.sqrt(len(A)))

    e1, s1, a1, sa1 = run(True, 11)
    e2, s2, a2, sa2 = run(False, 12)
    assert abs(e1 - e2) < 5.0 * math.hypot(s1, s2)
    assert abs(a1 - a2) < 5.0 * math.hypot(sa1, sa2) + 1e-3


def test_p11_bcc_ising_antiferromagnet_orders_below_and_disorders_above_tc():
    """2 species, NN only, V_AA = V_BB = +J', V_AB = -J': the BCC Ising antiferromagnet with
    conserved magnetisation, kT_c ~ 6.354 J'.  Long-range order parameter from a B2 start."""
    J = 100
    epi = np.array([[[J, -J], [-J, J]]], dtype=np.int32)
    dims = (16, 16, 16)
    N = 16 ** 3 * 2
    b2 = np.zeros(N, np.uint8)
    b2[1::2] = 1

    def lro(kT):
        o = oracle.Oracle(0, dims, 2, 1, epi, 4, make_accept_table(kT), 5)
        o.set_species(b2)
        o.sweep(150)
        s = o.species()
        return abs(float((s[0::2] == 0).mean()) - float((s[1::2] == 0).mean()))

    assert lro(int(0.6 * 6.354 * J)) > 0.8
    assert lro(int(1.6 * 6.354 * J)) < 0.15


def test_p12_b2_sro_exact_values():
    """B2: alpha_1^{AB} = -1, alpha_1^{AA} = +1, alpha_2^{AA} = -1, alpha_2^{AB} = +1 (Eq. 8)."""
    epi = np.zeros((2, 2, 2), np.int32)
    o = oracle.Oracle(0, (4, 4, 4), 2, 2, epi, 1, np.zeros(2, np.uint32), 0, init=False)
    s = np.zeros(o.n_sites, np.uint8)
    s[1::2] = 1
    o.set_species(s)
    alpha, counts = o.sro()
    assert np.allclose(alpha[0], [[1, -1], [-1, 1]], atol=1e-15)
    assert np.allclose(alpha[1], [[-1, 1], [1, -1]], atol=1e-15)
    assert counts[0, 0, 1] == o.n_sites // 2 * 8 and counts[0, 0, 0] == 0


def test_p12_sro_identities_and_random_limit():
    """sum_p c_p alpha_s^{p p'} = 0 for every p', s; alpha symmetric; small for a random
    solid solution ("at high temperature the alloy remains nearly random")."""
    cfg = scaled_config(3, (8, 8, 8))
    o = oracle.Oracle.from_config(cfg)
    alpha, counts = o.sro()
    n = np.bincount(o.species(), minlength=5).astype(float)
    c = n / n.sum()
    Z = (12, 6, 24)
    for s in range(3):
        assert np.allclose(alpha[s], alpha[s].T, atol=1e-12)
        assert np.allclose((c[None, :] * alpha[s]).sum(axis=1), 0.0, atol=1e-12)
        assert counts[s].sum() == cfg.n_sites * Z[s]
        assert np.abs(alpha[s]).max() < 6.0 / math.sqrt(cfg.n_sites * Z[s] * 0.2 * 0.2)
    # definition, retyped: alpha = 1 - N_s(p',p) N / (Z_s n_p' n_p)
    ref = 1.0 - counts[1] * n.sum() / (Z[1] * np.outer(n, n))
    assert np.allclose(alpha[1], ref, rtol=0, atol=1e-12)
    # very high temperature keeps it random
    o.set_temperature(make_accept_table(200000))
    o.sweep(5)
    hot = o.sro()[0]
    for s in range(3):
        assert np.abs(hot[s]).max() < 6.0 / math.sqrt(cfg.n_sites * Z[s] * 0.2 * 0.2)


def test_p12_sro_nan_for_absent_species():
    epi = np.zeros((1, 3, 3), np.int32)
    o = oracle.Oracle(0, (2, 2, 2), 3, 1, epi, 1, np.zeros(2, np.uint32), 0, init=False)
    s = np.zeros(16, np.uint8)
    s[::2] = 1
    o.set_species(s)
    alpha, _ = o.sro()
    assert np.isnan(alpha[0, 2, :]).all() and np.isnan(alpha[0, :, 2]).all()
    assert np.isfinite(alpha[0, :2, :2]).all()
