"""Pins P3 (closed-form energies), P4 (dE by brute force), P13 (energy from pair counts)."""
import numpy as np
import pytest

import oracle
from smcx_inputs import make_epi
from pygeom import PyLattice

NOACC = np.zeros(2, np.uint32)


def _mk(lat, dims, n_sp, n_shells, epi, seed=3, init=True):
    return oracle.Oracle(lat, dims, n_sp, n_shells, epi, 1, NOACC, seed, init=init)


@pytest.mark.parametrize("lat,n_shells,Z", [(0, 2, (8, 6)), (1, 3, (12, 6, 24)), (0, 4, (8, 6, 12, 24))])
def test_p3_single_species_closed_form(lat, n_shells, Z):
    epi = make_epi(n_shells, 3, 300, 11)
    o = _mk(lat, (4, 6, 4), 3, n_shells, epi, init=False)
    for p in range(3):
        o.set_species(np.full(o.n_sites, p, np.uint8))
        expect = sum(o.n_sites * Z[s] // 2 * int(epi[s, p, p]) for s in range(n_shells))
        assert o.energy() == expect


def test_p3_b2_closed_form():
    """A on the corner sublattice, B on the body sublattice, BCC with 2 shells:
    H = 4N V1(A,B) + (3N/2) (V2(A,A) + V2(B,B))."""
    epi = make_epi(2, 4, 300, 12)
    o = _mk(0, (4, 4, 6), 4, 2, epi, init=False)
    N = o.n_sites
    for A, B in ((0, 1), (2, 3), (3, 1)):
        s = np.empty(N, np.uint8)
        s[0::2] = A
        s[1::2] = B
        o.set_species(s)
        assert o.energy() == 4 * N * int(epi[0, A, B]) + (3 * N // 2) * int(epi[1, A, A] + epi[1, B, B])


def test_p3_fcc_l12_closed_form():
    """L1_2 (A on basis site 0, B on the three face sites), FCC first shell only: every A has 12 B
    neighbours; every B has 4 A and 8 B neighbours.  Bonds: AB = 12 N/4 = 3N, BB = (3N/4)*8/2 = 3N."""
    epi = make_epi(1, 2, 400, 13)
    o = _mk(1, (4, 4, 4), 2, 1, epi, init=False)
    N = o.n_sites
    s = np.ones(N, np.uint8)
    s[0::4] = 0
    o.set_species(s)
    assert o.energy() == 3 * N * int(epi[0, 0, 1]) + 3 * N * int(epi[0, 1, 1])


def test_p3_random_state_mean_energy():
    """Random equiatomic state: H within 6 sigma of sum_s (Z_s N/2) sum_ab P(a,b) V_s(a,b), with
    P(a,b) the exact without-replacement pair probability."""
    epi = make_epi(2, 4, 300, 14)
    o = _mk(0, (16, 16, 16), 4, 2, epi, seed=77)
    N = o.n_sites
    n = np.bincount(o.species(), minlength=4).astype(float)
    Z = (8, 6)
    mean = 0.0
    var = 0.0
    for s in range(2):
        P = np.outer(n, n) / (N * (N - 1.0))
        P[np.diag_indices(4)] = n * (n - 1.0) / (N * (N - 1.0))
        m1 = (P * epi[s]).sum()
        m2 = (P * epi[s].astype(float) ** 2).sum()
        nb = Z[s] * N / 2.0
        mean += nb * m1
        var += nb * (m2 - m1 * m1) * 4.0   # bonds sharing a site are correlated: generous factor
    assert abs(o.energy() - mean) < 6.0 * np.sqrt(var)


@pytest.mark.parametrize("lat,dims,n_sp,n_shells", [(0, (4, 4, 4), 4, 2), (1, (4, 4, 4), 5, 3),
                                                      (0, (2, 2, 2), 2, 2), (0, (4, 4, 4), 3, 4)])
def test_p4_delta_e_equals_full_recompute(lat, dims, n_sp, n_shells):
    """dE(i, dir) == H(sigma') - H(sigma) with H recomputed by the independent numpy geometry,
    for every site and every direction; and undoing the swap gives -dE."""
    epi = make_epi(n_shells, n_sp, 400, 21)
    o = _mk(lat, dims, n_sp, n_shells, epi, seed=5)
    pl = PyLattice(lat, dims, n_shells)
    sigma = o.species()
    H0 = pl.energy(sigma, epi)
    assert o.energy() == H0
    Z0 = pl.nbr[0].shape[1]
    checked = 0
    for i in range(pl.n_sites):
        for d in range(Z0):
            j = int(pl.nbr[0][i, d])
            s2 = sigma.copy()
            s2[i], s2[j] = sigma[j], sigma[i]
            dE = o.delta_e(i, d)
            assert dE == pl.energy(s2, epi) - H0
            if sigma[i] != sigma[j]:
                o.set_species(s2)
                assert o.delta_e(i, d) == -dE
                o.set_species(sigma)
                checked += 1
    assert checked > pl.n_sites


def test_p13_energy_from_pair_counts():
    for lat, n_sp, n_shells, dims in ((0, 4, 2, (8, 8, 8)), (1, 5, 3, (4, 4, 8))):
        epi = make_epi(n_shells, n_sp, 400, 31)
        o = _mk(lat, dims, n_sp, n_shells, epi, seed=9)
        counts = o.pair_counts()
        twice = int((epi.astype(np.int64) * counts).sum())
        assert twice % 2 == 0 and twice // 2 == o.energy()
        pl = PyLattice(lat, dims, n_shells)
        assert (counts == pl.pair_counts(o.species(), n_sp)).all()
