"""Pins P1 (Philox) and P2 (shells, neighbour map) for the oracle."""
import os

import numpy as np
import pytest

import oracle
from smcx_inputs import philox4x32_10 as py_philox
from pygeom import PyLattice, shells as py_shells

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def test_p1_philox_known_answers():
    n = 0
    for line in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        v = [int(t, 16) for t in line.split()]
        assert oracle.philox4x32_10(v[0:4], v[4:6]) == tuple(v[6:10])
        n += 1
    assert n == 3


def test_p1_philox_agrees_with_second_implementation():
    rng = np.random.default_rng(1)
    for _ in range(200):
        ctr = [int(x) for x in rng.integers(0, 2 ** 32, 4)]
        key = [int(x) for x in rng.integers(0, 2 ** 32, 2)]
        assert oracle.philox4x32_10(ctr, key) == py_philox(ctr, key)


def test_p2_shell_table():
    for line in open(os.path.join(GOLDEN, "shells.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, s, d2, z, reach = line.split()
        lat = oracle.BCC if name == "BCC" else oracle.FCC
        off = oracle.shell(lat, int(s))
        assert len(off) == int(z)
        assert ((off ** 2).sum(axis=1) == int(d2)).all()
        assert np.abs(off).max() == int(reach)
        # closed under inversion, no duplicates
        as_set = {tuple(o) for o in off}
        assert len(as_set) == len(off)
        assert all((-o[0], -o[1], -o[2]) in as_set for o in as_set)


@pytest.mark.parametrize("lat", [oracle.BCC, oracle.FCC])
def test_p2_shell_order_ascending_dz_dy_dx(lat):
    ref, _ = py_shells(lat, 4)
    for s in range(4):
        off = oracle.shell(lat, s)
        assert (off == ref[s]).all()
        keys = [(int(o[2]), int(o[1]), int(o[0])) for o in off]
        assert keys == sorted(keys)


def test_p2_bcc_direction_index_formula():
    off = oracle.shell(oracle.BCC, 0)
    for k, (dx, dy, dz) in enumerate(off):
        assert k == (dx > 0) | ((dy > 0) << 1) | ((dz > 0) << 2)


@pytest.mark.parametrize("lat,dims,n_shells", [(0, (4, 6, 8), 3), (1, (4, 6, 2), 3), (0, (2, 2, 2), 2)])
def test_p2_neighbour_map_against_position_lookup(lat, dims, n_shells):
    """oracle neighbour(i, s, k) equals a dictionary lookup of P(i)+d mod period."""
    n_sp = 2
    epi = np.zeros((n_shells, n_sp, n_sp), dtype=np.int32)
    o = oracle.Oracle(lat, dims, n_sp, n_shells, epi, 1, np.zeros(2, np.uint32), 0, init=False)
    pl = PyLattice(lat, dims, n_shells)
    assert o.n_sites == pl.n_sites
    for s in range(n_shells):
        for i in range(0, pl.n_sites, 3):
            for k in range(pl.nbr[s].shape[1]):
                assert o.neighbour(i, s, k) == pl.nbr[s][i, k]
