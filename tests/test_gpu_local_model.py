"""The nonlinear local-energy model (reading S12) on the GPU against the oracle
(pytest -m gpu): species after every sweep, energy trace, statistics and H of the model, bit for bit."""
import numpy as np
import pytest

import oracle
import paper_2509_20949_b200 as smcx
from smcx_inputs import composition_counts, make_accept_table, make_epi, make_local_weights

pytestmark = pytest.mark.gpu


def _pair(lattice, dims, n_sp, n_sh, seed, kT, amp1=200, amp2=25):
    w1, w2 = make_local_weights(n_sh, n_sp, amp1, amp2, seed)
    table = make_accept_table(kT)
    g = smcx.Lattice(lattice, dims, n_sp, n_sh, w1, table, seed, link_cell=4, kT_units=kT, local_quad=w2)
    o = oracle.Oracle(lattice, dims, n_sp, n_sh, w1, 4, table, seed)
    o.set_local_model(w2)
    return g, o


@pytest.mark.parametrize("lattice,dims,n_sp,n_sh,kT", [
    (smcx.BCC, (16, 16, 16), 4, 2, 900),
    (smcx.BCC, (24, 16, 32), 2, 1, 500),       # one shell, two species, a ragged grid of cells
    (smcx.FCC, (16, 16, 16), 5, 3, 2500),      # the paper's lattice type: 42 neighbours, 86 affected sites per trial
    (smcx.FCC, (16, 24, 16), 8, 2, 1500),      # most species the packed counters take
    (smcx.BCC, (16, 16, 16), 6, 2, 900),       # most species of the 5-bit count fields (32-bit count word)
    (smcx.FCC, (16, 16, 16), 7, 1, 1200),      # one more: 8-bit fields again
])
def test_local_model_against_the_oracle(lattice, dims, n_sp, n_sh, kT):
    g, o = _pair(lattice, dims, n_sp, n_sh, seed=41, kT=kT)
    assert g.kernel == smcx.KERNEL_LOCAL_WARP and g.storage == smcx.STORAGE_U8
    assert (g.species() == o.species()).all()
    assert g.energy() == o.energy() == g.running_energy()
    for _ in range(3):
        g.sweep(1)
        o.sweep(1)
        assert (g.species() == o.species()).all()
    g.sweep(3)                                   # graph replay
    o.sweep(3)
    assert (g.species() == o.species()).all()
    assert (g.energy_trace() == o.energy_trace()).all()
    assert g.stats() == o.stats() and g.stats()[2] > 0
    assert g.energy() == o.energy() == g.running_energy() == o.running_energy()
    ga, gc = g.sro()
    oa, oc = o.sro()
    assert (gc == oc).all() and np.allclose(ga, oa, rtol=1e-9, atol=1e-9, equal_nan=True)
    g.close()


def test_linear_symmetric_local_model_walks_the_epi_trajectory():
    """W2 = 0, W1 = V symmetric, threshold table of 2 kT: the local-model kernel must reproduce the trajectory of the
    pairwise kernels (energies doubled) -- two structurally different CUDA paths and the oracle agree."""
    dims, n_sp, n_sh, seed, kT = (16, 16, 16), 4, 2, 21, 600
    V = make_epi(n_sh, n_sp, 300, seed)
    epi = smcx.Lattice(smcx.BCC, dims, n_sp, n_sh, V, make_accept_table(kT), seed, link_cell=4, kT_units=kT)
    loc = smcx.Lattice(smcx.BCC, dims, n_sp, n_sh, V, make_accept_table(2 * kT), seed, link_cell=4, kT_units=2 * kT,
                       local_quad=np.zeros((n_sh, n_sp, n_sp, n_sp), dtype=np.int32))
    o = oracle.Oracle(smcx.BCC, dims, n_sp, n_sh, V, 4, make_accept_table(kT), seed)
    assert loc.energy() == 2 * epi.energy()
    epi.sweep(6)
    loc.sweep(6)
    o.sweep(6)
    assert (loc.species() == epi.species()).all() and (loc.species() == o.species()).all()
    assert (loc.energy_trace() == 2 * epi.energy_trace()).all()
    assert loc.stats() == epi.stats()
    epi.close()
    loc.close()


def test_local_model_on_the_papers_composition_with_cooling():
    g, o = _pair(smcx.FCC, (16, 16, 16), 5, 3, seed=5, kT=3000)
    counts = composition_counts(o.n_sites, (29, 29, 28, 7, 7))
    g.init_composition(counts)
    o.init_composition(counts)
    assert g.energy() == o.energy()
    for kT in (3000, 2000, 1200):
        table = make_accept_table(kT)
        g.set_temperature(kT, table)
        o.set_temperature(table)
        g.sweep(2)
        o.sweep(2)
        assert (g.species() == o.species()).all()
    assert (g.energy_trace() == o.energy_trace()).all() and g.energy() == o.energy() == g.running_energy()
    g.close()
