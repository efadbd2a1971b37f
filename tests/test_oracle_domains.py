"""Pins of the oracle's decomposed sweep (reading S11; lattice parallelism with ghost layers).

What fixes the result: every draw of a trial depends on the global cell id, slot, sweep and colour only (S4) and
the cells of a colour commute (pin P7), so a lattice cut into slabs that exchange their boundary layers must
reproduce the undivided sweep bit for bit.  The undivided sweep is pinned by P4-P10; here the slab protocol is
pinned against it, together with the negative controls that show the pins can fail.
"""
import numpy as np
import pytest

import oracle
from smcx_inputs import make_accept_table, make_epi


def _lattice(lattice, dims, n_species, n_shells, seed, kT=700, amp=300):
    epi = make_epi(n_shells, n_species, amp, seed)
    return oracle.Oracle(lattice, dims, n_species, n_shells, epi, 4, make_accept_table(kT), seed)


CASES = [
    # lattice, dims, species, shells, slabs
    (oracle.BCC, (16, 16, 32), 4, 2, 2),
    (oracle.BCC, (16, 16, 32), 4, 2, 4),
    (oracle.BCC, (8, 16, 40), 3, 2, 3),      # 5 row pairs over 3 slabs: 2 + 2 + 1
    (oracle.FCC, (8, 8, 16), 5, 3, 2),       # two rows per slab, the thinnest a slab can be
    (oracle.FCC, (8, 8, 32), 5, 3, 4),
]


@pytest.mark.parametrize("lattice,dims,n_species,n_shells,n_slabs", CASES)
def test_s11_slabs_reproduce_the_undivided_sweep(lattice, dims, n_species, n_shells, n_slabs):
    whole = _lattice(lattice, dims, n_species, n_shells, seed=77)
    cut = _lattice(lattice, dims, n_species, n_shells, seed=77)
    n = 7                                      # several origins, so the windows move both ways
    shifts = {whole.shift(t)[2] for t in range(n)}
    assert len(shifts) >= 3
    whole.sweep(n)
    assert cut.sweep_slabs(n, n_slabs, ghost=2, order_seed=5) == 0          # no read outside a slab's window
    assert (cut.species() == whole.species()).all()
    assert (cut.energy_trace() == whole.energy_trace()).all()
    assert cut.stats() == whole.stats()
    assert cut.energy() == whole.energy() == cut.running_energy()


def test_s11_result_does_not_depend_on_the_order_of_the_slabs_or_on_how_the_run_is_split():
    a = _lattice(oracle.BCC, (16, 16, 32), 4, 2, seed=3)
    b = _lattice(oracle.BCC, (16, 16, 32), 4, 2, seed=3)
    c = _lattice(oracle.BCC, (16, 16, 32), 4, 2, seed=3)
    assert a.sweep_slabs(6, 4, order_seed=1) == 0
    assert b.sweep_slabs(6, 4, order_seed=99) == 0
    assert c.sweep_slabs(2, 4, order_seed=7) == 0 and c.sweep_slabs(4, 2, order_seed=8) == 0   # 4 slabs, then 2
    assert (a.species() == b.species()).all() and (a.species() == c.species()).all()
    assert (a.energy_trace() == b.energy_trace()).all() and (a.energy_trace() == c.energy_trace()).all()


def test_s11_partition_cuts_on_pairs_of_link_cell_rows():
    o = _lattice(oracle.BCC, (8, 8, 40), 2, 1, seed=1)             # 10 rows = 5 pairs
    assert o.slab_partition(1) == [(0, 10)]
    assert o.slab_partition(2) == [(0, 6), (6, 4)]
    assert o.slab_partition(3) == [(0, 4), (4, 4), (8, 2)]
    assert o.slab_partition(5) == [(0, 2), (2, 2), (4, 2), (6, 2), (8, 2)]
    with pytest.raises(ValueError):
        o.slab_partition(6)                                        # fewer than one row pair per slab
    for d in (2, 3, 4, 5):
        rows = o.slab_partition(d)
        assert all(first % 2 == 0 and count % 2 == 0 and count >= 2 for first, count in rows)
        assert rows[0][0] == 0 and sum(c for _, c in rows) == 10
        assert all(rows[k][0] + rows[k][1] == rows[k + 1][0] for k in range(d - 1))


def test_s11_negative_controls_a_thin_ghost_layer_or_a_missing_exchange_is_noticed():
    whole = _lattice(oracle.BCC, (16, 16, 32), 4, 2, seed=12)
    whole.sweep(4)
    # one ghost layer: the LIZ+ of a boundary cell reaches r0 + R = 3 half-units = 2 conventional cells
    thin = _lattice(oracle.BCC, (16, 16, 32), 4, 2, seed=12)
    assert thin.sweep_slabs(4, 2, ghost=1) > 0
    # right ghost width, no messages after the colour passes: stale copies, different trajectory
    mute = _lattice(oracle.BCC, (16, 16, 32), 4, 2, seed=12)
    mute.sweep_slabs(4, 2, ghost=2, exchange=False)
    assert (mute.species() != whole.species()).any()
    # a wider ghost layer than needed changes nothing
    wide = _lattice(oracle.BCC, (16, 16, 32), 4, 2, seed=12)
    assert wide.sweep_slabs(4, 2, ghost=3) == 0
    assert (wide.species() == whole.species()).all()


def test_s11_poison_is_never_read_by_the_undivided_sweep():
    o = _lattice(oracle.FCC, (8, 8, 16), 5, 3, seed=4)
    before = o.species().copy()
    assert before.max() < 5
    o.sweep(2)
    assert np.bincount(o.species(), minlength=5).tolist() == np.bincount(before, minlength=5).tolist()


def test_s11_with_the_local_energy_model_needs_three_ghost_layers():
    """Reading S12 on slabs: a trial of the local model reads neighbours of neighbours (reach r0 + 2R = 5 half-units = 3
    conventional cells), so the window needs H = 3 ghost layers and the pass message carries H + 1 = 4 layers; with those
    the decomposed sweep equals the undivided one, with the pair model's two ghost layers poison is read."""
    from smcx_inputs import make_local_weights

    def lat():
        w1, w2 = make_local_weights(2, 4, 200, 25, 13)
        o = oracle.Oracle(oracle.BCC, (16, 16, 32), 4, 2, w1, 4, make_accept_table(900), 13)
        o.set_local_model(w2)
        return o

    whole, cut, thin = lat(), lat(), lat()
    whole.sweep(5)
    assert cut.sweep_slabs(5, 2, ghost=3, order_seed=3) == 0
    assert (cut.species() == whole.species()).all() and (cut.energy_trace() == whole.energy_trace()).all()
    assert cut.energy() == whole.energy() == cut.running_energy()
    assert thin.sweep_slabs(5, 2, ghost=2) > 0
