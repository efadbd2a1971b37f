"""Replica ensemble + replica exchange on the GPU against the oracle (pytest -m gpu), through the C ABI:
which replica sits in which temperature slot, the accept flags of every round, the running energies and
the species arrays of every slot must be identical (S9; Eq. 5-6)."""
import numpy as np
import pytest

import oracle
import paper_2509_20949_b200 as smcx
from smcx_inputs import make_accept_table, replica_ladder, scaled_config

pytestmark = pytest.mark.gpu

KERNELS = [smcx.KERNEL_WARP_PER_CELL, smcx.KERNEL_GROUP_PER_CELL, smcx.KERNEL_THREAD_PER_CELL,
           smcx.KERNEL_THREAD_PERSISTENT]
KERNEL_IDS = ["warp", "group", "thread", "persistent"]


def _ensemble(cfg, kTs, seeds, xseed, kernel):
    tables = [make_accept_table(k) for k in kTs]
    g = smcx.Ensemble(cfg.lattice, cfg.dims, cfg.n_species, cfg.n_shells, cfg.epi(), kTs, tables, seeds, xseed,
                      link_cell=cfg.link_cell, kernel=kernel)
    reps = [oracle.Oracle.from_config(cfg, seed=seeds[r], accept=tables[r]) for r in range(len(kTs))]
    return g, reps, tables


def _assert_slots_equal(g, o_at_slot, o_ids):
    st = g.state()
    assert st["replica_at_slot"].tolist() == o_ids
    assert st["energy_at_slot"].tolist() == [o.running_energy() for o in o_at_slot]
    for p, o in enumerate(o_at_slot):
        r = int(st["replica_at_slot"][p])
        assert (g.replicas[r].species() == o.species()).all(), f"slot {p}"
        assert g.replicas[r].energy() == o.energy()
        assert g.replicas[r].stats() == o.stats()
    return st


@pytest.mark.parametrize("kernel", KERNELS, ids=KERNEL_IDS)
def test_exchange_rounds_match_the_oracle(kernel):
    """Five replicas of the 16^3 BCC config on a ladder with a mixed accept/reject history: step by
    step (sweeps, then one exchange round of alternating parity) against the oracle."""
    cfg = scaled_config(1, (16, 16, 16))
    kTs = replica_ladder(700, 5, cfg.n_sites, 30.0 * np.sqrt(cfg.n_sites))
    assert kTs == [700, 730, 760, 790, 820]
    seeds = [9100 + 17 * r for r in range(5)]
    g, reps, tables = _ensemble(cfg, kTs, seeds, 4242, kernel)
    for o in reps:
        o.tag = reps.index(o)
    n_acc = np.zeros(4, dtype=np.int64)
    n_att = np.zeros(4, dtype=np.int64)
    for rnd in range(12):
        g.sweep(2)
        for o in reps:
            o.sweep(2)
        g.exchange(rnd & 1)
        flags = oracle.replica_exchange(reps, kTs, tables, rnd & 1, 4242, rnd)
        n_acc += np.array(flags)
        n_att[(rnd & 1)::2] += 1
        st = g.state()
        assert st["last_flags"].tolist() == flags, rnd
        assert st["rounds"] == rnd + 1
        assert st["replica_at_slot"].tolist() == [o.tag for o in reps]
    st = _assert_slots_equal(g, reps, [o.tag for o in reps])
    assert st["accepted"].tolist() == n_acc.tolist() and st["attempted"].tolist() == n_att.tolist()
    assert 0 < n_acc.sum() < n_att.sum()            # both outcomes occurred
    # after the exchanges every replica sweeps at the temperature of its new slot
    g.sweep(3)
    for o in reps:
        o.sweep(3)
    _assert_slots_equal(g, reps, [o.tag for o in reps])
    for p, o in enumerate(reps):
        r = o.tag
        assert (g.replicas[r].energy_trace() == o.energy_trace()).all()
    g.close()


def test_run_is_the_same_as_step_by_step():
    """smcx_ensemble_run(rounds, k) == rounds x (sweep(k); exchange(round parity)), enqueued without
    any host synchronisation in between; also the anneal-length tables (different lengths per slot)."""
    cfg = scaled_config(1, (16, 16, 24))
    kTs = [430, 520, 610, 860]
    seeds = [77, 78, 79, 80]
    g, reps, tables = _ensemble(cfg, kTs, seeds, 5, smcx.KERNEL_AUTO)
    assert len({t.size for t in tables}) == 4
    for o in reps:
        o.tag = reps.index(o)
    g.run(9, 3)
    for rnd in range(9):
        for o in reps:
            o.sweep(3)
        oracle.replica_exchange(reps, kTs, tables, rnd & 1, 5, rnd)
    st = _assert_slots_equal(g, reps, [o.tag for o in reps])
    assert st["rounds"] == 9
    g.close()


def test_fcc_five_species_ensemble_with_the_sub_warp_kernel():
    """FCC, 5 species, 3 shells (the shape of config 3, and of the paper's alloy): the ensemble runs the
    sub-warp kernel; slots, energies and species against the oracle after graph-replayed rounds."""
    from smcx_inputs import make_epi
    lat, dims, n_sp, n_sh, w = 1, (16, 16, 8), 5, 3, 4
    epi = make_epi(n_sh, n_sp, 400, 1003)
    kTs = [650, 690, 730]
    tables = [make_accept_table(k) for k in kTs]
    seeds = [31, 32, 33]
    g = smcx.Ensemble(lat, dims, n_sp, n_sh, epi, kTs, tables, seeds, 99, link_cell=w)
    assert g.replicas[0].kernel == smcx.KERNEL_GROUP_PER_CELL
    reps = [oracle.Oracle(lat, dims, n_sp, n_sh, epi, w, tables[r], seeds[r]) for r in range(3)]
    for o in reps:
        o.tag = reps.index(o)
    g.run(6, 2)
    for rnd in range(6):
        for o in reps:
            o.sweep(2)
        oracle.replica_exchange(reps, kTs, tables, rnd & 1, 99, rnd)
    _assert_slots_equal(g, reps, [o.tag for o in reps])
    g.close()


@pytest.mark.parametrize("lat,dims,n_sp,n_sh,kernel", [
    (1, (16, 16, 8), 5, 3, smcx.KERNEL_FCC_THREAD),
    (0, (16, 8, 16), 6, 2, smcx.KERNEL_BCC4_THREAD),
], ids=["fcc_thread", "bcc4_thread"])
def test_ensembles_on_the_packed_kernels(lat, dims, n_sp, n_sh, kernel):
    """Replica exchange with the packed 4-bit kernels: their acceptance reads the head of the threshold table from
    shared memory and relies on a property of the table the host checks at upload; in an ensemble the tables move
    between replicas on the device (replica_apply_tables_kernel), with different lengths padded to the longest."""
    from smcx_inputs import make_epi
    w = 4
    epi = make_epi(n_sh, n_sp, 400, 1003)
    kTs = [300, 690, 1500]
    tables = [make_accept_table(k) for k in kTs]
    seeds = [41, 42, 43]
    g = smcx.Ensemble(lat, dims, n_sp, n_sh, epi, kTs, tables, seeds, 77, link_cell=w, kernel=kernel)
    assert g.replicas[0].kernel == kernel and g.replicas[0].storage == smcx.STORAGE_4BIT
    reps = [oracle.Oracle(lat, dims, n_sp, n_sh, epi, w, tables[r], seeds[r]) for r in range(3)]
    for o in reps:
        o.tag = reps.index(o)
    g.run(6, 2)
    for rnd in range(6):
        for o in reps:
            o.sweep(2)
        oracle.replica_exchange(reps, kTs, tables, rnd & 1, 77, rnd)
    st = _assert_slots_equal(g, reps, [o.tag for o in reps])
    assert int(st["attempted"].sum()) > 0
    g.close()


def test_two_replicas_parity_one_is_a_no_op():
    cfg = scaled_config(1, (16, 16, 16))
    kTs = [600, 640]
    g, reps, tables = _ensemble(cfg, kTs, [1, 2], 3, smcx.KERNEL_AUTO)
    g.sweep(1)
    g.exchange(1)                                   # no pair (1,2) with two replicas
    st = g.state()
    assert st["attempted"].tolist() == [0] and st["rounds"] == 1 and st["replica_at_slot"].tolist() == [0, 1]
    g.close()


def test_ensemble_argument_checks():
    cfg = scaled_config(1, (16, 16, 16))
    t = make_accept_table(600)
    with pytest.raises(smcx.SmcxError):
        smcx.Ensemble(cfg.lattice, cfg.dims, cfg.n_species, cfg.n_shells, cfg.epi(), [600], [t], [1], 1)
    with pytest.raises(smcx.SmcxError):
        smcx.Ensemble(cfg.lattice, cfg.dims, cfg.n_species, cfg.n_shells, cfg.epi(), [600, 0], [t, t], [1, 2], 1)


@pytest.mark.skipif(not __import__("os").environ.get("SMCX_SLOW"), reason="long run; set SMCX_SLOW=1")
def test_long_exchange_run_slow():
    """Eight replicas, 300 graph-replayed rounds of (2 sweeps + exchange): slots, counters, energies and species
    against the oracle at the end (dozens of accepted exchanges in between)."""
    cfg = scaled_config(1, (16, 16, 16))
    kTs = replica_ladder(600, 8, cfg.n_sites, 25.0 * np.sqrt(cfg.n_sites))
    seeds = [500 + r for r in range(8)]
    g, reps, tables = _ensemble(cfg, kTs, seeds, 2024, smcx.KERNEL_AUTO)
    for o in reps:
        o.tag = reps.index(o)
    g.run(300, 2)
    n_acc = np.zeros(7, dtype=np.int64)
    for rnd in range(300):
        for o in reps:
            o.sweep(2)
        n_acc += np.array(oracle.replica_exchange(reps, kTs, tables, rnd & 1, 2024, rnd))
    st = _assert_slots_equal(g, reps, [o.tag for o in reps])
    assert st["accepted"].tolist() == n_acc.tolist() and n_acc.sum() > 30
    g.close()


def _ladder_hitting(T_target, dE, kT_hi=2_100_000_000):
    """Integer temperatures (kT_0 < kT_1) for which floor(exp(Delta) 2^32) == T_target with the fractional part of
    exp(Delta) 2^32 well inside (0.25, 0.75), Delta = (kT_1 - kT_0) dE / (kT_0 kT_1), dE = E_0 - E_1 < 0: for kT_1
    near 2^31 one unit of kT_0 moves the threshold by a fraction of a unit, so a scan over kT_1 finds one quickly."""
    want = np.log((T_target + 0.5) / 4294967296.0)                 # Delta* < 0
    for kT1 in range(kT_hi, kT_hi - 4000, -1):
        kT0 = int(round(1.0 / (1.0 / kT1 + want / dE)))            # 1/kT0 - 1/kT1 = Delta*/dE
        if not 0 < kT0 < kT1:
            continue
        x = np.exp(oracle.exchange_delta(0, -dE, kT0, kT1)) * 4294967296.0
        if int(np.floor(x)) == T_target and 0.25 < x - np.floor(x) < 0.75:
            return kT0, kT1
    raise AssertionError("no ladder found")


@pytest.mark.parametrize("offset,expect", [(+1, 1), (0, 0), (-1, 0)], ids=["u=T-1", "u=T", "u=T+1"])
def test_exchange_decision_at_the_threshold(offset, expect):
    """S9's integer decision `u < floor(exp(Delta) 2^32)` exactly at its edge (Eq. 5): the two
    temperatures are constructed so that the threshold T is the Philox draw of the round plus 1, plus 0 and minus 1
    -- accept, reject, reject -- with exp(Delta) 2^32 far enough from an integer that CUDA's exp and libm's cannot
    round to different sides.  Energies: replica 0 a pure crystal (E = 0), replica 1 the B2 state (E = 4 N v)."""
    lat, dims, v = 0, (16, 16, 16), 15_000
    N = 2 * 16 ** 3
    epi = np.array([[[0, v], [v, 0]]], dtype=np.int32)
    dE = -4 * N * v                                                  # E_0 - E_1
    xseed = next(s for s in range(10_000, 20_000) if oracle.exchange_draw(s, 0, 0) > 0.90 * 2 ** 32
                 and oracle.exchange_draw(s, 0, 0) < 0.99 * 2 ** 32)
    u = oracle.exchange_draw(xseed, 0, 0)
    kT0, kT1 = _ladder_hitting(u + offset, dE)
    assert bool(oracle.exchange_accept(0, -dE, kT0, kT1, u)) == bool(expect)
    tiny = np.array([0xFFFFFFFF, 0], dtype=np.uint32)               # no sweeps are run: any table will do
    g = smcx.Ensemble(lat, dims, 2, 1, epi, [kT0, kT1], [tiny, tiny], [1, 2], xseed)
    s0 = np.zeros(N, np.uint8)
    s1 = np.zeros(N, np.uint8)
    s1[1::2] = 1
    g.replicas[0].set_species(s0)
    g.replicas[1].set_species(s1)
    assert g.replicas[0].running_energy() == 0 and g.replicas[1].running_energy() == -dE
    g.exchange(0)
    st = g.state()
    assert st["last_flags"].tolist() == [expect] and st["attempted"].tolist() == [1]
    assert st["replica_at_slot"].tolist() == ([1, 0] if expect else [0, 1])
    g.close()
