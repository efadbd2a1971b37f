"""Pins P5-P7, P14 and the S3/S4/S6 schedule details for the oracle."""
import numpy as np
import pytest

import oracle
from smcx_inputs import get_config, make_accept_table, make_epi, philox4x32_10, scaled_config
from pygeom import PyLattice

TAG_SHIFT, TAG_TRIAL, TAG_INIT = 1, 2, 3


def _small(cfg_id=1, dims=(8, 8, 8), **over):
    cfg = scaled_config(cfg_id, dims)
    return cfg, oracle.Oracle.from_config(cfg, **over)


def test_p5_p6_conservation_and_energy_bookkeeping():
    cfg, o = _small(1, (16, 16, 16))
    hist0 = np.bincount(o.species(), minlength=cfg.n_species)
    assert (hist0 == cfg.n_sites // cfg.n_species).all()
    E0 = o.energy()
    assert o.running_energy() == E0
    for t in range(6):
        o.sweep(1)
        assert (np.bincount(o.species(), minlength=cfg.n_species) == hist0).all()
        assert o.energy() == o.running_energy() == o.energy_trace()[t]
    sweeps, trials, accepted = o.stats()
    assert sweeps == 6 and trials == 6 * cfg.n_sites and 0 < accepted < trials


def test_p5_p6_fcc_three_shells():
    cfg, o = _small(3, (8, 8, 8))
    hist0 = np.bincount(o.species(), minlength=5)
    assert sorted(hist0)[0] >= cfg.n_sites // 5 and hist0.sum() == cfg.n_sites
    o.sweep(3)
    assert (np.bincount(o.species(), minlength=5) == hist0).all()
    assert o.energy() == o.running_energy()


@pytest.mark.parametrize("cfg_id,dims", [(1, (16, 16, 16)), (3, (8, 8, 16))])
def test_p7_same_colour_cells_commute_and_each_site_visited_once(cfg_id, dims):
    cfg = scaled_config(cfg_id, dims)
    runs = []
    for mode in (0, 1, 2):
        o = oracle.Oracle.from_config(cfg)
        assert o.lc_valid()
        o.count_visits(True)
        o.sweep(3, order_mode=mode, order_seed=123)
        assert (o.visits() == 3).all()          # every site exactly once per step
        runs.append((o.species(), o.energy_trace()))
    for s, tr in runs[1:]:
        assert (s == runs[0][0]).all() and (tr == runs[0][1]).all()


def test_p7_link_cell_below_bound_is_order_dependent():
    """w=1 violates 2w >= 2 r0 + R: the oracle reports it and the result depends on cell order."""
    cfg = scaled_config(1, (8, 8, 8))
    outs = []
    for mode in (0, 1):
        o = oracle.Oracle.from_config(cfg, link_cell=1)
        assert not o.lc_valid()
        o.sweep(2, order_mode=mode)
        outs.append(o.species())
    assert (outs[0] != outs[1]).any()


def test_lc_validity_bound():
    """S2: BCC 2 shells and FCC 3 shells need w >= 2; BCC 4 shells need w >= 3."""
    def valid(lat, n_shells, w, L):
        epi = np.zeros((n_shells, 2, 2), np.int32)
        return oracle.Oracle(lat, (L, L, L), 2, n_shells, epi, w, np.zeros(2, np.uint32), 0,
                             init=False).lc_valid()
    assert not valid(0, 2, 1, 8) and valid(0, 2, 2, 8) and valid(0, 2, 4, 8)
    assert not valid(1, 3, 1, 8) and valid(1, 3, 2, 8)
    assert not valid(0, 4, 2, 12) and valid(0, 4, 3, 12)
    assert not valid(0, 2, 4, 12)       # 12 is not divisible by 2w = 8


def test_p14_determinism_and_resume():
    cfg = scaled_config(1, (8, 8, 8))
    a = oracle.Oracle.from_config(cfg)
    b = oracle.Oracle.from_config(cfg)
    c = oracle.Oracle.from_config(cfg, seed=cfg.seed + 1)
    a.sweep(5)
    b.sweep(2)
    b.sweep(3)
    c.sweep(5)
    assert (a.species() == b.species()).all() and (a.energy_trace() == b.energy_trace()).all()
    assert (a.species() != c.species()).any()


def test_s3_shift_is_the_documented_philox_draw_and_covers_the_range():
    cfg, o = _small(1)
    key = (cfg.seed & 0xFFFFFFFF, cfg.seed >> 32)
    seen = set()
    for t in range(200):
        r = philox4x32_10((0, 0, t, TAG_SHIFT), key)
        expect = tuple((r[a] * cfg.link_cell) >> 32 for a in range(3))
        assert o.shift(t) == expect
        seen.add(expect)
    assert len(seen) > 50 and all(0 <= v < cfg.link_cell for s in seen for v in s)


def test_s3_s4_one_sweep_against_python_restatement():
    """One LC sweep on BCC 4^3 (w=2: one cell per colour) replayed in pure Python from the text
    of S3/S4, with dE from full energy recomputation.  A consistency check of indices and
    counter layout (not an independent pin: it restates the same reading)."""
    n_sp, w, dims, seed, kT = 3, 2, (4, 4, 4), 4242, 500
    epi = make_epi(2, n_sp, 300, seed)
    T = make_accept_table(kT)
    o = oracle.Oracle(0, dims, n_sp, 2, epi, w, T, seed)
    pl = PyLattice(0, dims, 2)
    sigma = o.species().astype(np.int64)
    key = (seed & 0xFFFFFFFF, seed >> 32)
    E = pl.energy(sigma, epi)
    trace = []
    nc = [d // w for d in dims]
    for t in range(2):
        r = philox4x32_10((0, 0, t, TAG_SHIFT), key)
        org = [(r[a] * w) >> 32 for a in range(3)]
        for colour in range(8):
            for cz in range(nc[2]):
                for cy in range(nc[1]):
                    for cx in range(nc[0]):
                        if (cx & 1) | ((cy & 1) << 1) | ((cz & 1) << 2) != colour:
                            continue
                        cell = (cz * nc[1] + cy) * nc[0] + cx
                        for k in range(w * w * w * 2):
                            b, rest = k % 2, k // 2
                            lx, ly, lz = rest % w, (rest // w) % w, rest // (w * w)
                            x = (org[0] + cx * w + lx) % dims[0]
                            y = (org[1] + cy * w + ly) % dims[1]
                            z = (org[2] + cz * w + lz) % dims[2]
                            i = ((z * dims[1] + y) * dims[0] + x) * 2 + b
                            rr = philox4x32_10((cell, k >> 1, t, TAG_TRIAL | (colour << 8)), key)
                            wd, u = (rr[2], rr[3]) if k & 1 else (rr[0], rr[1])
                            j = int(pl.nbr[0][i, (wd * 8) >> 32])
                            if sigma[i] == sigma[j]:
                                continue
                            s2 = sigma.copy()
                            s2[i], s2[j] = sigma[j], sigma[i]
                            dE = pl.energy(s2, epi) - E
                            if dE <= 0 or (dE < len(T) and u < int(T[dE])):
                                sigma, E = s2, E + dE
        trace.append(E)
    o.sweep(2)
    assert (o.species() == sigma).all()
    assert list(o.energy_trace()) == trace


def test_s6_initial_state_is_a_seeded_permutation_with_exact_counts():
    for N_dims, n_sp in (((2, 2, 2), 2), ((4, 2, 2), 3), ((4, 4, 6), 5), ((6, 4, 4), 4)):
        epi = np.zeros((1, n_sp, n_sp), np.int32)
        o = oracle.Oracle(0, N_dims, n_sp, 1, epi, 1, np.zeros(2, np.uint32), 99)
        N = o.n_sites
        perm = np.array([o.init_permutation(i) for i in range(N)])
        assert sorted(perm) == list(range(N))                      # bijection of [0, N)
        assert (o.species() == perm % n_sp).all()
        counts = np.bincount(o.species(), minlength=n_sp)
        assert (counts == [N // n_sp + (p < N % n_sp) for p in range(n_sp)]).all()
        o2 = oracle.Oracle(0, N_dims, n_sp, 1, epi, 1, np.zeros(2, np.uint32), 100)
        assert N <= 16 or (o2.species() != o.species()).any()


def test_s6_feistel_round_function_is_the_documented_philox_draw():
    """pi(i) replayed in Python from S6 (4 rounds, F = philox((R, round, 0, TAG_INIT))[0] & mask)."""
    seed, dims = 31337, (4, 4, 6)
    epi = np.zeros((1, 2, 2), np.int32)
    o = oracle.Oracle(0, dims, 2, 1, epi, 1, np.zeros(2, np.uint32), seed)
    N = o.n_sites
    h = 1
    while (1 << (2 * h)) < N:
        h += 1
    mask = (1 << h) - 1
    key = (seed & 0xFFFFFFFF, seed >> 32)
    for i in range(0, N, 7):
        v = i
        while True:
            left, right = v >> h, v & mask
            for rnd in range(4):
                f = philox4x32_10((right, rnd, 0, TAG_INIT), key)[0] & mask
                left, right = right, left ^ f
            v = (left << h) | right
            if v < N:
                break
        assert o.init_permutation(i) == v


def test_s6_equiatomic_counts_config3_remainder():
    cfg = get_config(3)
    N = cfg.n_sites
    assert N % 5 == 3
    assert [N // 5 + (p < 3) for p in range(5)] == [1677722] * 3 + [1677721] * 2


def test_resume_from_a_checkpoint_is_exact():
    """Checkpoint = (species array, sweep counter, seed): a fresh oracle given both continues the run bit for
    bit (the draws depend on the counters only), while a wrong counter gives a different trajectory."""
    cfg = scaled_config(1, (16, 16, 16))
    a = oracle.Oracle.from_config(cfg)
    a.sweep(4)
    saved, t = a.species().copy(), a.stats()[0]
    a.sweep(3)
    b = oracle.Oracle.from_config(cfg)
    b.set_species(saved)
    b.set_sweep_counter(t)
    b.sweep(3)
    assert (a.species() == b.species()).all()
    assert (a.energy_trace(4, 3) == b.energy_trace(4, 3)).all() and b.stats()[:2] == a.stats()[:2]
    with pytest.raises(IndexError):
        b.energy_trace(0, 1)                      # the trace restarts at the resume point
    c = oracle.Oracle.from_config(cfg)
    c.set_species(saved)
    c.set_sweep_counter(t + 1)
    c.sweep(3)
    assert (a.species() != c.species()).any()


@pytest.mark.parametrize("cfg_id,dims,threads", [(1, (16, 16, 16), 2), (1, (24, 16, 32), 5), (3, (16, 8, 16), 4),
                                                 (3, (8, 8, 8), 16)])
def test_p7_threads_over_the_cells_of_a_colour_change_nothing(cfg_id, dims, threads):
    """Multi-thread twin of P7 (the OpenMP pragma on the per-colour cell loop "must reproduce
    the 1-thread result bit for bit"): initial state, species after every sweep, trace, counters, visit counts,
    recomputed energy and pair counts are those of the plain loop, also with more threads than cells of a colour
    (FCC 8^3 has one) and with the shuffled cell order."""
    cfg = scaled_config(cfg_id, dims)
    one = oracle.Oracle.from_config(cfg)
    many = oracle.Oracle.from_config(cfg, threads=threads)
    assert one.threads == 1 and many.threads == threads
    assert (one.species() == many.species()).all()                  # S6 under threads
    assert one.energy() == many.energy()
    many.count_visits(True)
    for t in range(4):
        one.sweep(1)
        many.sweep(1, order_mode=2 if t & 1 else 0, order_seed=7)
        assert (one.species() == many.species()).all()
    assert (many.visits() == 4).all()
    assert (one.energy_trace() == many.energy_trace()).all()
    assert one.stats() == many.stats()
    assert one.energy() == many.energy() == many.running_energy()
    assert (one.sro()[1] == many.sro()[1]).all()
    counts = [cfg.n_sites - 3 * (cfg.n_sites // 5)] + [cfg.n_sites // 5] * 3 + [0] * (cfg.n_species - 4)
    one.init_composition(counts)
    many.init_composition(counts)
    assert (one.species() == many.species()).all()                  # S10 under threads
    many.set_threads(1)
    one.set_threads(3)
    one.sweep(2)
    many.sweep(2)
    assert (one.species() == many.species()).all() and one.running_energy() == many.running_energy()
