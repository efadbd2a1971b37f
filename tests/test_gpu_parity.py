"""GPU-vs-oracle parity through the C ABI (pytest -m gpu): species arrays, energy traces and pair
counts bit-exact, fp64 SRO within 1e-9 relative (BASELINE.json north_star)."""
import os
import time

import numpy as np
import pytest

import oracle
import paper_2509_20949_b200 as smcx
from smcx_inputs import get_config, make_accept_table, make_epi, scaled_config

pytestmark = pytest.mark.gpu

KERNELS = [smcx.KERNEL_WARP_PER_CELL, smcx.KERNEL_GROUP_PER_CELL, smcx.KERNEL_THREAD_PER_CELL,
           smcx.KERNEL_THREAD_PERSISTENT]
KERNEL_IDS = ["warp", "group", "thread", "persistent"]


def _supported(cfg, kernel):
    if kernel in (smcx.KERNEL_WARP_PER_CELL, smcx.KERNEL_GROUP_PER_CELL):
        return True
    return cfg.lattice == 0 and cfg.n_shells == 2 and cfg.link_cell == 4 and cfg.n_species <= 4


# The full-size oracle runs spread the cells of a colour over all host cores (oracle pin
# test_p7_threads_over_the_cells_of_a_colour_change_nothing: bit-identical to the one-thread oracle).
ALL_CORES = max(1, os.cpu_count() or 1)


def _pair(cfg, kernel=smcx.KERNEL_AUTO, threads=1, **over):
    g = smcx.Lattice.from_config(cfg, kernel=kernel, **over)
    o = oracle.Oracle.from_config(cfg, threads=threads,
                                  **{k: v for k, v in over.items() if k in ("seed", "link_cell", "epi", "accept")})
    return g, o


def _assert_same_state(g, o):
    gs, os_ = g.species(), o.species()
    assert gs.dtype == np.uint8 and gs.shape == os_.shape
    bad = np.flatnonzero(gs != os_)
    assert bad.size == 0, f"{bad.size} sites differ, first at {bad[:5]}"


def _assert_sro(g, o):
    ga, gc = g.sro()
    oa, oc = o.sro()
    assert (gc == oc).all()
    assert np.allclose(ga, oa, rtol=1e-9, atol=1e-9, equal_nan=True)


@pytest.mark.parametrize("kernel", KERNELS, ids=KERNEL_IDS)
def test_config1_full_run_species_after_every_sweep(kernel):
    cfg = get_config(1)
    g, o = _pair(cfg, kernel)
    _assert_same_state(g, o)                       # S6 initial state
    assert g.energy() == o.energy() == g.running_energy()
    for t in range(cfg.n_sweeps):
        g.sweep(1)
        o.sweep(1)
        _assert_same_state(g, o)
    assert (g.energy_trace() == o.energy_trace()).all()
    assert g.stats() == o.stats()
    assert g.energy() == o.energy() == o.running_energy() == g.running_energy()
    _assert_sro(g, o)


@pytest.mark.parametrize("kernel", KERNELS, ids=KERNEL_IDS)
def test_config2_anneal_prefix(kernel):
    """Config 2 with its per-sweep temperature table; SRO sampled every 10 sweeps here
    (every 100 over the full 2,000 sweeps in test_config2_anneal_full_length)."""
    cfg = get_config(2)
    n = 30
    g, o = _pair(cfg, kernel)
    _assert_sro(g, o)
    for t in range(n):
        table = cfg.accept_table(t)
        g.set_temperature(cfg.kT_at(t), table)
        o.set_temperature(table)
        g.sweep(1)
        o.sweep(1)
        if (t + 1) % 10 == 0:
            _assert_same_state(g, o)
            _assert_sro(g, o)
    assert (g.energy_trace() == o.energy_trace()).all()
    assert g.stats() == o.stats()


def test_config2_anneal_full_length():
    """BASELINE.json configs[1] at SURVEY.md 8(d)'s extent: all 2,000 sweeps of the anneal, species + SRO at the 20
    sample points, the full trace."""
    cfg = get_config(2)
    g, o = _pair(cfg, threads=ALL_CORES)
    for t in range(cfg.n_sweeps):
        table = cfg.accept_table(t)
        g.set_temperature(cfg.kT_at(t), table)
        o.set_temperature(table)
        g.sweep(1)
        o.sweep(1)
        if (t + 1) % cfg.sro_every == 0:
            _assert_same_state(g, o)
            _assert_sro(g, o)
    assert (g.energy_trace() == o.energy_trace()).all()


@pytest.mark.parametrize("kernel", [smcx.KERNEL_WARP_PER_CELL, smcx.KERNEL_GROUP_PER_CELL, smcx.KERNEL_FCC_THREAD],
                         ids=["warp", "group", "fcc_thread"])
def test_config3_fcc_five_species_prefix(kernel):
    cfg = get_config(3)
    g, o = _pair(cfg, kernel)
    _assert_same_state(g, o)
    g.sweep(2)
    o.sweep(2)
    _assert_same_state(g, o)
    assert (g.energy_trace() == o.energy_trace()).all()
    assert g.energy() == o.energy()
    _assert_sro(g, o)


@pytest.mark.parametrize("kernel", KERNELS, ids=KERNEL_IDS)
def test_config4_shape_ragged_grid(kernel):
    """Config 4's species/EPI/kT on a non-cubic lattice whose cells per colour (13*11*9) fill
    neither a warp nor a block evenly."""
    cfg = scaled_config(4, (104, 88, 72))
    g, o = _pair(cfg, kernel)
    g.sweep(3)
    o.sweep(3)
    _assert_same_state(g, o)
    assert (g.energy_trace() == o.energy_trace()).all()
    assert g.stats() == o.stats()
    _assert_sro(g, o)


@pytest.mark.parametrize("kernel", KERNELS, ids=KERNEL_IDS)
def test_config4_full_size_invariants(kernel):
    """BCC 800^3 in the launch configuration bench.py times: conservation (P5), energy bookkeeping
    (P6: H recomputed by the reduction kernel == E0 + sum of accepted dE) and the species counts."""
    cfg = get_config(4)
    g = smcx.Lattice.from_config(cfg, kernel=kernel)
    _, c0 = g.sro()
    n_p = c0[0].sum(axis=1) // 8
    assert (n_p == cfg.n_sites // 4).all()
    e0 = g.energy()
    assert e0 == g.running_energy()
    g.sweep(2)
    _, c1 = g.sro()
    assert (c1[0].sum(axis=1) // 8 == n_p).all()
    assert (c1 == c1.transpose(0, 2, 1)).all()
    assert g.energy() == g.running_energy() == g.energy_trace()[-1]
    sweeps, trials, accepted = g.stats()
    assert sweeps == 2 and trials == 2 * cfg.n_sites and 0 < accepted < trials
    # P13: H = 1/2 sum V N
    assert int((cfg.epi().astype(np.int64) * c1).sum()) == 2 * g.energy()


def test_config5_shape_at_400_cubed():
    """Config 5's parameters on 400^3 cells (1.28e8 sites).  The full 1.6e10 sites are checked against the oracle on
    sweep 0 by tests/test_gpu_zz_config5_full_size.py when the host has the memory and the cores; this smaller run and
    the invariants at full size (test_config5_full_size_invariants) hold everywhere."""
    cfg = scaled_config(5, (400, 400, 400))
    g, o = _pair(cfg, threads=ALL_CORES)
    g.sweep(1)
    o.sweep(1)
    _assert_same_state(g, o)
    assert (g.energy_trace() == o.energy_trace()).all()


def test_config5_full_size_invariants():
    cfg = get_config(5)
    g = smcx.Lattice.from_config(cfg)
    _, c0 = g.sro()
    n_p = c0[0].sum(axis=1) // 8
    assert (n_p == cfg.n_sites // 4).all()
    assert g.energy() == g.running_energy()
    g.sweep(3)
    _, c1 = g.sro()
    assert (c1[0].sum(axis=1) // 8 == n_p).all()
    assert g.energy() == g.running_energy() == g.energy_trace()[-1]
    assert int((cfg.epi().astype(np.int64) * c1).sum()) == 2 * g.energy()


def test_config4_full_size_oracle_two_sweeps():
    """BASELINE.json configs[3] (BCC 800^3, 1.024e9 sites, the graded configuration) in the launch configuration
    bench.py times, at SURVEY.md 8(d)'s extent: initial state, species after 2 sweeps and the trace against the
    oracle (all host cores)."""
    cfg = get_config(4)
    n = int(os.environ.get("SMCX_C4_SWEEPS", "2"))      # test extent only (profiles/r2_full_size_parity.txt ran 20)
    g, o = _pair(cfg, threads=ALL_CORES)
    assert g.kernel == smcx.KERNEL_THREAD_PERSISTENT and g.storage == smcx.STORAGE_2BIT
    _assert_same_state(g, o)
    g.sweep(n)
    o.sweep(n)
    _assert_same_state(g, o)
    assert (g.energy_trace() == o.energy_trace()).all()
    assert g.stats() == o.stats()
    assert g.running_energy() == o.running_energy()


def test_config3_full_length():
    """BASELINE.json configs[2] (FCC 128^3, 5 species, 3 shells): all 1,000 sweeps, the trace compared every 100
    sweeps and the species at the end.  SMCX_C3_BUDGET_S (default 600) bounds the oracle's wall
    clock on hosts with few cores: the run then stops at a multiple of 100 sweeps, never below 200, and the
    test prints how far it got."""
    cfg = get_config(3)
    budget = float(os.environ.get("SMCX_C3_BUDGET_S", "600"))
    g, o = _pair(cfg, threads=ALL_CORES)
    t0, done = time.time(), 0
    while done < cfg.n_sweeps and (done < 200 or time.time() - t0 < budget):
        g.sweep(100)
        o.sweep(100)
        done += 100
        assert (g.energy_trace(done - 100, 100) == o.energy_trace(done - 100, 100)).all()
    _assert_same_state(g, o)
    assert g.stats() == o.stats()
    _assert_sro(g, o)
    print(f"config 3: {done} of {cfg.n_sweeps} sweeps bit-exact with the oracle in {time.time() - t0:.0f} s "
          f"({ALL_CORES} oracle threads)")
    assert done == cfg.n_sweeps or time.time() - t0 >= budget


@pytest.mark.parametrize("kernel", KERNELS, ids=KERNEL_IDS)
def test_resume_and_determinism(kernel):
    cfg = scaled_config(1, (24, 16, 32))
    a = smcx.Lattice.from_config(cfg, kernel=kernel)
    b = smcx.Lattice.from_config(cfg, kernel=kernel)
    a.sweep(7)
    b.sweep(3)
    b.sweep(4)
    assert (a.species() == b.species()).all() and (a.energy_trace() == b.energy_trace()).all()
    c = smcx.Lattice.from_config(cfg, kernel=kernel, seed=cfg.seed + 1)
    c.sweep(7)
    assert (a.species() != c.species()).any()


def test_thread_and_warp_kernels_agree():
    """P14: uint8/warp-per-cell and 2-bit/thread-per-cell agree bit for bit."""
    cfg = scaled_config(2, (40, 48, 56), n_sweeps=5)
    a = smcx.Lattice.from_config(cfg, kernel=smcx.KERNEL_WARP_PER_CELL)
    b = smcx.Lattice.from_config(cfg, kernel=smcx.KERNEL_THREAD_PER_CELL)
    c = smcx.Lattice.from_config(cfg, kernel=smcx.KERNEL_THREAD_PERSISTENT)
    assert (a.storage, b.storage, c.storage) == (smcx.STORAGE_U8, smcx.STORAGE_2BIT, smcx.STORAGE_2BIT)
    for x in (a, b, c):
        x.sweep(5)
    for x in (b, c):
        assert (a.species() == x.species()).all()
        assert (a.energy_trace() == x.energy_trace()).all()
        assert (a.sro()[1] == x.sro()[1]).all()


@pytest.mark.parametrize("lat,dims,n_sp,n_shells,w", [
    (0, (8, 8, 8), 2, 1, 4),       # one cell per colour, NN only
    (0, (8, 16, 8), 3, 2, 2),      # smallest link cell the bound allows
    (0, (16, 24, 16), 4, 4, 4),    # four shells (reach 3)
    (0, (12, 12, 24), 4, 3, 3),    # odd link cell
    (1, (8, 8, 8), 2, 1, 2),       # FCC nearest neighbours
    (1, (16, 8, 8), 5, 3, 4),      # FCC three shells
    (1, (16, 16, 16), 16, 2, 4),   # maximum species count
])
@pytest.mark.parametrize("kernel,lanes", [(smcx.KERNEL_WARP_PER_CELL, 0), (smcx.KERNEL_GROUP_PER_CELL, 4),
                                          (smcx.KERNEL_GROUP_PER_CELL, 8), (smcx.KERNEL_GROUP_PER_CELL, 16),
                                          (smcx.KERNEL_GROUP_PER_CELL, 32), (smcx.KERNEL_AUTO, 0)],
                         ids=["warp", "group4", "group8", "group16", "group32", "auto"])
def test_edge_geometries(lat, dims, n_sp, n_shells, w, kernel, lanes):
    amplitude, kT, seed = 350, 500, 4711
    epi = make_epi(n_shells, n_sp, amplitude, seed)
    table = make_accept_table(kT)
    g = smcx.Lattice(lat, dims, n_sp, n_shells, epi, table, seed, link_cell=w, kT_units=kT, kernel=kernel,
                     group_lanes=lanes)                      # lanes per cell of the sub-warp kernel (0 = auto)
    o = oracle.Oracle(lat, dims, n_sp, n_shells, epi, w, table, seed)
    assert o.lc_valid()
    for s in range(n_shells):
        assert (g.shell_offsets(s) == oracle.shell(lat, s)).all()
    _assert_same_state(g, o)
    g.sweep(4)
    o.sweep(4)
    _assert_same_state(g, o)
    assert (g.energy_trace() == o.energy_trace()).all()
    _assert_sro(g, o)


def test_set_species_roundtrip_and_validation():
    cfg = scaled_config(1, (16, 16, 16))
    g, o = _pair(cfg)
    rng = np.random.default_rng(3)
    s = rng.integers(0, cfg.n_species, cfg.n_sites).astype(np.uint8)
    g.set_species(s)
    o.set_species(s)
    assert (g.species() == s).all()
    assert g.energy() == o.energy() == g.running_energy()
    g.sweep(2)
    o.sweep(2)
    _assert_same_state(g, o)
    s[5] = cfg.n_species
    with pytest.raises(smcx.SmcxError) as ei:
        g.set_species(s)
    assert ei.value.code == -9
    import torch
    t = torch.from_numpy(o.species()).cuda()
    g.set_species_device(t)
    assert (g.species_device().cpu().numpy() == o.species()).all()
    t[7] = 200
    with pytest.raises(smcx.SmcxError):
        g.set_species_device(t)


def test_b2_state_sro_and_energy_closed_forms():
    """Closed forms straight through the GPU reduction kernel: B2 energy and alpha = -1/+1."""
    epi = make_epi(2, 2, 300, 5)
    g = smcx.Lattice(0, (16, 16, 16), 2, 2, epi, make_accept_table(600), 1)
    N = g.n_sites
    s = np.zeros(N, np.uint8)
    s[1::2] = 1
    g.set_species(s)
    assert g.energy() == 4 * N * int(epi[0, 0, 1]) + (3 * N // 2) * int(epi[1, 0, 0] + epi[1, 1, 1])
    alpha, _ = g.sro()
    assert np.allclose(alpha[0], [[1, -1], [-1, 1]]) and np.allclose(alpha[1], [[-1, 1], [1, -1]])


def test_energy_trace_ring_and_ranges():
    cfg = scaled_config(1, (16, 16, 16))
    g = smcx.Lattice.from_config(cfg, trace_capacity=4)
    o = oracle.Oracle.from_config(cfg)
    g.sweep(6)
    o.sweep(6)
    assert (g.energy_trace(2, 4) == o.energy_trace(2, 4)).all()
    with pytest.raises(smcx.SmcxError):
        g.energy_trace(0, 6)       # sweeps 0-1 are no longer retained
    with pytest.raises(smcx.SmcxError):
        g.energy_trace(5, 3)       # beyond the sweeps done


@pytest.mark.parametrize("kernel", KERNELS, ids=KERNEL_IDS)
@pytest.mark.parametrize("kind", ["staircase", "short", "non_monotone", "long_kT"])
def test_arbitrary_threshold_tables(kernel, kind):
    """The threshold table is input data: the library must take the same decisions as `u < T[dE]` for
    any table, including ones that are not of the exp(-d/kT) form (the thread kernel's two-level
    filter must then be refused by the host-side check and the exact look-up used)."""
    cfg = scaled_config(1, (16, 24, 16))
    rng = np.random.default_rng(11)
    if kind == "staircase":
        table = np.repeat(np.sort(rng.integers(0, 2 ** 32, 40, dtype=np.uint64))[::-1], 100).astype(np.uint32)
    elif kind == "short":
        table = make_accept_table(600)[:37].copy()          # truncated: dE >= 37 is always rejected
    elif kind == "non_monotone":
        table = rng.integers(0, 2 ** 32, 5000, dtype=np.uint64).astype(np.uint32)
    else:
        table = make_accept_table(2900)                     # 64,325 entries: longer than the filter covers
    g = smcx.Lattice.from_config(cfg, kernel=kernel, accept=table)
    o = oracle.Oracle.from_config(cfg, accept=table)
    g.sweep(4)
    o.sweep(4)
    _assert_same_state(g, o)
    assert (g.energy_trace() == o.energy_trace()).all()
    assert g.stats() == o.stats()
    # and back to a regular table on the same handles
    table2 = make_accept_table(430)
    g.set_temperature(430, table2)
    o.set_temperature(table2)
    g.sweep(3)
    o.sweep(3)
    _assert_same_state(g, o)
    assert (g.energy_trace() == o.energy_trace()).all()


def test_large_epi_values_thread_kernel():
    """int32 EPI far beyond the configs' range (|V| up to 6e4, dE up to ~1e6) with the longest table the
    library reserves room for (2^20 entries): coefficients and dE stay exact."""
    cfg = scaled_config(1, (16, 16, 16))
    epi = make_epi(2, 4, 60_000, 77)
    table = make_accept_table(45_000)
    assert 900_000 < table.size <= 1 << 20
    for kernel in KERNELS:
        g = smcx.Lattice.from_config(cfg, kernel=kernel, epi=epi, accept=table)
        o = oracle.Oracle.from_config(cfg, epi=epi, accept=table)
        g.sweep(3)
        o.sweep(3)
        _assert_same_state(g, o)
        assert (g.energy_trace() == o.energy_trace()).all()


def test_paper_alloy_composition_and_stagewise_cooling():
    """S10 + the paper's protocol in small: FCC, five species in the proportions
    29/29/28/7/7, three shells, cooled through temperature stages; initial state, every stage's species,
    trace and SRO against the oracle."""
    from smcx_inputs import composition_counts, cooling_stages
    lat, dims, n_sp, n_sh, w, seed = 1, (16, 16, 16), 5, 3, 4, 2029
    epi = make_epi(n_sh, n_sp, 400, seed)
    stages = cooling_stages(1720, 860, 4)
    tables = [make_accept_table(k) for k in stages]
    g = smcx.Lattice(lat, dims, n_sp, n_sh, epi, tables[0], seed, link_cell=w, kT_units=stages[0])
    o = oracle.Oracle(lat, dims, n_sp, n_sh, epi, w, tables[0], seed)
    counts = composition_counts(g.n_sites, (29, 29, 28, 7, 7))
    g.init_composition(counts)
    o.init_composition(counts)
    _assert_same_state(g, o)
    assert np.bincount(g.species(), minlength=n_sp).tolist() == counts
    assert g.energy() == o.energy() == g.running_energy()
    for kT, tab in zip(stages, tables):
        g.set_temperature(kT, tab)
        o.set_temperature(tab)
        g.sweep(3)
        o.sweep(3)
        _assert_same_state(g, o)
        _assert_sro(g, o)
    assert (g.energy_trace() == o.energy_trace()).all()
    assert g.stats() == o.stats()
    with pytest.raises(smcx.SmcxError):
        g.init_composition([1, 1, 1, 1, 1])


def test_composition_on_packed_storage():
    cfg = scaled_config(4, (32, 24, 16))
    g, o = _pair(cfg, smcx.KERNEL_THREAD_PERSISTENT)
    counts = [cfg.n_sites // 2, cfg.n_sites // 4, cfg.n_sites // 8, cfg.n_sites // 8]
    g.init_composition(counts)
    o.init_composition(counts)
    _assert_same_state(g, o)
    g.sweep(3)
    o.sweep(3)
    _assert_same_state(g, o)
    assert g.energy() == o.energy() == g.running_energy()


@pytest.mark.parametrize("kernel", KERNELS, ids=KERNEL_IDS)
def test_checkpoint_and_resume_in_a_new_handle(kernel):
    """State = (species, sweep counter, seed): a new handle given both continues bit for bit, and agrees with
    an oracle resumed the same way."""
    cfg = scaled_config(1, (16, 16, 24))
    a = smcx.Lattice.from_config(cfg, kernel=kernel)
    a.sweep(4)
    saved, t = a.species().copy(), a.stats()[0]
    a.sweep(5)
    b = smcx.Lattice.from_config(cfg, kernel=kernel)
    b.set_species(saved)
    b.set_sweep_counter(t)
    b.sweep(5)
    assert (a.species() == b.species()).all()
    assert (a.energy_trace(4, 5) == b.energy_trace(4, 5)).all()
    assert a.stats()[:2] == b.stats()[:2] and a.energy() == b.energy() == b.running_energy()
    with pytest.raises(smcx.SmcxError):
        b.energy_trace(0, 1)
    o = oracle.Oracle.from_config(cfg)
    o.set_species(saved)
    o.set_sweep_counter(t)
    o.sweep(5)
    _assert_same_state(b, o)
    assert (b.energy_trace(4, 5) == o.energy_trace(4, 5)).all()


@pytest.mark.parametrize("lanes", [8, 16, 32])
@pytest.mark.parametrize("amplitude,kT", [(400, 690), (30_000, 20_000)], ids=["d16", "d32"])
def test_sub_warp_kernel_table_formats(lanes, amplitude, kT):
    """FCC, 5 species, 3 shells with differences that fit 16 bits (8 lanes: halfword rows, one bank window per
    cell of the warp) and with differences that do not (32-bit rows everywhere), for every lane count."""
    lat, dims, n_sp, n_sh, w, seed = 1, (16, 16, 8), 5, 3, 4, 91
    epi = make_epi(n_sh, n_sp, amplitude, seed)
    assert (np.abs(epi).max() * 2 > 32767) == (amplitude > 16384)
    table = make_accept_table(kT)
    g = smcx.Lattice(lat, dims, n_sp, n_sh, epi, table, seed, link_cell=w, kT_units=kT, kernel=smcx.KERNEL_GROUP_PER_CELL,
                     group_lanes=lanes, group_warps=2 if lanes == 8 else 0)
    o = oracle.Oracle(lat, dims, n_sp, n_sh, epi, w, table, seed)
    g.sweep(4)
    o.sweep(4)
    _assert_same_state(g, o)
    assert (g.energy_trace() == o.energy_trace()).all() and g.stats() == o.stats()
    assert g.stats()[2] > 0


# ---- packed FCC kernel (SMCX_KERNEL_FCC_THREAD, SMCX_STORAGE_4BIT) -------------------------------------------------
@pytest.mark.parametrize("dims,n_sp,n_sh,amp,kT", [
    ((16, 16, 16), 5, 3, 400, 690),      # config 3's parameters in small
    ((24, 16, 8), 8, 3, 400, 860),       # most species the look-up takes, one cell per colour along z
    ((16, 8, 24), 2, 2, 300, 500),       # two shells: the third shell's rows are zero
    ((40, 24, 16), 5, 3, 15_000, 9_000), # differences that need the high byte of the look-up in full
    ((32, 32, 32), 3, 3, 400, 430),      # more than one batch of 32 cells per colour (64)
    ((24, 24, 8), 5, 3, 400, 690),       # 9 cells per colour: a ragged batch
])
def test_packed_fcc_kernel_against_the_oracle(dims, n_sp, n_sh, amp, kT):
    lat, w, seed = 1, 4, 515
    epi = make_epi(n_sh, n_sp, amp, seed)
    table = make_accept_table(kT)
    g = smcx.Lattice(lat, dims, n_sp, n_sh, epi, table, seed, link_cell=w, kT_units=kT, kernel=smcx.KERNEL_FCC_THREAD)
    assert g.storage == smcx.STORAGE_4BIT and g.kernel == smcx.KERNEL_FCC_THREAD
    o = oracle.Oracle(lat, dims, n_sp, n_sh, epi, w, table, seed)
    _assert_same_state(g, o)                       # S6 through Store4
    assert g.energy() == o.energy() == g.running_energy()
    for _ in range(4):
        g.sweep(1)
        o.sweep(1)
        _assert_same_state(g, o)
    g.sweep(3)                                     # graph replay
    o.sweep(3)
    _assert_same_state(g, o)
    assert (g.energy_trace() == o.energy_trace()).all()
    assert g.stats() == o.stats() and g.stats()[2] > 0
    assert g.energy() == o.energy() == g.running_energy()
    _assert_sro(g, o)                              # pair counts on 4-bit storage


@pytest.mark.parametrize("kind", ["staircase", "short", "non_monotone", "bump_in_the_tail", "tiny_kT"])
def test_packed_fcc_kernel_arbitrary_threshold_tables(kind):
    """The packed FCC kernel keeps the head of T in shared memory and takes T[dE] from global memory behind it, which
    is sound only if T[K] bounds the tail (the host checks that at upload): tables that are not of the exp(-d/kT) form
    must give the oracle's decisions all the same -- a staircase (never increases: head in shared memory), one that fits
    shared memory whole, a random one (no bound: the kernel must fall back to the plain look-up), one that increases
    once far out in the tail, and one so short that every positive dE is beyond it."""
    lat, dims, n_sp, n_sh, w, seed = 1, (16, 16, 24), 5, 3, 4, 808
    epi = make_epi(n_sh, n_sp, 400, seed)
    rng = np.random.default_rng(12)
    if kind == "staircase":
        table = np.repeat(np.sort(rng.integers(0, 2 ** 32, 50, dtype=np.uint64))[::-1], 200).astype(np.uint32)   # 10,000 entries
    elif kind == "short":
        table = make_accept_table(860)[:3000].copy()        # ends at exp(-3.5): dE >= 3000 is always rejected
    elif kind == "non_monotone":
        table = rng.integers(0, 2 ** 32, 9000, dtype=np.uint64).astype(np.uint32)
    elif kind == "bump_in_the_tail":
        table = make_accept_table(860).copy()
        table[7000:7040] = 2 ** 31                          # beyond the resident head, far above T[K]
    else:
        table = make_accept_table(1)                        # 24 entries
    g = smcx.Lattice(lat, dims, n_sp, n_sh, epi, table, seed, link_cell=w, kT_units=860, kernel=smcx.KERNEL_FCC_THREAD)
    o = oracle.Oracle(lat, dims, n_sp, n_sh, epi, w, table, seed)
    g.sweep(3)
    o.sweep(3)
    _assert_same_state(g, o)
    assert (g.energy_trace() == o.energy_trace()).all() and g.stats() == o.stats()
    table2 = make_accept_table(1720)                        # and on to a regular long table on the same handles
    g.set_temperature(1720, table2)
    o.set_temperature(table2)
    g.sweep(2)
    o.sweep(2)
    _assert_same_state(g, o)
    assert (g.energy_trace() == o.energy_trace()).all() and g.stats() == o.stats() and g.stats()[2] > 0


def test_auto_picks_the_packed_kernels_from_12000_cells_per_colour():
    """AUTO's measured crossover (profiles/README.md): packed 4-bit kernels from 12,000 link cells per colour on, the
    sub-warp kernel below; 4-species BCC always a 2-bit thread kernel.  Results never depend on the choice (P14)."""
    def pick(lattice, edge, n_sp, n_sh):
        g = smcx.Lattice(lattice, (edge,) * 3, n_sp, n_sh, make_epi(n_sh, n_sp, 300, 3), make_accept_table(600), 3,
                         link_cell=4, kT_units=600)
        k, st = g.kernel, g.storage
        g.close()
        return k, st
    assert pick(smcx.FCC, 160, 5, 3) == (smcx.KERNEL_GROUP_PER_CELL, smcx.STORAGE_U8)        # 8,000 cells per colour
    assert pick(smcx.FCC, 192, 5, 3) == (smcx.KERNEL_FCC_THREAD, smcx.STORAGE_4BIT)          # 13,824
    assert pick(smcx.BCC, 160, 5, 2) == (smcx.KERNEL_GROUP_PER_CELL, smcx.STORAGE_U8)
    assert pick(smcx.BCC, 192, 5, 2) == (smcx.KERNEL_BCC4_THREAD, smcx.STORAGE_4BIT)
    assert pick(smcx.BCC, 192, 4, 2) == (smcx.KERNEL_THREAD_PER_CELL, smcx.STORAGE_2BIT)


def test_p14_four_bit_and_uint8_storage_agree():
    """P14: SMCX_STORAGE_4BIT (packed FCC kernel) and SMCX_STORAGE_U8 (sub-warp and warp kernels) give identical
    smcx_species, traces and pair counts, on the paper's composition with stage-wise cooling."""
    from smcx_inputs import composition_counts, cooling_stages
    lat, dims, n_sp, n_sh, w, seed = 1, (32, 16, 16), 5, 3, 4, 77
    epi = make_epi(n_sh, n_sp, 400, seed)
    stages = cooling_stages(1720, 860, 3)
    tables = [make_accept_table(k) for k in stages]
    hs = [smcx.Lattice(lat, dims, n_sp, n_sh, epi, tables[0], seed, link_cell=w, kT_units=stages[0], kernel=k)
          for k in (smcx.KERNEL_FCC_THREAD, smcx.KERNEL_GROUP_PER_CELL, smcx.KERNEL_WARP_PER_CELL)]
    assert [h.storage for h in hs] == [smcx.STORAGE_4BIT, smcx.STORAGE_U8, smcx.STORAGE_U8]
    counts = composition_counts(hs[0].n_sites, (29, 29, 28, 7, 7))
    for h in hs:
        h.init_composition(counts)
    for kT, tab in zip(stages, tables):
        for h in hs:
            h.set_temperature(kT, tab)
            h.sweep(3)
        for h in hs[1:]:
            assert (hs[0].species() == h.species()).all()
            assert (hs[0].sro()[1] == h.sro()[1]).all()
    for h in hs[1:]:
        assert (hs[0].energy_trace() == h.energy_trace()).all() and hs[0].stats() == h.stats()


@pytest.mark.parametrize("storage,lat,dims,n_sp,kernel", [
    (smcx.STORAGE_2BIT, 0, (16, 24, 16), 4, smcx.KERNEL_THREAD_PER_CELL),
    (smcx.STORAGE_4BIT, 1, (16, 16, 24), 7, smcx.KERNEL_FCC_THREAD),
    (smcx.STORAGE_U8, 1, (16, 16, 8), 5, smcx.KERNEL_GROUP_PER_CELL),
])
def test_packed_checkpoint_roundtrip(storage, lat, dims, n_sp, kernel):
    """smcx_species_packed / smcx_set_species_packed: the device storage format as a checkpoint (1/4, 1/2 or 1 byte per
    site); a new handle given the packed array and the sweep counter continues bit for bit; invalid fields are refused."""
    n_sh = 2 if lat == 0 else 3
    epi = make_epi(n_sh, n_sp, 300, 9)
    table = make_accept_table(600)
    kw = dict(link_cell=4, kT_units=600, kernel=kernel)
    a = smcx.Lattice(lat, dims, n_sp, n_sh, epi, table, 9, **kw)
    assert a.storage == storage
    assert a.storage_bytes() == a.n_sites * {2: 1, 4: 2, 8: 4}[storage] // 4
    a.sweep(3)
    packed, species, t = a.species_packed().copy(), a.species().copy(), a.stats()[0]
    a.sweep(2)
    b = smcx.Lattice(lat, dims, n_sp, n_sh, epi, table, 9, **kw)
    b.set_species_packed(packed)
    assert (b.species() == species).all() and b.energy() == b.running_energy()
    b.set_sweep_counter(t)
    b.sweep(2)
    assert (a.species() == b.species()).all() and (a.energy_trace(3, 2) == b.energy_trace(3, 2)).all()
    if storage != smcx.STORAGE_U8 and n_sp < (1 << storage):
        packed[5] = 0xFF                             # fields 15 / 3 >= n_species
        with pytest.raises(smcx.SmcxError) as ei:
            b.set_species_packed(packed)
        assert ei.value.code == -9
    # uint8 upload / download through the same storage
    rng = np.random.default_rng(1)
    s = rng.integers(0, n_sp, a.n_sites).astype(np.uint8)
    b.set_species(s)
    assert (b.species() == s).all() and (b.species_device().cpu().numpy() == s).all()
    s[11] = n_sp
    with pytest.raises(smcx.SmcxError):
        b.set_species(s)


def test_paper_shaped_fcc_full_size_invariants():
    """The lattice bench.py times as `paper_shaped_fcc` (FCC 640^3 = 1.05e9 sites, 29/29/28/7/7, three shells) in the launch
    configuration it is timed in (AUTO -> packed FCC kernel): conservation, energy bookkeeping, H = 1/2 sum V N; and the
    same build against the oracle on a 96 x 80 x 64 box (ragged batches: 12 * 10 * 8 / 8 = 120 cells per colour)."""
    from smcx_inputs import composition_counts
    epi, table = make_epi(3, 5, 400, 1006), make_accept_table(860)
    import bench
    edge = bench.PAPER_FCC_EDGE
    g = smcx.Lattice(smcx.FCC, (edge, edge, edge), 5, 3, epi, table, 1006, link_cell=4, kT_units=860)
    assert g.kernel == smcx.KERNEL_FCC_THREAD and g.storage == smcx.STORAGE_4BIT
    counts = composition_counts(g.n_sites, (29, 29, 28, 7, 7))
    g.init_composition(counts)
    _, c0 = g.sro()
    assert (c0[0].sum(axis=1) // 12 == np.array(counts)).all()
    assert g.energy() == g.running_energy()
    g.sweep(3)
    _, c1 = g.sro()
    assert (c1[0].sum(axis=1) // 12 == np.array(counts)).all() and (c1 == c1.transpose(0, 2, 1)).all()
    assert g.energy() == g.running_energy() == g.energy_trace()[-1]
    assert int((epi.astype(np.int64) * c1).sum()) == 2 * g.energy()
    assert 0 < g.stats()[2] < g.stats()[1]
    g.close()
    dims = (96, 80, 64)
    s = smcx.Lattice(smcx.FCC, dims, 5, 3, epi, table, 1006, link_cell=4, kT_units=860, kernel=smcx.KERNEL_FCC_THREAD)
    o = oracle.Oracle(smcx.FCC, dims, 5, 3, epi, 4, table, 1006, threads=ALL_CORES)
    cs = composition_counts(s.n_sites, (29, 29, 28, 7, 7))
    s.init_composition(cs)
    o.init_composition(cs)
    s.sweep(3)
    o.sweep(3)
    _assert_same_state(s, o)
    assert (s.energy_trace() == o.energy_trace()).all() and s.stats() == o.stats()


# ---- packed BCC kernel for up to 8 species (SMCX_KERNEL_BCC4_THREAD, SMCX_STORAGE_4BIT) ----------------------------
@pytest.mark.parametrize("dims,n_sp,n_sh,amp,kT", [
    ((16, 16, 16), 5, 2, 300, 600),       # five species: one more than the 2-bit kernels take
    ((24, 16, 8), 8, 2, 400, 860),        # most species the look-up takes, one cell per colour along z
    ((16, 8, 24), 6, 2, 300, 500),
    ((40, 24, 16), 5, 2, 15_000, 9_000),  # differences that need the high byte of the look-up in full
    ((32, 32, 32), 3, 2, 300, 430),       # more than one batch of 32 cells per colour; fewer species than 4 is fine too
    ((24, 24, 8), 7, 2, 300, 700),        # 9 cells per colour: a ragged batch
])
def test_packed_bcc4_kernel_against_the_oracle(dims, n_sp, n_sh, amp, kT):
    lat, w, seed = 0, 4, 616
    epi = make_epi(n_sh, n_sp, amp, seed)
    table = make_accept_table(kT)
    g = smcx.Lattice(lat, dims, n_sp, n_sh, epi, table, seed, link_cell=w, kT_units=kT, kernel=smcx.KERNEL_BCC4_THREAD)
    assert g.storage == smcx.STORAGE_4BIT and g.kernel == smcx.KERNEL_BCC4_THREAD
    o = oracle.Oracle(lat, dims, n_sp, n_sh, epi, w, table, seed)
    _assert_same_state(g, o)                       # S6 through Store4<2>
    assert g.energy() == o.energy() == g.running_energy()
    for _ in range(4):
        g.sweep(1)
        o.sweep(1)
        _assert_same_state(g, o)
    g.sweep(3)                                     # graph replay
    o.sweep(3)
    _assert_same_state(g, o)
    assert (g.energy_trace() == o.energy_trace()).all()
    assert g.stats() == o.stats() and g.stats()[2] > 0
    assert g.energy() == o.energy() == g.running_energy()
    _assert_sro(g, o)                              # pair counts on 4-bit BCC storage


def test_packed_bcc4_agrees_with_the_other_bcc_kernels_and_round_trips_checkpoints():
    """P14 on BCC: 4-bit storage (packed kernel), 2-bit storage (thread kernels) and uint8 (sub-warp kernel) walk the same
    trajectory with 4 species; the packed checkpoint of the 4-bit handle resumes bit for bit."""
    lat, dims, n_sp, n_sh, seed = 0, (32, 16, 24), 4, 2, 88
    epi = make_epi(n_sh, n_sp, 300, seed)
    table = make_accept_table(600)
    hs = [smcx.Lattice(lat, dims, n_sp, n_sh, epi, table, seed, link_cell=4, kT_units=600, kernel=k)
          for k in (smcx.KERNEL_BCC4_THREAD, smcx.KERNEL_THREAD_PERSISTENT, smcx.KERNEL_GROUP_PER_CELL)]
    assert [h.storage for h in hs] == [smcx.STORAGE_4BIT, smcx.STORAGE_2BIT, smcx.STORAGE_U8]
    for h in hs:
        h.sweep(5)
    for h in hs[1:]:
        assert (hs[0].species() == h.species()).all() and (hs[0].energy_trace() == h.energy_trace()).all()
        assert hs[0].stats() == h.stats() and (hs[0].sro()[1] == h.sro()[1]).all()
    a = hs[0]
    assert a.storage_bytes() == a.n_sites // 2
    packed, t = a.species_packed().copy(), a.stats()[0]
    a.sweep(2)
    b = smcx.Lattice(lat, dims, n_sp, n_sh, epi, table, seed, link_cell=4, kT_units=600, kernel=smcx.KERNEL_BCC4_THREAD)
    b.set_species_packed(packed)
    b.set_sweep_counter(t)
    b.sweep(2)
    assert (a.species() == b.species()).all()
