"""Lattice parallelism on one GPU (pytest -m gpu): a lattice cut into slabs with ghost layers (reading S11,
PAPER.md:85, 147) must reproduce the undivided oracle bit for bit -- species, energy trace, statistics, pair counts.
All slabs live on the one device of the box; messages are device-to-device copies (smcx_domain_group_*) or tensor
copies driven by the per-rank driver (paper_2509_20949_b200.distributed with its in-process world)."""
import numpy as np
import pytest

import oracle
import paper_2509_20949_b200 as smcx
from paper_2509_20949_b200 import distributed
from smcx_inputs import composition_counts, get_config, make_accept_table, make_epi, scaled_config

pytestmark = pytest.mark.gpu


def _kw(lattice, dims, n_species, n_shells, seed, kT=700, amp=300):
    return dict(lattice=lattice, dims=dims, n_species=n_species, n_shells=n_shells,
                epi=make_epi(n_shells, n_species, amp, seed), accept=make_accept_table(kT), seed=seed, link_cell=4)


def _oracle(kw):
    return oracle.Oracle(kw["lattice"], kw["dims"], kw["n_species"], kw["n_shells"], kw["epi"], kw["link_cell"],
                         kw["accept"], kw["seed"])


def _assert_same(g, o):
    assert (g.species() == o.species()).all()
    assert (g.energy_trace() == o.energy_trace()).all()
    assert g.stats() == o.stats()
    assert g.energy() == o.energy() == g.running_energy() == o.running_energy()
    ga, gc = g.sro()
    oa, oc = o.sro()
    assert (gc == oc).all() and np.allclose(ga, oa, rtol=1e-9, atol=1e-9, equal_nan=True)


BCC_KERNELS = [(smcx.KERNEL_THREAD_PERSISTENT, "persistent"), (smcx.KERNEL_THREAD_PER_CELL, "thread"),
               (smcx.KERNEL_GROUP_PER_CELL, "group"), (smcx.KERNEL_WARP_PER_CELL, "warp")]


@pytest.mark.parametrize("kernel", [k for k, _ in BCC_KERNELS], ids=[n for _, n in BCC_KERNELS])
@pytest.mark.parametrize("n_slabs,overlap", [(2, 1), (4, 1), (4, 2), (4, 0)])   # 1: fused / overlapped, 2: overlapped copies, 0: plain
def test_bcc_slabs_against_the_undivided_oracle(kernel, n_slabs, overlap):
    kw = _kw(smcx.BCC, (16, 16, 32), 4, 2, seed=77)
    o = _oracle(kw)
    g = smcx.DomainGroup(n_slabs, kernel=kernel, overlap=overlap, **kw)
    assert (g.species() == o.species()).all()                     # S6 through the windows
    assert g.energy() == o.energy() == g.running_energy()
    for _ in range(7):                                           # origins 0..3 occur: the windows move both ways
        g.sweep(1)
        o.sweep(1)
        assert (g.species() == o.species()).all()
    _assert_same(g, o)
    assert g.message_bytes > 0 and g.kernel_launches > 0
    packed = kernel in (smcx.KERNEL_THREAD_PERSISTENT, smcx.KERNEL_THREAD_PER_CELL)
    assert (g.fused_messages > 0) == (packed and overlap == 1)    # the packed kernels write their pass messages themselves
    g.close()


@pytest.mark.parametrize("kernel,storage", [(smcx.KERNEL_FCC_THREAD, smcx.STORAGE_4BIT), (smcx.KERNEL_GROUP_PER_CELL, smcx.STORAGE_U8)],
                         ids=["fcc_thread", "group"])
@pytest.mark.parametrize("dims,n_slabs", [((8, 8, 16), 2), ((16, 8, 32), 4), ((8, 8, 40), 3)])
def test_fcc_five_species_slabs_against_the_undivided_oracle(kernel, storage, dims, n_slabs):
    kw = _kw(smcx.FCC, dims, 5, 3, seed=31, kT=690, amp=400)
    o = _oracle(kw)
    for overlap in (1, 2):
        g = smcx.DomainGroup(n_slabs, kernel=kernel, storage=storage, overlap=overlap, **kw)
        g.sweep(6)
        if overlap == 1:
            o.sweep(6)
        _assert_same(g, o)
        assert (g.fused_messages > 0) == (kernel == smcx.KERNEL_FCC_THREAD and overlap == 1)
        g.close()


def test_uneven_slabs_anneal_upload_and_resume():
    """5 row pairs over 3 slabs (2 + 2 + 1); a new temperature every sweep; an uploaded state; a resume."""
    kw = _kw(smcx.BCC, (8, 16, 40), 3, 2, seed=5)
    o = _oracle(kw)
    g = smcx.DomainGroup(3, **kw)
    assert [m.info["row_count"] for m in g.members] == [4, 4, 2] == [c for _, c in o.slab_partition(3)]
    rng = np.random.default_rng(1)
    state = rng.integers(0, 3, size=o.n_sites, dtype=np.uint8)
    g.set_species(state)
    o.set_species(state)
    for t in range(5):
        table = make_accept_table(900 - 100 * t)
        g.set_temperature(900 - 100 * t, table)
        o.set_temperature(table)
        g.sweep(1)
        o.sweep(1)
    _assert_same(g, o)
    # checkpoint = (species, sweep counter); a fresh group continues the run bit for bit
    saved, t = g.species().copy(), g.stats()[0]
    g2 = smcx.DomainGroup(3, **kw)
    g2.set_temperature(500, make_accept_table(500))
    g2.set_species(saved)
    g2.set_sweep_counter(t)
    g2.sweep(3)
    o.sweep(3)
    assert (g2.species() == o.species()).all()
    assert (g2.energy_trace(t) == o.energy_trace()[t:]).all()
    g.close()
    g2.close()


def test_paper_alloy_composition_on_slabs():
    kw = _kw(smcx.FCC, (8, 8, 32), 5, 3, seed=9, kT=860, amp=400)
    o = _oracle(kw)
    counts = composition_counts(o.n_sites, (29, 29, 28, 7, 7))
    o.init_composition(counts)
    g = smcx.DomainGroup(2, **kw)
    g.init_composition(counts)
    assert (g.species() == o.species()).all()
    g.sweep(4)
    o.sweep(4)
    _assert_same(g, o)
    g.close()


@pytest.mark.parametrize("overlap", [True, False])
def test_per_rank_driver_with_an_in_process_world(overlap):
    """paper_2509_20949_b200.distributed.SlabRank, the code a torchrun job runs, with its slabs in one process."""
    kw = _kw(smcx.BCC, (16, 16, 32), 4, 2, seed=21)
    o = _oracle(kw)
    world = distributed.LocalWorld(4)
    slabs = [distributed.SlabRank(r, 4, world=world, overlap=overlap, **kw) for r in range(4)]
    distributed.run_local(slabs, 6)
    o.sweep(6)
    whole = np.full(o.n_sites, 255, dtype=np.uint8)
    for s in slabs:
        s.domain.species_into(whole)
    assert (whole == o.species()).all()
    assert sum(s.domain.running_energy() for s in slabs) == o.running_energy()
    assert (sum(s.domain.energy_trace() for s in slabs) == o.energy_trace()).all()
    half = sum(s.domain.pair_counts() for s in slabs)
    alpha, counts = smcx.sro_from_counts(half, **{k: kw[k] for k in kw})
    oa, oc = o.sro()
    assert (counts == oc).all() and np.allclose(alpha, oa, rtol=1e-9, atol=1e-9)
    assert not world.mail                                       # every message posted was delivered
    for s in slabs:
        s.close()


def test_config4_shape_slabs_at_a_size_the_oracle_finishes():
    """BASELINE config 4's workload (4 species, 2 shells, kT 60 meV) on 104 x 88 x 96 cells cut into 3 slabs, with the
    kernel AUTO picks per slab; ragged grid (the cells of a colour do not fill the last batch)."""
    cfg = scaled_config(4, (104, 88, 96), n_sweeps=3)
    o = oracle.Oracle.from_config(cfg, threads=4)
    g = smcx.DomainGroup.from_config(cfg, 3)
    g.sweep(3)
    o.sweep(3)
    _assert_same(g, o)
    g.close()


@pytest.mark.parametrize("lattice,dims,n_sp,n_sh,n_slabs", [(smcx.BCC, (16, 16, 32), 4, 2, 2), (smcx.FCC, (16, 16, 48), 5, 3, 3)])
def test_local_energy_model_on_slabs(lattice, dims, n_sp, n_sh, n_slabs):
    """Reading S12 on slabs: three ghost layers, four-layer pass messages; against the undivided oracle."""
    from smcx_inputs import make_local_weights
    w1, w2 = make_local_weights(n_sh, n_sp, 200, 25, 19)
    table = make_accept_table(1500)
    o = oracle.Oracle(lattice, dims, n_sp, n_sh, w1, 4, table, 19)
    o.set_local_model(w2)
    g = smcx.DomainGroup(n_slabs, lattice, dims, n_sp, n_sh, w1, table, 19, link_cell=4, local_quad=w2)
    assert all(m.info["ghost"] == 3 for m in g.members)
    assert g.energy() == o.energy() == g.running_energy()
    for _ in range(5):
        g.sweep(1)
        o.sweep(1)
        assert (g.species() == o.species()).all()
    _assert_same(g, o)
    g.close()


@pytest.mark.parametrize("kernel", [smcx.KERNEL_THREAD_PERSISTENT, smcx.KERNEL_GROUP_PER_CELL], ids=["persistent", "group"])
def test_pass_split_boundary_row_and_the_rest_at_the_same_time(kernel):
    """smcx_domain_pass_split (what the per-rank NCCL driver calls): the boundary row on a side stream, the other rows on
    the slab's stream, concurrently; messages moved by hand between three slabs."""
    import torch
    kw = _kw(smcx.BCC, (16, 16, 48), 4, 2, seed=33)
    o = _oracle(kw)
    slabs = [smcx.Domain(3, r, kernel=kernel, **kw) for r in range(3)]
    side = [torch.cuda.Stream() for _ in slabs]

    def move(plans):
        torch.cuda.synchronize()
        for r, (send, _) in enumerate(plans):
            if send[3]:
                dst = slabs[send[0]]
                recv = plans[send[0]][1]
                assert recv[0] == r and recv[3] == send[3]
                dst.storage_view(recv).copy_(slabs[r].storage_view(send))
        torch.cuda.synchronize()

    for _ in range(5):
        move([s.begin_sweep() for s in slabs])
        for colour in range(8):
            plans = [s.pass_messages(colour) for s in slabs]
            for s, st in zip(slabs, side):
                s.run_pass_split(colour, st)
            move(plans)
        for s in slabs:
            s.end_sweep()
    o.sweep(5)
    whole = np.full(o.n_sites, 255, dtype=np.uint8)
    for s in slabs:
        s.species_into(whole)
    assert (whole == o.species()).all()
    assert sum(s.running_energy() for s in slabs) == o.running_energy()
    for s in slabs:
        s.close()


@pytest.mark.parametrize("kernel,n_slabs", [(smcx.KERNEL_THREAD_PERSISTENT, 3), (smcx.KERNEL_GROUP_PER_CELL, 2)], ids=["persistent3", "group2"])
def test_connected_slabs_in_one_process(kernel, n_slabs):
    """smcx_domain_connect + smcx_domain_sweep_connected: every slab pushes its messages into its neighbours' storage and
    signals them through a flag the neighbour's stream waits for; no host code between the passes.  The slabs live in
    this process here (each on its own stream); tests/test_gpu_ipc_slabs.py runs them in separate processes."""
    import torch
    kw = _kw(smcx.BCC, (16, 16, 16 * n_slabs), 4, 2, seed=61)
    o = _oracle(kw)
    streams = [torch.cuda.Stream() for _ in range(n_slabs)]
    slabs = [smcx.Domain(n_slabs, r, kernel=kernel, stream=streams[r], **kw) for r in range(n_slabs)]
    for r, s in enumerate(slabs):
        s.connect(slabs[(r - 1) % n_slabs], slabs[(r + 1) % n_slabs])
    for n in (1, 4, 2):
        for s in slabs:
            s.sweep_connected(n)          # every call only enqueues: the slabs' streams sort the order out
    torch.cuda.synchronize()
    o.sweep(7)
    whole = np.full(o.n_sites, 255, dtype=np.uint8)
    for s in slabs:
        s.species_into(whole)
    assert (whole == o.species()).all()
    assert sum(s.running_energy() for s in slabs) == o.running_energy()
    assert (sum(s.energy_trace() for s in slabs) == o.energy_trace()).all()
    for s in slabs:
        s.close()


def test_connected_slabs_fcc_packed_and_local_model():
    """Connected slabs with the packed FCC kernel (messages fused into its write-back) and with the local-energy model
    (three ghost layers, messages copied), three slabs each, stepped in turns."""
    import torch
    from smcx_inputs import make_local_weights
    cases = []
    kw = _kw(smcx.FCC, (16, 16, 48), 5, 3, seed=83, kT=690, amp=400)
    cases.append((kw, dict(kernel=smcx.KERNEL_FCC_THREAD, storage=smcx.STORAGE_4BIT), None))
    w1, w2 = make_local_weights(2, 4, 200, 25, 29)
    kwl = dict(lattice=smcx.BCC, dims=(16, 16, 48), n_species=4, n_shells=2, epi=w1, accept=make_accept_table(1200), seed=29, link_cell=4)
    cases.append((kwl, dict(local_quad=w2), w2))
    for kw, extra, quad in cases:
        o = _oracle(kw)
        if quad is not None:
            o.set_local_model(quad)
        streams = [torch.cuda.Stream() for _ in range(3)]
        slabs = [smcx.Domain(3, r, stream=streams[r], **extra, **kw) for r in range(3)]
        for r, s in enumerate(slabs):
            s.connect(slabs[(r - 1) % 3], slabs[(r + 1) % 3])
        for _ in range(5):
            for s in slabs:
                s.sweep_connected(1)
        torch.cuda.synchronize()
        o.sweep(5)
        whole = np.full(o.n_sites, 255, dtype=np.uint8)
        for s in slabs:
            s.species_into(whole)
        assert (whole == o.species()).all()
        assert sum(s.running_energy() for s in slabs) == o.running_energy()
        for s in slabs:
            s.close()


def test_a_fourth_connected_slab_in_one_process_is_refused():
    """Streams that wait for a flag must not share a hardware work queue with the stream that sets it; with the default
    8 queues that allows three connected slabs (two streams each) per process -- the fourth is refused, not deadlocked."""
    kw = _kw(smcx.BCC, (16, 16, 64), 4, 2, seed=3)
    slabs = [smcx.Domain(4, r, **kw) for r in range(4)]
    for r in range(3):
        slabs[r].connect(slabs[(r - 1) % 4], slabs[(r + 1) % 4])
    with pytest.raises(smcx.SmcxError) as ei:
        slabs[3].connect(slabs[2], slabs[0])
    assert ei.value.code == -12
    for s in slabs:
        s.close()
    again = [smcx.Domain(2, r, **kw) for r in range(2)]          # closing gave the places back
    for r in range(2):
        again[r].connect(again[1 - r], again[1 - r])
    for s in again:
        s.close()


def test_packed_bcc4_kernel_on_slabs_with_fused_messages():
    """Five species on BCC (4-bit storage, SMCX_KERNEL_BCC4_THREAD) cut into 2 and 3 slabs; the kernel's write-back carries
    the pass messages."""
    kw = _kw(smcx.BCC, (16, 16, 48), 5, 2, seed=47)
    o = _oracle(kw)
    o.sweep(6)
    for n_slabs in (2, 3):
        g = smcx.DomainGroup(n_slabs, kernel=smcx.KERNEL_BCC4_THREAD, **kw)
        g.sweep(6)
        _assert_same(g, o)
        assert g.fused_messages > 0
        g.close()
