"""Host-side logic of lattice parallelism that needs no GPU: the slab partition and message plan of the C ABI
(smcx_domain_partition / smcx_domain_plan_messages) against the oracle's statement of the protocol (reading S11),
and a world_size-2 gloo run of the per-rank transport (paper_2509_20949_b200.distributed.exchange)."""
import os
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

import oracle
import paper_2509_20949_b200 as smcx
from smcx_inputs import make_accept_table, make_epi

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _kw(dims=(16, 16, 40), lattice=0, n_species=4, n_shells=2, seed=5):
    return dict(lattice=lattice, dims=dims, n_species=n_species, n_shells=n_shells, epi=make_epi(n_shells, n_species, 300, 1),
                accept=make_accept_table(600), seed=seed, link_cell=4)


def test_partition_matches_the_oracles_and_covers_the_lattice():
    kw = _kw()
    o = oracle.Oracle(kw["lattice"], kw["dims"], 4, 2, kw["epi"], 4, kw["accept"], kw["seed"], init=False)
    for d in (2, 3, 5):
        infos = [smcx.domain_partition(d, k, **kw) for k in range(d)]
        assert [(i["row_first"], i["row_count"]) for i in infos] == o.slab_partition(d)
        for k, i in enumerate(infos):
            assert i["lower"] == (k - 1) % d and i["upper"] == (k + 1) % d
            assert i["z_layers"] == i["row_count"] * 4 + 3 + 2 * i["ghost"] and i["ghost"] == 2
            assert i["z_base"] == (i["row_first"] * 4 - 2) % kw["dims"][2]
            assert i["owned_sites"] == i["row_count"] * 4 * 16 * 16 * 2
        assert sum(i["owned_sites"] for i in infos) == 16 * 16 * 40 * 2
    with pytest.raises(smcx.SmcxError):
        smcx.domain_partition(6, 0, **kw)            # 5 pairs of rows only
    with pytest.raises(smcx.SmcxError):
        smcx.domain_partition(2, 2, **kw)


def _layers(msg, layer_bytes):
    peer, tag, off, nbytes = msg
    assert off % layer_bytes == 0 and nbytes % layer_bytes == 0
    return list(range(off // layer_bytes, (off + nbytes) // layer_bytes))


@pytest.mark.parametrize("n_slabs", [2, 3, 5])
def test_message_plan_pairs_up_and_names_the_layers_of_reading_s11(n_slabs):
    kw = _kw()
    Lz = kw["dims"][2]
    o = oracle.Oracle(kw["lattice"], kw["dims"], 4, 2, kw["epi"], 4, kw["accept"], kw["seed"], init=False)
    infos = [smcx.domain_partition(n_slabs, k, **kw) for k in range(n_slabs)]
    lb = infos[0]["layer_bytes"]
    moved = False
    for sweep in range(6):
        oz, oz_prev = o.shift(sweep)[2], (o.shift(sweep - 1)[2] if sweep else 0)
        for phase in range(-1, 8):
            plans = [smcx.domain_plan_messages(n_slabs, k, sweep, phase, **kw) for k in range(n_slabs)]
            for k, (send, recv) in enumerate(plans):
                if send[3] == 0:
                    assert phase == -1 and recv[3] == 0 and (sweep == 0 or oz == oz_prev)
                    continue
                peer = send[0]
                peer_recv = plans[peer][1]
                assert peer_recv[0] == k and peer_recv[1] == send[1] and peer_recv[3] == send[3]
                # the same layers of the whole lattice on both sides
                mine = [(infos[k]["z_base"] + l) % Lz for l in _layers(send, lb)]
                theirs = [(infos[peer]["z_base"] + l) % Lz for l in _layers(peer_recv, lb)]
                assert mine == theirs
                a = oz + infos[k]["row_first"] * 4
                b = a + infos[k]["row_count"] * 4
                if phase == -1:
                    moved = True
                    a_old = oz_prev + infos[k]["row_first"] * 4
                    want = range(a_old + 2, a_old + 2 + (oz - oz_prev)) if oz > oz_prev else range(b - 2, b - 2 + (oz_prev - oz))
                    assert peer == (infos[k]["lower"] if oz > oz_prev else infos[k]["upper"])
                elif (phase >> 2) & 1 == 0:
                    want, expect_peer = range(a - 1, a + 2), infos[k]["lower"]
                    assert peer == expect_peer
                else:
                    want, expect_peer = range(b - 2, b + 1), infos[k]["upper"]
                    assert peer == expect_peer
                assert mine == [z % Lz for z in want]
                for l in _layers(send, lb) + _layers(plans[k][1], lb):
                    assert 0 <= l < infos[k]["z_layers"]
    assert moved


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_2509_20949_b200 import distributed
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    kw = _kw(dims=(16, 16, 32))
    info = smcx.domain_partition(world, rank, **kw)
    lb = info["layer_bytes"]
    # a host stand-in for the slab's species storage: every byte names (rank, storage layer)
    store = torch.zeros(info["z_layers"] * lb, dtype=torch.uint8)
    ok = True
    for sweep in range(4):
        for phase in range(-1, 8):
            for l in range(info["z_layers"]):
                store[l * lb:(l + 1) * lb] = 16 * rank + (l % 16)
            send, recv = smcx.domain_plan_messages(world, rank, sweep, phase, **kw)
            for work in distributed.exchange(dist, rank, store, send, recv):
                work.wait()
            if recv[3]:
                peer_info = smcx.domain_partition(world, recv[0], **kw)
                got = store[recv[2]: recv[2] + recv[3]].view(-1, lb)[:, 0].tolist()
                mine = [(info["z_base"] + l) % 32 for l in range(recv[2] // lb, (recv[2] + recv[3]) // lb)]
                want = [16 * recv[0] + ((z - peer_info["z_base"]) % 32) % 16 for z in mine]
                ok = ok and got == want
    q.put((rank, ok))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo_exchange_moves_the_planned_layers():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == [(0, True), (1, True)]


class _HostSlab:
    """Stand-in for binding.Domain with the same stepping calls, its species storage a CPU tensor: a "pass" stamps the
    layers of its outgoing message with (sweep, phase, rank), so that the receiver can tell whether the driver moved the
    right bytes at the right time.  The message plan is the library's own (smcx_domain_plan_messages, host arithmetic)."""

    def __init__(self, world, rank, kw):
        import torch
        self.world, self.rank, self.kw = world, rank, kw
        self.info = smcx.domain_partition(world, rank, **kw)
        self.lb = self.info["layer_bytes"]
        self._storage_view = torch.zeros(self.info["z_layers"] * self.lb, dtype=torch.uint8)
        self.sweep, self.log = 0, []

    def _stamp(self, phase):
        send, _ = smcx.domain_plan_messages(self.world, self.rank, self.sweep, phase, **self.kw)
        if send[3]:
            self._storage_view[send[2]: send[2] + send[3]] = (7 * self.sweep + 3 * (phase + 1) + 11 * self.rank) % 251

    def begin_sweep(self):
        self._stamp(-1)
        return smcx.domain_plan_messages(self.world, self.rank, self.sweep, -1, **self.kw)

    def pass_messages(self, colour):
        return smcx.domain_plan_messages(self.world, self.rank, self.sweep, colour, **self.kw)

    def run_pass(self, colour, part=0):
        self.log.append((self.sweep, colour, part))
        if part in (0, 1):
            self._stamp(colour)

    def check(self, phase):
        _, recv = smcx.domain_plan_messages(self.world, self.rank, self.sweep, phase, **self.kw)
        if not recv[3]:
            return True
        want = (7 * self.sweep + 3 * (phase + 1) + 11 * recv[0]) % 251
        return bool((self._storage_view[recv[2]: recv[2] + recv[3]] == want).all())

    def end_sweep(self):
        self.sweep += 1


def _driver_worker(rank, world, port, overlap, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_2509_20949_b200 import distributed
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    kw = _kw(dims=(16, 16, 32))
    slab = _HostSlab(world, rank, kw)
    drv = distributed.SlabRank(rank, world, dist=dist, overlap=overlap, domain=slab)
    ok = True
    for _ in range(5):                       # SlabRank.sweep, with a check after every phase
        drv.phase_end(drv.sweep_begin())
        ok = ok and slab.check(-1)
        for colour in range(8):
            drv.phase_end(drv.pass_begin(colour))
            ok = ok and slab.check(colour)
        drv.sweep_end()
    parts = sorted({p for _, _, p in slab.log})
    q.put((rank, ok, parts, drv.message_bytes > 0))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("overlap", [True, False])
def test_two_rank_gloo_run_of_the_per_rank_driver(overlap):
    """paper_2509_20949_b200.distributed.SlabRank -- the loop a torchrun job runs -- over gloo with a host stand-in for
    the slab: every phase of five sweeps delivers the neighbour's stamped layers, with and without overlap."""
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 33500 + os.getpid() % 2000 + (1 if overlap else 0)
    procs = [ctx.Process(target=_driver_worker, args=(r, 2, port, overlap, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    want_parts = [1, 2] if overlap else [0]
    assert res == [(0, True, want_parts, True), (1, True, want_parts, True)]
