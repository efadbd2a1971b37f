"""Connected slabs in separate PROCESSES (pytest -m gpu): one process per slab, as under torchrun with one process per
GPU, here all on the box's one GPU.  Each process exports its slab's storage with CUDA IPC, maps its neighbours', and
runs smcx_domain_sweep_connected: ghost layers are written by the sweep kernels straight into the neighbour process's
memory and signalled through flags the neighbour's stream waits for.  torch.distributed (gloo) only carries the IPC
handles and the final comparison; no kernel waits for another process's kernel (streams wait on memory values)."""
import os
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, kernel, q):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import torch
    import torch.distributed as dist
    import paper_2509_20949_b200 as smcx
    from smcx_inputs import make_accept_table, make_epi
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dims = (16, 16, 16 * world)
    kw = dict(lattice=smcx.BCC, dims=dims, n_species=4, n_shells=2, epi=make_epi(2, 4, 300, 71), accept=make_accept_table(700),
              seed=71, link_cell=4)
    slab = smcx.Domain(world, rank, kernel=kernel, library_workspace=True, **kw)
    handles = [None] * world
    dist.all_gather_object(handles, slab.ipc_export())
    slab.ipc_connect(handles[(rank - 1) % world], handles[(rank + 1) % world])
    dist.barrier()                                   # every slab is connected (flags zeroed) before any slab sweeps
    slab.sweep_connected(3)
    slab.sweep_connected(3)
    slab.synchronize()
    n_sites = dims[0] * dims[1] * dims[2] * 2
    part = np.zeros(n_sites, dtype=np.uint8)
    slab.species_into(part)
    parts = [None] * world
    dist.all_gather_object(parts, (part, slab.running_energy(), slab.energy_trace()))
    dist.barrier()                                   # nobody unmaps a neighbour that is still being written to
    slab.close()
    if rank == 0:
        whole = np.sum([p[0] for p in parts], axis=0).astype(np.uint8)   # owned layers are disjoint, the rest is 0
        q.put((whole, sum(p[1] for p in parts), np.sum([p[2] for p in parts], axis=0)))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,kernel", [(2, 3), (3, 3), (2, 4)], ids=["2-persistent", "3-persistent", "2-group"])
def test_slabs_in_separate_processes_over_cuda_ipc(world, kernel):
    import oracle
    from smcx_inputs import make_accept_table, make_epi
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 35500 + os.getpid() % 2000 + 7 * world + kernel
    procs = [ctx.Process(target=_worker, args=(r, world, port, kernel, q)) for r in range(world)]
    for p in procs:
        p.start()
    whole, e_run, trace = q.get(timeout=300)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    o = oracle.Oracle(0, (16, 16, 16 * world), 4, 2, make_epi(2, 4, 300, 71), 4, make_accept_table(700), 71)
    o.sweep(6)
    assert (whole == o.species()).all()
    assert e_run == o.running_energy() and (trace == o.energy_trace()).all()


def test_bench_slab_mode_under_torchrun_with_two_ranks_on_the_one_gpu():
    """`bench.py --gpus 2` as the driver launches it (torchrun, one rank per slab), both ranks on this box's one GPU and
    gloo instead of NCCL for the handles / reductions: the whole N > 1 path -- connected slabs over CUDA IPC, device-timed
    sweeps, end-to-end leg, the JSON line -- runs and reports the one lattice's throughput (strong scaling)."""
    import json
    import subprocess
    port = 36500 + os.getpid() % 2000
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--gpus", "2", "--config", "2", "--steps", "4",
           "--warmup", "3", "--dist-backend", "gloo"]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stdout[-2000:] + out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    d = json.loads(line)
    assert d["n_gpus"] == 2 and d["scaling"] == "strong" and d["value"] > 0 and d["e2e"]["value"] > 0
    assert "CUDA IPC" in d["config"]["parallelism"] and d["gpu_launches"] > 0
