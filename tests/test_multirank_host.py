"""Host-side logic of the N > 1 path ("replicas only"): world_size-2 gloo run on CPU of the
rank->seed mapping and of the whole-job aggregation (units summed, time = max over ranks)."""
import os
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    local_ms = 10.0 * (rank + 1)            # rank 1 is the slow one
    units = 1000.0 * (rank + 1)
    value, max_ms = bench.aggregate_over_ranks(local_ms, units, dist, None)
    q.put((rank, value, max_ms, bench.replica_seed(1004, rank)))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_aggregation_and_seeds():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, value, max_ms, seed in res:
        assert max_ms == 20.0                          # max over ranks
        assert abs(value - 3000.0 / 0.020) < 1e-6      # whole-job units / slowest rank's time
    assert res[0][3] != res[1][3] and res[0][3] == 1004


def test_single_rank_aggregation_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    value, ms = bench.aggregate_over_ranks(5.0, 100.0)
    assert ms == 5.0 and abs(value - 20000.0) < 1e-9
