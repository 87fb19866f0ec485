"""Multi-GPU plumbing of bench.py on CPU: the path does not shard ("replicas only"), so
the only cross-rank logic is a barrier and the MAX of the per-rank times.  World size 2, gloo, 127.0.0.1."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, e2e = bench.max_over_ranks([10.0 + 5.0 * rank, 40.0 - 3.0 * rank], torch.device("cpu"), world)
    dist.barrier()
    if rank == 0:
        out.put((ms, e2e, bench.replica_value(1000 * 1000, 20, world, ms)))
    dist.destroy_process_group()


def test_replica_timing_is_max_over_ranks_and_value_is_aggregate():
    ctx = mp.get_context("spawn")
    out = ctx.SimpleQueue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    ms, e2e, value = out.get()
    assert ms == 15.0 and e2e == 40.0                     # slowest rank decides
    assert abs(value - 2 * 1e6 * 20 / 15e-3) < 1e-3       # whole-job aggregate over both replicas


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([3.0, 4.0], torch.device("cpu"), 1) == [3.0, 4.0]
    assert bench.replica_value(100, 2, 1, 1000.0) == 200.0
