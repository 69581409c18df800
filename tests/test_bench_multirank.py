"""The N > 1 path of bench.py on CPU: world_size 2, gloo.  The hot path does not shard on one GPU
(north_star fixes one GPU; replicas only), so the only multi-rank logic is
the max-over-ranks timing rule and the whole-job aggregation."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms = [10.0, 30.0][rank]          # rank 1 is the slow one
    e2e = [0.5, 0.2][rank]
    got = bench.max_over_ranks([ms, e2e])
    dist.barrier()
    out.put((rank, got, bench.aggregate_value(1000, 4, world, got[0])))
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_world2_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = [out.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, got, value in res:
        assert got == [30.0, 0.5]                                  # every rank sees the slowest time
        assert value == pytest.approx(1000 * 4 * 2 / 30.0e-3)      # units of all ranks / max time


def test_single_process_is_identity():
    import bench
    assert bench.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]
