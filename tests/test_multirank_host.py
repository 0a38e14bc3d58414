"""Host-side logic of the N > 1 bench path on CPU (gloo, world_size 2): the path does not shard in this build
("replicas only"), so the only cross-rank steps are the barrier around the timed region, the
max-over-ranks of the per-rank device time and the aggregation of the replicas' throughput on rank 0."""
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
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms_local = 10.0 + 5.0 * rank                      # rank 1 is the slow replica
    ms = bench.max_over_ranks(ms_local, torch.device("cpu"))
    value = bench.aggregate_throughput(voxels=1000, steps=4, ms=ms, world=world)
    dist.barrier()
    if rank == 0:
        out.put((ms, value))
    dist.destroy_process_group()


def test_replica_aggregation_world_size_2():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    ms, value = out.get(timeout=120)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    assert ms == pytest.approx(15.0)                   # the max over ranks, not rank 0's own time
    assert value == pytest.approx(2 * 1000 * 4 / 15e-3 / 1e9)   # both replicas' voxel-iterations over that time


def test_single_rank_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(3.0, torch.device("cpu")) == 3.0
    assert bench.aggregate_throughput(voxels=10, steps=2, ms=1.0, world=1) == pytest.approx(10 * 2 / 1e-3 / 1e9)
