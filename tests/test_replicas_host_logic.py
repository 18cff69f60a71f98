"""N > 1 in bench.py means N independent replicas of the product, one per GPU, with no data-path collective (DESIGN.md §8:
the product couples all particles through the global Stokes solve and does not shard).  The only cross-rank logic is the
seed of each replica and the max-over-ranks of the timed region; both are checked here with two gloo ranks on the CPU."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    import bench
    import workloads
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    try:
        ms_local = 100.0 + 7.0 * rank                       # rank 1 is the slower replica
        ms = bench.max_over_ranks(dist, ms_local, torch.device("cpu"))
        n = 4096
        prob, pos, F, T = workloads.monolayer_bw(n=n, seed=bench.replica_seed(1005, rank), name="replica")
        out.put((rank, ms, bench.whole_job_value(n, world, ms), float(pos[:, 0].sum()), prob.nx))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_replicas_max_time_and_distinct_particles():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    (r0, ms0, v0, sx0, nx0), (r1, ms1, v1, sx1, nx1) = res
    assert ms0 == ms1 == 107.0                                   # every rank sees the slowest rank's time
    assert v0 == v1 == pytest.approx(2 * 4096 / 0.107)           # whole-job particles/s of both replicas
    assert sx0 != sx1 and nx0 == nx1                             # same recipe and grid, different particles


def test_single_process_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(None, 3.5, None) == 3.5
    assert bench.replica_seed(1005, 0) == 1005
