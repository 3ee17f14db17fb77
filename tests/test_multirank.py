"""N > 1 is replicas only: every rank advances its own seeded scene, there is
no data-path collective, and bench.py reports units of all ranks / time of the slowest rank.
These tests run that host logic with world_size 2 over gloo on CPU."""
import os
import socket
import sys

import numpy as np
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
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_2403_11156_b200 import scenes
    assert bench.dist_env() == (rank, rank, world)
    sc = scenes.splash(n_target=2e4, seed=rank)          # what bench.py does: seed = rank
    ms_local = 10.0 + 5.0 * rank                          # rank 1 is the slow one
    ms_max = bench.max_over_ranks(ms_local, world, "cpu")
    value = bench.job_throughput(sc.n_fluid, 7, ms_max, world)
    digest = float(np.asarray(sc.boundary_pos, dtype=np.float64).sum())
    gathered = [None] * world
    dist.all_gather_object(gathered, (sc.n_fluid, digest, ms_max, value))
    if rank == 0:
        out.put(gathered)
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_replicas_time_is_max_over_ranks_and_value_is_whole_job():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = q.get(timeout=240)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (n0, d0, m0, v0), (n1, d1, m1, v1) = res
    assert m0 == m1 == 15.0                               # the slowest rank's time on every rank
    assert n0 == n1                                       # same workload size on every replica (weak scaling)
    assert d0 != d1                                       # ... but independently seeded obstacles
    assert v0 == v1 == pytest.approx(2 * n0 * 7 / 15.0e-3)


def test_single_rank_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(3.5, 1, "cpu") == 3.5
    assert bench.job_throughput(1000, 10, 2.0, 1) == pytest.approx(1000 * 10 / 2e-3)
