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


# ------------------------------------------------------------------ x-slab sharding: the exchange schedule (NEXT-2)

class _RecordingSlab:
    """Stand-in for a slab (the SlabOps interface of paper_2403_11156_b200/slabs.py) on CPU tensors: particles are
    points on a line that drift to the right by `dx` per step, no physics.  It CHECKS what the schedule promises:
    a ghost refresh delivers exactly the values of the particles that were sent as ghosts at the start of the step,
    in the same order (here the value of particle g is g itself); phases arrive in the documented order."""

    def __init__(self, x, gid, x_lo, x_hi, h, dx, iters):
        self.x, self.g = x.clone(), gid.clone()
        self.x_lo, self.x_hi, self.h, self.dx = x_lo, x_hi, h, dx
        self.iters = iters                     # (divergence, density) iterations the scripted error sums ask for
        self.phases, self.loops = [], []
        self.ghost_g = [None, None]
        self.sent = [None, None]
        self.it = {0: 0, 1: 0}
        self.mode = 0

    def template(self, what):
        return [((1,), torch.float32), ((), torch.int32)] if what in ("migrate", "ghosts") else [((1,), torch.float32)]

    def migrate_out(self):
        self.x = self.x + self.dx              # "integration" of the previous step
        left, right = self.x < self.x_lo, self.x >= self.x_hi
        out = []
        for m in (left, right):
            out.append((self.x[m].reshape(-1, 1).clone(), self.g[m].clone()) if m.any() else None)
        keep = ~(left | right)
        self.x, self.g = self.x[keep], self.g[keep]
        return out[0], out[1]

    def migrate_in(self, a, b):
        for pl in (a, b):
            if pl is not None and len(pl[0]):
                self.x = torch.cat([self.x, pl[0].reshape(-1)]); self.g = torch.cat([self.g, pl[1]])
        return len(self.x)

    def ghosts_out(self, has_left, has_right):
        out = []
        for d, (on, m) in enumerate(((has_left, self.x < self.x_lo + self.h), (has_right, self.x >= self.x_hi - self.h))):
            self.sent[d] = self.g[m].clone() if on else None
            out.append((self.x[m].reshape(-1, 1).clone(), self.g[m].clone()) if on else None)
        return out[0], out[1]

    def ghosts_in(self, a, b):
        for d, pl in enumerate((a, b)):
            self.ghost_g[d] = None if pl is None else pl[1].clone()
            if pl is not None and len(pl[0]):
                gx = pl[0].reshape(-1)
                assert ((gx < self.x_lo) if d == 0 else (gx >= self.x_hi)).all()          # ghosts lie across the cut ...
                assert ((gx >= self.x_lo - self.h) if d == 0 else (gx < self.x_hi + self.h)).all()   # ... within h of it

    def phase(self, ph):
        self.phases.append(ph)

    def refresh_out(self, field):
        return tuple(None if s is None else (s.to(torch.float32).reshape(-1, 1) + 1000.0 * field,) for s in self.sent)

    def refresh_in(self, field, a, b):
        for d, pl in enumerate((a, b)):
            if self.ghost_g[d] is None:
                assert pl is None
                continue
            assert torch.equal(pl[0].reshape(-1), self.ghost_g[d].to(torch.float32) + 1000.0 * field)

    def read_error_sum(self):
        # scripted: an error above every tolerance until the wanted iteration count is reached, then 0
        from paper_2403_11156_b200 import slabs
        want = self.iters[self.mode]
        self.it[self.mode] += 1
        return (len(self.x) << slabs.ACC_FRAC_BITS) if self.it[self.mode] < want else 0

    def set_loop(self, mode, cont, it, err):
        self.loops.append((mode, cont, it))
        if not cont:
            self.it[mode] = 0
            self.mode = 1 - mode               # divergence loop done -> density loop next, and back


def _slab_worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2403_11156_b200 import scenes, slabs
    n, h, dx = 400, 0.04, 0.013
    x_all = torch.linspace(0.0, 1.0, n)
    cut = 0.5
    lo, hi = (-3e38, cut) if rank == 0 else (cut, 3e38)
    mine = (x_all >= lo) & (x_all < hi)
    slab = _RecordingSlab(x_all[mine], torch.arange(n, dtype=torch.int32)[mine], lo, hi, h, dx, iters=(2, 3))
    prm = scenes.default_params(0.01, 4e-4)
    runner = slabs.SlabRunner([slab], slabs.DistExchange("cpu"), prm)
    steps = 6
    runner.run(steps)
    gathered = [None] * world
    dist.all_gather_object(gathered, dict(g=slab.g.tolist(), phases=slab.phases, loops=slab.loops, log=runner.log,
                                          stats=runner.stats, n_global=runner.n_global))
    if rank == 0:
        out.put(gathered)
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_slab_exchange_schedule_two_ranks_gloo():
    """Two ranks, one slab each, over gloo: particles migrate across the cut and every one stays owned by exactly one
    rank; ghost refreshes deliver the ghost layer's values in the order it was sent (checked inside the stand-in on
    both ranks); both ranks take the SAME loop decisions (one all-reduce per solver iteration) and run the passes in
    the order of DESIGN.md section 1, with a KR refresh after every P-pass and a VEL refresh after every C-pass that is
    followed by another pass."""
    from paper_2403_11156_b200 import slabs as S
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_slab_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    a, b = q.get(timeout=240)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert sorted(a["g"] + b["g"]) == list(range(400))                      # nobody lost, nobody duplicated
    assert len(b["g"]) > 200 and len(a["g"]) < 200                         # the drift moved particles across the cut
    assert a["n_global"] == b["n_global"] == 400
    assert a["loops"] == b["loops"] and a["phases"] == b["phases"] and a["log"] == b["log"]
    assert a["stats"]["total_it_v"] == 2 * 6 and a["stats"]["total_it_d"] == 3 * 6
    one_step = [S.PH_BEGIN, S.PH_DENSITY_DIVP, S.PH_C_DIV, S.PH_P_DIV, S.PH_C_DIV,
                S.PH_P_DENS_FIRST, S.PH_C_DENS, S.PH_P_DENS, S.PH_C_DENS, S.PH_P_DENS, S.PH_C_DENS, S.PH_END]
    assert a["phases"] == one_step * 6
    log = a["log"][: a["log"].index("step", 1)]
    assert log == ["step", "xchg:migrate", "allreduce", "xchg:ghosts", "phase:0",
                   "phase:1", "xchg:KR", "allreduce", "phase:2", "xchg:VEL",
                   "phase:3", "xchg:KR", "allreduce", "phase:2", "xchg:VEL",
                   "phase:5", "xchg:KR", "allreduce", "phase:7",
                   "xchg:VEL", "phase:6", "xchg:KR", "allreduce", "phase:7",
                   "xchg:VEL", "phase:6", "xchg:KR", "allreduce", "phase:7", "phase:8"]


def test_slab_schedule_local_exchange_three_slabs():
    """The same schedule with all slabs in one process (the one-device configuration of the GPU test): a middle slab
    talks to both neighbours."""
    from paper_2403_11156_b200 import scenes, slabs as S
    n, h, dx = 600, 0.04, -0.011
    x_all = torch.linspace(0.0, 1.0, n)
    cuts = [-3e38, 0.33, 0.66, 3e38]
    sl = []
    for k in range(3):
        m = (x_all >= cuts[k]) & (x_all < cuts[k + 1])
        sl.append(_RecordingSlab(x_all[m], torch.arange(n, dtype=torch.int32)[m], cuts[k], cuts[k + 1], h, dx, iters=(1, 2)))
    runner = S.SlabRunner(sl, S.LocalExchange(3), scenes.default_params(0.01, 4e-4))
    runner.run(8)
    assert sorted(sum((s.g.tolist() for s in sl), [])) == list(range(n))
    assert len(sl[0].g) > 200 and len(sl[2].g) < 200
    assert runner.stats["total_it_v"] == 8 and runner.stats["total_it_d"] == 16
