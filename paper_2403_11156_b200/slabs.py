"""x-slab domain decomposition of the DFSPH step across GPUs.

Host logic only: WHICH pass runs next, WHAT is exchanged with the x-neighbours and WHEN, and the loop predicates
(reading R14) evaluated once for the whole domain.  Every arithmetic step and every selection / gather / scatter runs
in the library's kernels (include/sph.h, "Slab mode"); transfers are torch copies (slabs of one device) or
torch.distributed send / recv + all-reduce (one slab per rank: NCCL over NVLink on GPUs, gloo in the CPU test of the
schedule).  The paper itself runs on one GPU.

Per step and slab (h = support radius, n_g = particles within h of a cut, ~n^(2/3) of the slab):
  migration      particles that crossed a cut:  36 B each  (pos4, vel4, id), with the x-neighbours
  ghost layers   36 B x n_g per side, once per step
  ghost refresh  16 B x n_g per side after EVERY pass that writes a field the next pass gathers:
                 KR after each P-pass (density / divergence), VEL after each C-pass and the viscosity kernel
                 -> 2 refreshes per solver iteration, 7 per step at the minimum iteration counts
  loop control   one 8-byte integer all-reduce per solver iteration (fixed-point error sums: the total does not depend
                 on the partition)
Config 4 cut into x-slabs: a 2 x 2 m face x h = 0.02 m holds ~40k particles -> 0.64 MB per refresh and side.

`SlabOps` is what the schedule needs from a slab; `GpuSlab` implements it on the C ABI.  `tests/test_multirank.py`
runs the same schedule on two gloo ranks with a recording stand-in.
"""
from __future__ import annotations

import ctypes as C
from typing import List, Optional, Sequence, Tuple

(PH_BEGIN, PH_DENSITY_DIVP, PH_C_DIV, PH_P_DIV, PH_VISCOSITY, PH_P_DENS_FIRST, PH_P_DENS, PH_C_DENS, PH_END) = range(9)
F_KR, F_VEL = 0, 1
ACC_FRAC_BITS = 20        # the library's fixed-point error sums: 2^-20 units (sph.h, sph_slab_read_error_sum)


# ------------------------------------------------------------------------------------------------ exchange back ends
class LocalExchange:
    """All slabs live in this process (one device): slab k's right neighbour is slab k + 1."""

    def __init__(self, n_slabs: int):
        self.n_local = n_slabs
        self.first = 0
        self.n_total = n_slabs

    def neighbor_exchange(self, to_left: List, to_right: List, template=None) -> Tuple[List, List]:
        n = self.n_local
        from_left = [to_right[k - 1] if k > 0 else None for k in range(n)]
        from_right = [to_left[k + 1] if k + 1 < n else None for k in range(n)]
        return from_left, from_right

    def allreduce_sum(self, value: int) -> int:
        return int(value)


class DistExchange:
    """One slab per rank of a torch.distributed process group (rank = slab index, neighbours rank +- 1)."""

    def __init__(self, device="cpu", group=None):
        import torch.distributed as dist
        self.dist = dist
        self.group = group
        self.rank = dist.get_rank(group)
        self.n_total = dist.get_world_size(group)
        self.n_local = 1
        self.first = self.rank
        self.device = device

    def _swap(self, payload, peer: Optional[int], tag_out: int, tag_in: int):
        """Send `payload` (tuple of tensors with equal leading length, or None) to `peer`, receive the peer's."""
        import torch
        if peer is None:
            return None
        dist = self.dist
        n_out = 0 if payload is None else int(payload[0].shape[0])
        cnt_out = torch.tensor([n_out], dtype=torch.int64, device=self.device)
        cnt_in = torch.zeros(1, dtype=torch.int64, device=self.device)
        reqs = [dist.isend(cnt_out, peer, group=self.group, tag=tag_out), dist.irecv(cnt_in, peer, group=self.group, tag=tag_in)]
        for r in reqs:
            r.wait()
        n_in = int(cnt_in.item())
        template = self._template
        recv = [torch.empty((n_in,) + shp, dtype=dt, device=self.device) for shp, dt in template]
        reqs = []
        if n_out:
            reqs += [dist.isend(t.contiguous(), peer, group=self.group, tag=tag_out) for t in payload]
        if n_in:
            reqs += [dist.irecv(t, peer, group=self.group, tag=tag_in) for t in recv]
        for r in reqs:
            r.wait()
        return tuple(recv)

    def neighbor_exchange(self, to_left: List, to_right: List, template=None) -> Tuple[List, List]:
        """template: [(trailing shape, dtype), ...] of the payload's tensors (a rank with nothing to send still has
        to allocate what it receives)."""
        left = self.rank - 1 if self.rank > 0 else None
        right = self.rank + 1 if self.rank + 1 < self.n_total else None
        self._template = list(template)
        # even ranks talk to the right first, odd ranks to the left first: no cyclic wait
        if self.rank % 2 == 0:
            fr = self._swap(to_right[0], right, 1, 2)
            fl = self._swap(to_left[0], left, 2, 1)
        else:
            fl = self._swap(to_left[0], left, 2, 1)
            fr = self._swap(to_right[0], right, 1, 2)
        return [fl], [fr]

    def allreduce_sum(self, value: int) -> int:
        import torch
        t = torch.tensor([int(value)], dtype=torch.int64, device=self.device)
        self.dist.all_reduce(t, group=self.group)
        return int(t.item())


# ------------------------------------------------------------------------------------------------ a slab on the C ABI
def _on_stream(fn):
    """Run a GpuSlab method with the simulation's stream as torch's current stream (copies and, for NCCL, the
    collectives are then ordered with the library's kernels)."""
    def wrapped(self, *a, **kw):
        with self.torch.cuda.stream(self.sim.stream):
            return fn(self, *a, **kw)
    wrapped.__name__ = fn.__name__
    wrapped.__doc__ = fn.__doc__
    return wrapped


class GpuSlab:
    """One x-slab as an ordinary library simulation (capacity-sized, host-driven launches) plus the buffers the
    schedule moves around.  Argument marshalling only: selection, gather and scatter are library kernels."""

    def __init__(self, scene, x_lo: float, x_hi: float, capacity: int, halo_capacity: int, device: int = 0, stream=None,
                 **overrides):
        import numpy as np
        import torch
        from . import binding as B
        self.B, self.torch = B, torch
        self.x_lo, self.x_hi = float(x_lo), float(x_hi)
        self.h = float(scene.params["support_radius"])
        self.cap, self.hcap = int(capacity), int(halo_capacity)
        dev = torch.device("cuda", device)
        self.dev = dev
        pos = np.asarray(scene.fluid_pos, dtype=np.float32)
        own = (pos[:, 0] >= self.x_lo) & (pos[:, 0] < self.x_hi)
        self.n_owned = int(own.sum())
        if self.n_owned > self.cap:
            raise ValueError("slab capacity too small")
        prm = dict(scene.params)
        prm.update(overrides)
        prm["use_cuda_graph"] = 0
        # the simulation is created at CAPACITY (its workspace is laid out for that many particles)
        # (placeholder positions: the slab's own particles repeated up to the capacity; replaced before the first step)
        fill_p = np.resize(pos[own] if self.n_owned else pos, (self.cap, 3)).astype(np.float32)
        self.sim = B.Sim(fill_p, np.zeros((self.cap, 3), dtype=np.float32), scene.boundary_pos, scene.boundary_body,
                         scene.bodies, prm, device=device, stream=stream)
        f32, i32 = torch.float32, torch.int32
        self.pos4 = torch.zeros((self.cap, 4), dtype=f32, device=dev)
        self.vel4 = torch.zeros((self.cap, 4), dtype=f32, device=dev)
        self.gid = [torch.zeros(self.cap, dtype=i32, device=dev), torch.zeros(self.cap, dtype=i32, device=dev)]
        self.cur = 0
        self.scratch = torch.zeros(self.cap + 64 + self.cap // 1024, dtype=i32, device=dev)
        self.side = [dict(pos=torch.zeros((self.hcap, 4), dtype=f32, device=dev), vel=torch.zeros((self.hcap, 4), dtype=f32, device=dev),
                          gid=torch.zeros(self.hcap, dtype=i32, device=dev), idx=torch.zeros(self.hcap, dtype=i32, device=dev),
                          buf=torch.zeros((self.hcap, 4), dtype=f32, device=dev), n=0) for _ in range(2)]
        self.ghost_first = [0, 0]
        self.ghost_n = [0, 0]
        n = self.n_owned
        ids = np.nonzero(own)[0].astype(np.int32)
        with torch.cuda.stream(self.sim.stream):
            self.pos4[:n, :3] = torch.as_tensor(pos[own], device=dev)
            self.vel4[:n, :3] = torch.as_tensor(np.asarray(scene.fluid_vel, dtype=np.float32)[own], device=dev)
            self.gid[0][:n] = torch.as_tensor(ids, device=dev)
        self.first_step = True

    # ---- selection helpers (library kernel sph_select_range)
    def _select(self, src_pos, src_vel, gid, key, key_lt, n, lo, hi, out_pos, out_vel, out_gid, out_idx, max_out):
        cnt = C.c_int(0)
        L = self.B.load()
        p = lambda t: C.c_void_p(t) if isinstance(t, int) else (C.c_void_p(t.data_ptr()) if t is not None else None)
        rc = L.sph_select_range(C.c_void_p(self.sim.stream.cuda_stream), p(src_pos), p(src_vel), p(gid), p(key), int(key_lt), int(n),
                                float(lo), float(hi), p(out_pos), p(out_vel), p(out_gid), p(out_idx), int(max_out),
                                p(self.scratch), self.scratch.numel(), C.byref(cnt))
        if rc != 0:
            raise self.B.SphError(rc, "sph_select_range")
        if cnt.value > max_out:
            raise RuntimeError("slab buffer too small: %d selected, room for %d" % (cnt.value, max_out))
        return int(cnt.value)

    # ---- SlabOps
    def template(self, what: str):
        """Tensors of a payload: particles (migrate / ghosts) = pos4, vel4, id; a field refresh = one float4 per ghost."""
        t = self.torch
        if what in ("migrate", "ghosts"):
            return [((4,), t.float32), ((4,), t.float32), ((), t.int32)]
        return [((4,), t.float32)]

    @_on_stream
    def migrate_out(self):
        """Split the owned particles of the last step's store into stay / to-left / to-right (deterministic order).
        Returns the two payloads (pos4, vel4, gid) for the neighbours; the stayers are already in the new buffers."""
        t = self.torch
        INF = 3.0e38
        new = 1 - self.cur
        if self.first_step:
            # nothing has moved yet: the initial partition is the owned set
            self.gid[new][:self.n_owned] = self.gid[self.cur][:self.n_owned]
            self.cur = new
            self.n_stay = self.n_owned
            return None, None
        sp, sv, sk, n, nown = self.sim.sph_slab_store()
        gsrc = self.gid[self.cur]
        self.n_stay = self._select(sp, sv, gsrc, sk, nown, n, self.x_lo, self.x_hi, self.pos4, self.vel4, self.gid[new], None, self.cap)
        out = []
        for d, (lo, hi) in enumerate(((-INF, self.x_lo), (self.x_hi, INF))):
            s = self.side[d]
            k = self._select(sp, sv, gsrc, sk, nown, n, lo, hi, s["pos"], s["vel"], s["gid"], None, self.hcap)
            out.append((s["pos"][:k].clone(), s["vel"][:k].clone(), s["gid"][:k].clone()) if k else None)
        self.cur = new
        return out[0], out[1]

    @_on_stream
    def migrate_in(self, from_left, from_right):
        n = self.n_stay
        for pl in (from_left, from_right):
            if pl is None or pl[0].shape[0] == 0:
                continue
            k = int(pl[0].shape[0])
            if n + k > self.cap:
                raise RuntimeError("slab capacity exceeded by migration")
            self.pos4[n:n + k] = pl[0]; self.vel4[n:n + k] = pl[1]; self.gid[self.cur][n:n + k] = pl[2]
            n += k
        self.n_owned = n
        return n

    @_on_stream
    def ghosts_out(self, has_left: bool, has_right: bool):
        """Ghost layers for the neighbours: owned particles within h of the cuts (their indices are kept for the refreshes)."""
        INF = 3.0e38
        out = []
        for d, (on, lo, hi) in enumerate(((has_left, -INF, self.x_lo + self.h), (has_right, self.x_hi - self.h, INF))):
            s = self.side[d]
            s["n"] = 0
            if not on:
                out.append(None)
                continue
            k = self._select(self.pos4, self.vel4, self.gid[self.cur], None, 0, self.n_owned, lo, hi, s["pos"], s["vel"], s["gid"], s["idx"], self.hcap)
            s["n"] = k
            out.append((s["pos"][:k].clone(), s["vel"][:k].clone(), s["gid"][:k].clone()))
        return out[0], out[1]

    @_on_stream
    def ghosts_in(self, from_left, from_right):
        n = self.n_owned
        for d, pl in enumerate((from_left, from_right)):
            k = 0 if pl is None else int(pl[0].shape[0])
            self.ghost_first[d], self.ghost_n[d] = n, k
            if k:
                if n + k > self.cap:
                    raise RuntimeError("slab capacity exceeded by ghosts")
                self.pos4[n:n + k] = pl[0]; self.vel4[n:n + k] = pl[1]; self.gid[self.cur][n:n + k] = pl[2]
                n += k
        self.n_total = n
        self.sim.sph_slab_set_particles(self.pos4, self.vel4, self.n_owned, n - self.n_owned)
        self.first_step = False

    def phase(self, ph: int):
        self.sim.sph_slab_phase(ph)

    @_on_stream
    def refresh_out(self, field: int):
        out = []
        for d, peer in enumerate((self.has_left, self.has_right)):
            s = self.side[d]
            if not peer:
                out.append(None)
                continue
            if s["n"]:
                self.sim.sph_slab_gather(field, s["idx"], s["n"], s["buf"])
            out.append((s["buf"][:s["n"]].clone(),))
        return out[0], out[1]

    @_on_stream
    def refresh_in(self, field: int, from_left, from_right):
        for d, pl in enumerate((from_left, from_right)):
            k = self.ghost_n[d]
            if k == 0:
                continue
            if pl is None or int(pl[0].shape[0]) != k:
                raise RuntimeError("ghost refresh does not match the ghost layer received at the start of the step")
            self.sim.sph_slab_scatter(field, self.ghost_first[d], k, pl[0].contiguous())

    def read_error_sum(self) -> int:
        return self.sim.sph_slab_read_error_sum()

    def set_loop(self, mode: int, cont: int, it: int, err: float):
        self.sim.sph_slab_set_loop(mode, cont, it, err)

    # ---- results (tests): owned particles of the store with their global ids
    @_on_stream
    def owned_state(self):
        import numpy as np
        t = self.torch
        sp, sv, sk, n, nown = self.sim.sph_slab_store()
        op = t.zeros((self.cap, 4), dtype=t.float32, device=self.dev)
        ov = t.zeros((self.cap, 4), dtype=t.float32, device=self.dev)
        og = t.zeros(self.cap, dtype=t.int32, device=self.dev)
        k = self._select(sp, sv, self.gid[self.cur], sk, nown, n, -3.0e38, 3.0e38, op, ov, og, None, self.cap)
        return og[:k].cpu().numpy(), op[:k, :3].cpu().numpy(), ov[:k, :3].cpu().numpy()

    def close(self):
        self.sim.close()


# ------------------------------------------------------------------------------------------------ the schedule
class SlabRunner:
    """The DFSPH step of sph_step_dfsph cut into x-slabs: same passes, same order, ghost refreshes
    and global loop decisions in between.  `slabs`: the local SlabOps objects (all of them for LocalExchange, one for
    DistExchange); `params`: the scene's parameter dictionary (loop limits and tolerances of reading R14)."""

    def __init__(self, slabs: Sequence, exchange, params):
        self.slabs = list(slabs)
        self.ex = exchange
        self.p = params
        self.log: List[str] = []          # what happened, in order (the schedule tests read it)
        for k, s in enumerate(self.slabs):
            s.has_left = exchange.first + k > 0
            s.has_right = exchange.first + k + 1 < exchange.n_total
        self.n_global = 0
        self.stats = dict(steps=0, total_it_v=0, total_it_d=0, it_v=0, it_d=0, err_v=0.0, err_rho=0.0)

    def _xchg(self, what, outs):
        self.log.append("xchg:" + what)
        fl, fr = self.ex.neighbor_exchange([o[0] for o in outs], [o[1] for o in outs], self.slabs[0].template(what))
        return list(zip(fl, fr))

    def _refresh(self, field):
        ins = self._xchg("KR" if field == F_KR else "VEL", [s.refresh_out(field) for s in self.slabs])
        for s, (a, b) in zip(self.slabs, ins):
            s.refresh_in(field, a, b)

    def _phase(self, ph):
        self.log.append("phase:%d" % ph)
        for s in self.slabs:
            s.phase(ph)

    def _decide(self, mode: int, first: bool, it_prev: int) -> Tuple[int, int]:
        """Reading R14 for the whole domain: the error measured by this iteration's P-pass decides whether another
        iteration follows its C-pass.  Returns (cont, iteration number)."""
        p = self.p
        total = self.ex.allreduce_sum(sum(s.read_error_sum() for s in self.slabs))
        self.log.append("allreduce")
        err = (total / float(1 << ACC_FRAC_BITS)) / max(self.n_global, 1)
        if mode == 0:
            on = bool(p["enable_divergence_solve"]) and p["max_iter_divergence"] > 0
            eta, mn, mx = p["eta_divergence"], p["min_iter_divergence"], p["max_iter_divergence"]
        else:
            on = p["max_iter_density"] > 0
            eta, mn, mx = p["eta_density"], p["min_iter_density"], p["max_iter_density"]
        if not on:
            cont, it, err = 0, 0, 0.0
        else:
            it = 1 if first else it_prev + 1
            forced = p["min_iter_divergence" if mode == 0 else "min_iter_density"] if p.get("force_iterations", 0) else -1
            cont = int(it < forced) if forced > 0 else int((err > eta or it < mn) and it < mx)
        for s in self.slabs:
            s.set_loop(mode, cont, it, err)
        key = ("it_v", "err_v") if mode == 0 else ("it_d", "err_rho")
        self.stats[key[0]], self.stats[key[1]] = it, err
        return cont, it

    def step(self):
        self.log.append("step")
        # 1. migration, then ghost layers (selected from the NEW owned sets)
        ins = self._xchg("migrate", [s.migrate_out() for s in self.slabs])
        owned = sum(s.migrate_in(a, b) for s, (a, b) in zip(self.slabs, ins))
        self.n_global = self.ex.allreduce_sum(owned)
        self.log.append("allreduce")
        ins = self._xchg("ghosts", [s.ghosts_out(s.has_left, s.has_right) for s in self.slabs])
        for s, (a, b) in zip(self.slabs, ins):
            s.ghosts_in(a, b)
        # 2. the passes of DESIGN.md section 1
        self._phase(PH_BEGIN)
        self._phase(PH_DENSITY_DIVP)
        self._refresh(F_KR)
        cont, it = self._decide(0, True, 0)
        self._phase(PH_C_DIV)
        self._refresh(F_VEL)
        while cont:
            self._phase(PH_P_DIV)
            self._refresh(F_KR)
            cont, it = self._decide(0, False, it)
            self._phase(PH_C_DIV)
            self._refresh(F_VEL)
        self.stats["total_it_v"] += it
        if self.p["viscosity_mode"] == 1:
            self._phase(PH_VISCOSITY)
            self._refresh(F_VEL)
        self._phase(PH_P_DENS_FIRST)
        self._refresh(F_KR)
        cont, it = self._decide(1, True, 0)
        self._phase(PH_C_DENS)
        while cont:
            self._refresh(F_VEL)
            self._phase(PH_P_DENS)
            self._refresh(F_KR)
            cont, it = self._decide(1, False, it)
            self._phase(PH_C_DENS)
        self.stats["total_it_d"] += it
        self._phase(PH_END)
        self.stats["steps"] += 1

    def run(self, n_steps: int):
        for _ in range(n_steps):
            self.step()


def make_local_slabs(scene, n_slabs: int, device: int = 0, slack: float = 1.6, fractions=None, **overrides):
    """n_slabs x-slabs of one scene on ONE device (test / development configuration): cuts at equal particle counts, or
    at the given cumulative particle fractions (n_slabs - 1 values)."""
    import numpy as np
    x = np.sort(np.asarray(scene.fluid_pos, dtype=np.float32)[:, 0])
    fr = [k / n_slabs for k in range(1, n_slabs)] if fractions is None else list(fractions)
    assert len(fr) == n_slabs - 1
    ux = np.unique(x)

    def cut_at(f):                         # between two distinct x values (a lattice plane is never cut in two)
        k = int(np.searchsorted(ux, x[min(int(len(x) * f), len(x) - 1)]))
        return float(0.5 * (ux[max(k - 1, 0)] + ux[k]))
    cuts = [-3.0e38] + [cut_at(f) for f in fr] + [3.0e38]
    import torch
    share = max(b - a for a, b in zip([0.0] + fr, fr + [1.0]))
    cap = int(len(x) * share * slack) + 4096
    stream = torch.cuda.Stream(torch.device("cuda", device))      # one stream for all slabs of the device: program order = data order
    slabs = [GpuSlab(scene, cuts[k], cuts[k + 1], cap, max(cap // 3, 4096), device=device, stream=stream, **overrides)
             for k in range(n_slabs)]
    return SlabRunner(slabs, LocalExchange(n_slabs), dict(scene.params, **overrides)), cuts
