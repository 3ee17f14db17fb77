#!/usr/bin/env python
"""bench.py -- DFSPH particle-steps/s on BASELINE.json's headline workload (config 4: 1.23M fluid
particles, two blocks colliding against four static obstacles in a 4x2x2 m tank), one B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A "step" is one pass of the whole hot path: grid build, density +
alpha + neighbour lists, divergence-free solve, gravity, constant-density solve, integration.
Prints ONE JSON line (rank 0).  N > 1: independent replicas, one per GPU (the path has no
exchange step in this version: DESIGN.md section 8), reported as weak scaling.

--impl reference times the fp64 CPU oracle (oracle/), as it stands, on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "DFSPH particle-steps/sec at 1.23M particles (1 B200); achieved HBM GB/s vs peak"
UNIT = "particle-steps/s"
FP32_LANES_PER_SM = 128
N_SM = 148


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(", ") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            if len(r) < 9:
                continue
            try:
                sm.append(float(r[1])); smax.append(float(r[2]))
            except ValueError:
                continue
            for nm, v in zip(names, r[5:9]):
                if v.strip().lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return dict(sm_mhz=(sm[len(sm) // 2] if sm else None), sm_max_mhz=(max(smax) if smax else None),
                    reasons=sorted(reasons), samples=len(sm))


def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


# ---------------------------------------------------------------------------------------------
# Algorithmic work per fluid particle of each kernel.
#  bytes_8d   : SURVEY.md section 8(d) "compulsory HBM bytes" of the row(s) the kernel realises (own inputs read
#               once + outputs written once, neighbours cache-served): A4 24 B, P-pass 44 B, C-pass 52 B, A9 40 B,
#               A1-A3 ~110 B + ~10 B per cell.  The headline roofline.frac uses THIS figure.
#  bytes_lists: the same plus what this design adds on top of 8(d): the per-step neighbour list (2 B per fluid,
#               4 B per boundary neighbour) and the packed count word -- real traffic, but the design's own choice.
#  nf / nbd = mean fluid / boundary neighbours, cand = mean candidates tested by the list builder.
def kernel_work(name, nf_mean, nb_mean, cand_mean, cells_per_particle=0.0):
    lst = 2.0 * nf_mean + 4.0 * nb_mean
    nn = nf_mean + nb_mean
    if name == "k_build_lists":        # first half of A4: pos in (16); lists + count out are the design's own stream
        return dict(bytes_8d=16.0, bytes_lists=16 + 4 + lst, flops=8.0 * cand_mean, row="A4 (list build)")
    if name == "k_density_alpha":      # A4 (pos -> rho, alpha) fused with the first P-pass of A5 (vel in, kappa/rho out)
        return dict(bytes_8d=44.0, bytes_lists=32 + 4 + lst + 4 + 4 + 16, flops=45.0 * nn + 25, row="A4 + first A5 P")
    if name == "k_solver_p":
        return dict(bytes_8d=44.0, bytes_lists=32 + 4 + 4 + lst + 16, flops=27.0 * nn + 12, row="A5/A7 P")
    if name == "k_solver_c":           # one launch in three also integrates (A9, 40 B)
        return dict(bytes_8d=52.0 + 40.0 / 3.0, bytes_lists=16 + 4 + lst + 16 + 16 + (4 + 36) / 3.0, flops=26.0 * nn + 12,
                    row="A5/A7 C (+A6, A9)")
    if name in ("k_reorder", "k_sort_scatter"):
        return dict(bytes_8d=80.0, bytes_lists=4 + 4 + 8 + 36 + 16 + 32 + 4, flops=0.0, row="A3")
    if name == "k_cell_key_hist":
        return dict(bytes_8d=30.0, bytes_lists=16 + 4 + 4 + 8, flops=10.0, row="A1")
    return None


def step_bytes_8d(mean_it_v, mean_it_d, cells_per_particle):
    """SURVEY 8(d) compulsory bytes of one whole DFSPH step per fluid particle (viscosity off): grid A1-A3
    (~110 B + ~10 B per cell), A4 24, P 44 and C 52 per solver iteration, A9 40."""
    return 110.0 + 10.0 * cells_per_particle + 24.0 + (mean_it_v + mean_it_d) * (44.0 + 52.0) + 40.0


def csrc_sha16():
    """Hash of the kernel sources: an ncu profile names the sources it was captured from."""
    import glob
    import hashlib
    h = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(ROOT, "paper_2403_11156_b200", "csrc", "*.cu*"))):
        h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


NCU_PROFILE = "profiles/r2_ncu_full_summary.md"


def read_ncu_profile(path=None):
    """Parse the committed `ncu --set full` summary (a markdown table: one column per profiled launch, one row per
    metric; a `csrc_sha16:` line names the kernel sources it was captured from).
    Returns {kernel name: {metric: float}}, sha or None."""
    path = os.path.join(ROOT, path or NCU_PROFILE)
    if not os.path.exists(path):
        return {}, None
    sha, cols, out = None, None, {}
    for line in open(path):
        if line.startswith("csrc_sha16:"):
            sha = line.split(":", 1)[1].strip().strip("`")
        if not line.startswith("|"):
            continue
        cells = [c.strip() for c in line.strip().strip("|").split("|")]
        if cells[0] == "metric":
            cols = cells[2:]
            for c in cols:
                out.setdefault(c, {})
        elif cols and not set(cells[0]) <= set("-") and len(cells) >= 2 + len(cols):
            for c, v in zip(cols, cells[2:]):
                try:
                    out[c][cells[0]] = float(v.replace(",", ""))
                except ValueError:
                    pass
    return out, sha


def ncu_for_kernel(prof, name):
    for col, m in prof.items():
        if name in col:
            return m
    return None


FINE_X = 2      # the library splits every grid cell into 2 slabs along x: x-runs cover 2.5 of the 3 cell widths


def max_over_ranks(ms_local, world, device):
    """Replicas-only multi-GPU: the job's time is the slowest rank's."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(n_units_per_rank, steps, ms_max, world):
    """Whole-job particle-steps/s: every rank advanced its own replica by `steps` steps in ms_max."""
    return world * n_units_per_rank * steps / (ms_max * 1e-3)


def run_ours(args):
    import torch
    import torch.distributed as dist
    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    from paper_2403_11156_b200 import binding as B, build, scenes
    build.build()
    B.load()
    peaks = load_peaks()

    if args.n_target:
        # scaling sweep of BASELINE.json configs[4]: the config-4 scene with every site count scaled
        sc = scenes.splash(n_target=args.n_target, seed=rank, name="config4_splash_sweep_%.3gM" % (args.n_target / 1e6))
    else:
        sc = scenes.config(args.config, seed=rank)
    if args.warm_start:
        sc.params.update(warm_start=1, warm_start_factor=0.5)
    if args.eta_density:
        sc.params["eta_density"] = args.eta_density
    K, W = args.steps, args.warmup
    sim = B.Sim.from_scene(sc, device=local_rank, use_cuda_graph=0 if args.no_graph else 1)
    stream = sim.stream
    step_of = lambda s_: {"dfsph": s_.sph_step_dfsph, "pcisph": s_.sph_step_pcisph, "wcsph": s_.sph_step_wcsph}[args.method]
    sim_step = step_of(sim)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident throughput: W warm-up steps, then exactly K timed steps
    sim_step(W)
    launches0 = sim.sph_launch_count()
    st0 = sim.sph_read_stats()
    clocks = ClockSampler(local_rank)
    barrier()
    clocks.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    sim_step(K)
    e1.record(stream)
    stream.synchronize()
    barrier()
    ck = clocks.stop()
    ms = e0.elapsed_time(e1)
    st1 = sim.sph_read_stats()
    launches = sim.sph_launch_count() - launches0
    ms_max = max_over_ranks(ms, world, "cuda")
    nf = sc.n_fluid
    value = job_throughput(nf, K, ms_max, world)
    mean_it_v = (st1["total_it_v"] - st0["total_it_v"]) / max(K, 1)
    mean_it_d = (st1["total_it_d"] - st0["total_it_d"]) / max(K, 1)

    # ---- end to end through the C ABI with HOST buffers: every step reads the new positions and velocities back into
    # pinned host memory and uploads them again as the next step's inputs (asynchronous host copies, is_host = 2:
    # the upload of the positions runs beside the download of the velocities -- PCIe is full duplex; every byte still
    # crosses the bus inside the timed region, and every upload waits for the download that fills its buffer)
    Ke = max(1, min(K, args.e2e_steps))
    ph = torch.empty((nf, 3), dtype=torch.float32).pin_memory()
    vh = torch.empty((nf, 3), dtype=torch.float32).pin_memory()
    sim.sph_read_state_host(B.POS, ph); sim.sph_read_state_host(B.VEL, vh)

    def e2e_step():
        sim_step(1)
        sim.sph_read_state_host_async(B.POS, ph)
        sim.sph_write_state_host_async(B.POS, ph)
        sim.sph_read_state_host_async(B.VEL, vh)
        sim.sph_write_state_host_async(B.VEL, vh)

    sim.sph_write_state(B.POS, ph); sim.sph_write_state(B.VEL, vh)
    for _ in range(3):
        e2e_step()
    sim.sph_host_sync()
    barrier()
    e0.record(stream)
    t0 = time.perf_counter()
    for _ in range(Ke):
        e2e_step()
    sim.sph_host_sync()
    e1.record(stream)
    stream.synchronize()
    wall = time.perf_counter() - t0
    barrier()
    ems = max(e0.elapsed_time(e1), wall * 1e3)
    e2e_value = job_throughput(nf, Ke, max_over_ranks(ems, world, "cuda"), world)

    # ---- the same metric later in the run: the driver's short default window (W + K = 25 steps) ends before
    # the blocks of config 4 reach the obstacles (step ~75); this window starts at step >= 130, on the
    # disordered post-impact state (reported beside the headline, not instead of it)
    impact = None
    if not args.no_impact_window:
        done = int(sim.sph_read_stats()["steps_done"])
        first = max(done, args.impact_first_step)
        if first > done:
            sim_step(first - done)
        Ki = max(1, min(K, 30))
        stA = sim.sph_read_stats()
        barrier()
        e0.record(stream)
        sim_step(Ki)
        e1.record(stream)
        stream.synchronize()
        barrier()
        stB = sim.sph_read_stats()
        ims = max_over_ranks(e0.elapsed_time(e1), world, "cuda")
        impact = {"first_step": first, "steps": Ki, "ms_per_step": ims / Ki, "value": job_throughput(nf, Ki, ims, world),
                  "unit": UNIT, "mean_it_v": (stB["total_it_v"] - stA["total_it_v"]) / Ki,
                  "mean_it_d": (stB["total_it_d"] - stA["total_it_d"]) / Ki, "v_max": stB["v_max"],
                  "err_rho_last": stB["err_rho"], "mean_fluid_neighbours": stB["mean_fluid_neighbors"],
                  "max_fluid_neighbours": stB["max_fluid_neighbors"]}
    sim.close()

    out = None
    if rank == 0:
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": sc.name, "n_fluid": nf, "n_boundary": sc.n_boundary,
                       "n_cells": int(sim.ncells), "dt": sc.params["dt"],
                       "solver": {"dfsph": "DFSPH", "pcisph": "PCISPH", "wcsph": "WCSPH"}[args.method] + (" + warm start" if args.warm_start else ""),
                       "eta_density": sc.params["eta_density"],
                       "mean_it_v": mean_it_v, "mean_it_d": mean_it_d,
                       "neighbour_passes_per_step": 1 + 2 * mean_it_v + 2 * mean_it_d,
                       "parallelism": "replicas x%d" % world if world > 1 else "1 GPU",
                       "launch_mode": "host-driven launches (--no-graph)" if args.no_graph else "one CUDA graph per step, device-side WHILE loops",
                       "l2": "no flush: the per-step working set (lists + SoA store, ~%d MB) exceeds the 126 MB L2"
                             % int(sim.workspace_bytes / 2 ** 20 * 0.6),
                       "err_rho_last": st1["err_rho"], "v_max_last": st1["v_max"]},
            "clocks": ck,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": nf * 24, "d2h_bytes_per_step": nf * 24,
                    "steps": Ke, "mode": "pinned host buffers, asynchronous copies (uploads on a second stream, chunk k of a field uploaded behind its download)"},
            "gpu_launches": int(launches),
        }
        if impact is not None:
            out["impact_phase"] = impact

    # ---- per-kernel CUDA-event timing over the same W + K steps (host-driven launch mode: events
    # cannot bracket nodes inside a graph's WHILE body), rank 0 only -> roofline of the dominant kernel
    if rank == 0 and not args.no_breakdown:
        sim2 = B.Sim.from_scene(sc, device=local_rank, use_cuda_graph=0)
        step_of(sim2)(W)
        sim2.sph_build_grid()   # no-op for the physics: refreshes lists for the statistics below
        cnt = sim2.sph_read_state(B.NEIGHBOR_COUNT).to(torch.float64)
        nf_mean, nb_mean = float(cnt[:, 0].mean()), float(cnt[:, 1].mean())
        cs = sim2.sph_read_state(B.CELL_START).to(torch.int64)
        occ = (cs[1:] - cs[:-1]).to(torch.float32).reshape(1, 1, sim2.nz, sim2.ny, sim2.nx)
        # candidates per particle of the 27-cell walk = occupancy of the 3x3x3 cell box around it
        box = 27.0 * torch.nn.functional.avg_pool3d(occ, 3, stride=1, padding=1, count_include_pad=True)
        cand_mean = float((occ * box).sum() / max(float(occ.sum()), 1.0)) * (2.0 + 1.0 / FINE_X) / 3.0
        sim2.sph_enable_kernel_timing(True)
        step_of(sim2)(K)
        kt = sim2.sph_read_kernel_times()
        sim2_ncells = sim2.ncells
        sim2.close()
        tot = sum(v[1] for v in kt.values())
        table = {k: {"launches": v[0], "ms_total": round(v[1], 3), "us_avg": round(1e3 * v[1] / v[0], 2),
                     "share": round(v[1] / tot, 4)} for k, v in sorted(kt.items(), key=lambda kv: -kv[1][1])}
        top = next(iter(table))
        cells_pp = float(sim2_ncells) / max(nf, 1)
        work = kernel_work(top, nf_mean, nb_mean, cand_mean)
        dur = 1e-3 * kt[top][1] / kt[top][0]
        fp32_peak = N_SM * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
        prof, prof_sha = read_ncu_profile()
        stale = prof_sha is not None and prof_sha != csrc_sha16()
        if stale:
            sys.stderr.write("bench.py: WARNING: %s was captured from other kernel sources (csrc_sha16 %s, now %s): "
                             "its DRAM traffic is NOT reported; re-capture it\n" % (NCU_PROFILE, prof_sha, csrc_sha16()))
        pm = None if stale else ncu_for_kernel(prof, top)
        traffic = (pm["dram__bytes_read.sum"] + pm["dram__bytes_write.sum"]) * 1e6 if pm and "dram__bytes_read.sum" in pm else None
        roof = {"kernel": top, "row": work["row"] if work else None, "avg_us": round(dur * 1e6, 2),
                "share_of_step": table[top]["share"], "traffic": traffic,
                "traffic_source": NCU_PROFILE if traffic is not None else None,
                "l1tex_throughput_pct_ncu": pm.get("l1tex__throughput.avg.pct_of_peak_sustained_active") if pm else None,
                "issue_active_pct_ncu": pm.get("smsp__issue_active.avg.pct_of_peak_sustained_active") if pm else None,
                "peak_source": peaks["source"] + " (MEASURED_PEAKS.json)"}
        if work:
            gbs = work["bytes_8d"] * nf / dur / 1e9
            gbs_l = work["bytes_lists"] * nf / dur / 1e9
            tfl = work["flops"] * nf / dur / 1e12
            roof.update({"bound": "hbm", "algorithmic_bytes": work["bytes_8d"] * nf,
                         "algorithmic_bytes_per_particle": work["bytes_8d"],
                         "achieved": gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": gbs / peaks["hbm_gbs"],
                         "frac_with_lists": gbs_l / peaks["hbm_gbs"], "bytes_with_lists_per_particle": work["bytes_lists"],
                         "traffic_over_algorithmic": (traffic / (work["bytes_8d"] * nf)) if traffic else None,
                         "alu_achieved_tflops": tfl, "alu_frac": tfl / fp32_peak,
                         "note": "frac = SURVEY 8(d) compulsory bytes / event-timed duration / measured HBM peak; the list "
                                 "passes are bound by L1 gather wavefronts and instruction issue (see l1tex / issue figures), "
                                 "not by HBM"})
        sb = step_bytes_8d(mean_it_v, mean_it_d, cells_pp) * nf
        out["roofline_step"] = {"bound": "hbm", "algorithmic_bytes": sb, "achieved": sb / (ms_max / K * 1e-3) / 1e9,
                                "peak": peaks["hbm_gbs"], "unit": "GB/s",
                                "frac": sb / (ms_max / K * 1e-3) / 1e9 / peaks["hbm_gbs"],
                                "what": "SURVEY 8(d) bytes of the whole step / ms_per_step"}
        per_kernel = {}
        for k in table:
            w = kernel_work(k, nf_mean, nb_mean, cand_mean)
            if w:
                d = 1e-3 * kt[k][1] / kt[k][0]
                km = None if stale else ncu_for_kernel(prof, k)
                per_kernel[k] = {"row": w["row"], "us_avg": table[k]["us_avg"], "share": table[k]["share"],
                                 "hbm_frac": round(w["bytes_8d"] * nf / d / 1e9 / peaks["hbm_gbs"], 4),
                                 "hbm_frac_with_lists": round(w["bytes_lists"] * nf / d / 1e9 / peaks["hbm_gbs"], 4),
                                 "fp32_tflops": round(w["flops"] * nf / d / 1e12, 2),
                                 "dram_bytes_ncu": ((km["dram__bytes_read.sum"] + km["dram__bytes_write.sum"]) * 1e6
                                                    if km and "dram__bytes_read.sum" in km else None)}
        out["roofline"] = roof
        out["kernels"] = per_kernel
        out["kernel_time_table"] = table
        out["config"].update({"mean_fluid_neighbours": nf_mean, "mean_boundary_neighbours": nb_mean,
                              "mean_candidates": cand_mean,
                              "kernel_ms_per_step_sum": tot / K})

    # ---- the oracle on the host cores, bounded sample (rank 0, N = 1 only)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = time_oracle(sc, budget_s=args.cpu_budget)
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def time_oracle(sc, budget_s=20.0, steps=None):
    """Oracle (as it stands) on this box's host cores: DFSPH steps of the same scene from its
    initial state, as many as fit the budget (at least 2)."""
    from oracle import sphref
    sphref.build()
    o = sphref.Sim.from_scene(sc)
    t0 = time.perf_counter()
    o.step_dfsph()
    t1 = time.perf_counter() - t0
    n = steps if steps is not None else max(2, min(50, int(budget_s / max(t1, 1e-6))))
    t0 = time.perf_counter()
    for _ in range(n):
        o.step_dfsph()
    dt = time.perf_counter() - t0
    so = o.stats()
    o.close()
    return {"value": sc.n_fluid * n / dt, "unit": UNIT, "cores": sphref.num_threads(), "kind": "oracle",
            "sample": "%d DFSPH steps of %s (%d fluid particles) after 1 untimed step; it_v=%d it_d=%d in the last"
                      % (n, sc.name, sc.n_fluid, so["it_v"], so["it_d"]),
            "s_per_step": dt / n}


def run_reference(args):
    """Reference arm = the fp64 oracle on the host cores (there is no other reference
    implementation: /root/reference holds only the paper).  Each step is one oracle DFSPH step on
    a bounded sample of the workload: the config-4 scene generator at a particle count chosen so
    that W + K steps end within ~2 minutes."""
    rank, _, world = dist_env()
    if rank != 0:
        return
    from paper_2403_11156_b200 import scenes
    from oracle import sphref
    sphref.build()
    K, W = args.steps, args.warmup
    full = scenes.config(args.config, seed=0)
    o = sphref.Sim.from_scene(full)
    t0 = time.perf_counter(); o.step_dfsph(); t_full = time.perf_counter() - t0
    o.close()
    budget = 120.0
    frac = min(1.0, budget / max((K + W) * t_full, 1e-9))
    if frac >= 1.0 or args.config != 4:
        sc = full
    else:
        sc = scenes.splash(n_target=max(2e4, 1.23e6 * frac), seed=0, name="config4_splash_sample")
    o = sphref.Sim.from_scene(sc)
    for _ in range(W):
        o.step_dfsph()
    t0 = time.perf_counter()
    for _ in range(K):
        o.step_dfsph()
    dt = time.perf_counter() - t0
    o.close()
    value = sc.n_fluid * K / dt
    sample = "%d oracle DFSPH steps on the config-4 scene generator at %d fluid particles (%.1f%% of 1.23M)" % (
        K, sc.n_fluid, 100.0 * sc.n_fluid / 1.23e6)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K,
        "warmup": W, "ms_per_step": 1e3 * dt / K, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": full.name, "n_fluid": full.n_fluid, "n_boundary": full.n_boundary, "dt": full.params["dt"],
                   "solver": "DFSPH", "sample_n_fluid": sc.n_fluid},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": sphref.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--e2e-steps", type=int, default=50)
    ap.add_argument("--cpu-budget", type=float, default=20.0)
    ap.add_argument("--no-graph", action="store_true",
                    help="host-driven launches instead of the CUDA graph (ncu cannot profile kernel nodes of a "
                         "graph that has conditional nodes): for profiling commands only")
    ap.add_argument("--n-target", type=float, default=0.0,
                    help="scaling sweep: config-4 scene proportions at this many fluid particles (250e3 / 4e6 / 8e6); "
                         "not the headline line")
    ap.add_argument("--no-breakdown", action="store_true")
    ap.add_argument("--no-impact-window", action="store_true")
    ap.add_argument("--impact-first-step", type=int, default=130)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--method", default="dfsph", choices=["dfsph", "pcisph", "wcsph"],
                    help="step method (the headline metric is DFSPH; the others are the library's other solvers on the same scene)")
    ap.add_argument("--warm-start", action="store_true", help="DFSPH with warm start (reading R27); not the headline line")
    ap.add_argument("--eta-density", type=float, default=0.0, help="override the density tolerance (0: the config's 1e-3)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
