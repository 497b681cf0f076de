#!/usr/bin/env python
"""bench.py - throughput of the Sim(3) Gauss-Newton step (libsim3ba) on synthetic graphs shaped like
BASELINE.json's configs.  One "step" = one pass of the whole hot path (a1-a8: per-match residual /
Jacobian, block reduction, assembly, Cholesky solve, retraction) over the workload's graph.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference] [--probe-fp64]

Default workload: BASELINE configs[4] (C5, the largest single-GPU configuration: 2000 keyframes 512x384, 6003 edges,
1.18e9 candidate matches, n = 14000); the same line carries `per_config` entries for C1-C4 and the tracker shape.
Prints ONE JSON line (contract in the task statement; field meanings in DESIGN.md "Measurement").
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "valid correspondences/s through one Sim(3) GN iteration (a1-a8)"
UNIT = "corr/s"
SMI_QUERY = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
             "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
FLOP_PER_MATCH = 300.0      # fp32 flop per valid match of kernel 1 (FMA = 2)


# ------------------------------------------------------------------------------------------------
def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def load_traffic(config_id: int):
    """dram bytes per launch of the dominant kernel from the committed ncu capture, if any."""
    path = os.path.join(ROOT, "profiles", "roofline_traffic.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f).get(f"C{config_id}", {}).get("k_accumulate_dram_bytes_per_launch")
    return None


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons DURING the timed region."""

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={SMI_QUERY}", "--format=csv,noheader,nounits",
                 "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), [x.strip() for x in line.split(",")]))

    def mark(self):
        """Host time stamp; samples are attributed to the timed region by their arrival time."""
        return time.perf_counter()

    def stop(self, t0=None, t1=None):
        """Statistics over the samples that arrived in [t0, t1]."""
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.kill()                          # gone before anything else is timed: a polling nvidia-smi slows driver calls
        try:
            self.proc.wait(timeout=5)
        except Exception:
            pass
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (t, r) in self.rows if t0 is None or (t0 <= t <= t1 + 0.03)]
        in_region = len(rows)
        if not rows:
            rows = [r for (_, r) in self.rows]
        for r in rows:
            try:
                sm.append(float(r[1]))
                mx.append(float(r[2]))
                for nm, v in zip(names, r[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                continue
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm), "samples_in_timed_region": in_region}


def dist_setup(n_gpus: int):
    """One process per GPU (torchrun).  Returns (rank, world, local_rank)."""
    import torch
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        backend = "nccl" if torch.cuda.is_available() else "gloo"
        if not dist.is_initialized():
            dist.init_process_group(backend=backend)
    return rank, world, local


def aggregate_over_ranks(ms_local: float, units_local: float, device=None):
    """Replicas-only weak scaling: barrier'd ranks each ran the same number of
    steps; job time = MAX over ranks, job units = SUM over ranks.  Works on gloo (CPU) and nccl."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return ms_local, units_local
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    u = torch.tensor([units_local], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()


# ------------------------------------------------------------------------------------------------
def workload_description(g, cfg_id):
    from sim3ba_inputs import config_params
    s = g.spec
    name = f"BASELINE configs[{cfg_id - 1}] {s.name}" if cfg_id else s.name
    lam = config_params(cfg_id).get("lm_lambda", 0.0)
    return {"workload": f"{name}: {g.n_kf} keyframes {s.width}x{s.height}, "
                        f"{g.n_edges} edges, {int(s.p_out * 100)}% outlier matches, preset sigma=1 kappa=0.05"
                        + (f", lambda={lam:g} (Eq. 7 damping: the undamped step leaves the basin on this chain, DESIGN.md section 5)" if lam else ""),
            "lm_lambda": lam,
            "n_kf": g.n_kf, "hw": g.hw, "n_edges": g.n_edges, "system_n": 7 * g.n_kf,
            "candidates_per_step": int(g.n_edges) * int(g.hw), "gn_iters_per_pose_reset": s.n_iters}


def tracker_graph():
    """The tracker's shape: one relative pose against a fixed keyframe -- N = 2, E = 1, n = 7."""
    from sim3ba_inputs import CONFIGS, make_graph
    return make_graph(CONFIGS[2].scaled(name="tracker-2kf", kf_per_agent=2, offsets=(1,), valid_frac=(0.9,), cyclic=False, n_iters=4))


def pin_in_place(a):
    """Page-locks a NumPy array where it is (cudaHostRegister) and returns it as a torch tensor: the graph is not held twice on
    the host (C5: 11 GB per rank).  Falls back to a pinned copy."""
    import torch
    t = torch.from_numpy(a)
    try:
        rc = torch.cuda.cudart().cudaHostRegister(t.data_ptr(), t.numel() * t.element_size(), 0)
        if int(rc) == 0 and t.is_pinned():
            return t
    except Exception:
        pass
    return t.pin_memory()


class Workload:
    """A graph resident on the device behind a libsim3ba context, with its seeded start."""

    def __init__(self, g, dev, pinned: bool, cfg_id: int = 0):
        import torch
        from sim3ba_inputs import config_params
        from paper_2605_30488_b200 import Sim3BA, make_params
        self.g, self.dev = g, dev
        self.preset = config_params(cfg_id)          # the preset + what this config adds (C5: lm_lambda)
        mk = pin_in_place if pinned else torch.from_numpy
        self.h_pts, self.h_cf, self.h_ed, self.h_mt = mk(g.points), mk(g.conf), torch.from_numpy(g.edges), mk(g.match)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        self.d_pts, self.d_cf = self.h_pts.to(dev, non_blocking=True), self.h_cf.to(dev, non_blocking=True)
        self.d_ed, self.d_mt = self.h_ed.to(dev, non_blocking=True), self.h_mt.to(dev, non_blocking=True)
        self.ba = Sim3BA(self.d_pts, self.d_cf, self.d_ed, self.d_mt, g.fixed_kf, make_params(**self.preset), g.spec.height, g.spec.width)
        torch.cuda.synchronize()
        self.upload_ms = (time.perf_counter() - t0) * 1e3
        self.upload_bytes = sum(t.numel() * t.element_size() for t in (self.h_pts, self.h_cf, self.h_ed, self.h_mt))
        # seeded start; config 3 hands out independent per-agent gauges: the library synchronises them, untimed
        self.ba.set_poses(torch.from_numpy(g.poses_init).to(dev))
        for e, moving, moving_is_i in g.meta.get("gauge_sync_plan", []):
            self.ba.gauge_sync(e, moving, moving_is_i)
        self.poses0 = self.ba.get_poses().clone()
        self.n_reset = max(1, g.spec.n_iters)
        self.ba.step()
        torch.cuda.synchronize()
        self.n_valid = int(self.ba.edge_stats()[0].sum().item())      # counted by the library itself

    def steps(self, n_steps, flush, timed=True):
        """n_steps GN iterations, CUDA events around each, L2 flushed and poses reset (every n_reset steps) untimed."""
        import torch
        total_ms = 0.0
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for s in range(n_steps):
            if s % self.n_reset == 0:
                self.ba.set_poses(self.poses0)
            flush.fill_(s & 0xFF)                 # L2 flush between timed iterations (untimed)
            torch.cuda.synchronize()
            ev0.record()
            self.ba.step()
            ev1.record()
            torch.cuda.synchronize()
            if timed:
                total_ms += ev0.elapsed_time(ev1)
        return total_ms

    def phases(self, n_steps, flush):
        """Per-kernel device times (CUDA events recorded by the library on its stream) over a second, identical loop."""
        import numpy as np
        import torch
        self.ba.set_profiling(True)
        ph, sp = [], []
        for s in range(n_steps):
            if s % self.n_reset == 0:
                self.ba.set_poses(self.poses0)
            flush.fill_(s & 0xFF)
            torch.cuda.synchronize()
            self.ba.step()
            ph.append(self.ba.phase_ms())
            sp.append(self.ba.solve_phase_us())
        self.ba.set_profiling(False)
        return np.asarray(ph)[:, :5].mean(axis=0), np.asarray(sp)[:, :6].mean(axis=0)

    def close(self):
        import torch
        from paper_2605_30488_b200 import release_memory
        self.ba.close()
        del self.d_pts, self.d_cf, self.d_ed, self.d_mt, self.h_pts, self.h_cf, self.h_mt
        torch.cuda.empty_cache()
        release_memory()


def rooflines(w: Workload, cfg_id, ph, ms_per_step, hbm_peak, peak_src, n_sms, sm_max_mhz, fp64_peaks):
    """Rooflines of kernel 1 (algorithmic bytes, stream accounting, fp32 ALU) and of the solve (plan flops over FP64 peak)."""
    g = w.g
    cand = g.n_edges * g.hw
    bytes_min = 4.0 * cand + 16.0 * g.n_kf * g.hw          # unique bytes: every index + every packed pixel once
    bytes_stream = 36.0 * cand                              # no-reuse accounting (4 idx + 16 X_i + 16 X_j)
    k1_s = max(float(ph[0]), 1e-9) * 1e-3
    traffic = load_traffic(cfg_id) if cfg_id else None
    roof = {"bound": "hbm", "kernel": "k_accumulate", "achieved": bytes_min / k1_s / 1e9, "peak": hbm_peak, "unit": "GB/s",
            "frac": bytes_min / k1_s / 1e9 / hbm_peak, "traffic": traffic, "peak_source": peak_src,
            "algorithmic_bytes_per_launch": bytes_min,
            "frac_dram_bytes": (traffic / k1_s / 1e9 / hbm_peak) if traffic else None,
            "achieved_stream_accounting": bytes_stream / k1_s / 1e9,
            "frac_stream_accounting": bytes_stream / k1_s / 1e9 / hbm_peak,
            "note": "kernel 1 sits on the ridge: HBM traffic equals the unique bytes (ncu), the binding resource is fp32 issue "
                    "(roofline_alu); north_star's 60 % HBM figure is met only on the no-reuse stream accounting"}
    alu_peak = n_sms * 128 * 2 * sm_max_mhz * 1e6
    alu = {"bound": "alu", "kernel": "k_accumulate", "achieved": FLOP_PER_MATCH * w.n_valid / k1_s / 1e12, "peak": alu_peak / 1e12,
           "unit": "TFLOP/s", "frac": FLOP_PER_MATCH * w.n_valid / k1_s / alu_peak, "flop_per_valid_match": FLOP_PER_MATCH}
    info = w.ba.solver_info()
    bb = w.ba.bb_info()
    solve_s = max(float(ph[3]) + float(ph[2]), 1e-9) * 1e-3
    dfma, dmma = fp64_peaks
    solve = {"bound": "fp64", "kernel": "k_solve_bb" if bb["valid"] else "k_solve", "plan_flops": info["flops"],
             "achieved": info["flops"] / solve_s / 1e12, "peak": max(dfma, dmma), "unit": "TFLOP/s",
             "frac": info["flops"] / solve_s / 1e12 / max(dfma, dmma, 1e-9),
             "peak_source": f"measured here by sim3ba_probe_fp64: DFMA {dfma:.1f} TF, DMMA m8n8k4 {dmma:.1f} TF",
             "dense_equivalent_flops": (7.0 * g.n_kf) ** 3 / 3.0,
             "note": "the band + border plan removes the flops (dense n^3/3 above) instead of speeding them up; what is left is a "
                     "chain of dependent 7x7 pivots: latency-bound by construction"}
    return roof, alu, solve, dict(bb, mode="band + border block Cholesky (2)" if bb["valid"] else "tile-sparse (0)")


def per_config_entry(cfg_id, g, dev, flush, steps, hbm_peak, peak_src, n_sms, sm_max_mhz, fp64_peaks):
    import torch
    w = Workload(g, dev, pinned=False, cfg_id=cfg_id)
    w.steps(3, flush, timed=False)
    ms = w.steps(steps, flush) / steps
    ph, sp = w.phases(min(steps, 10), flush)
    roof, alu, solve, solver = rooflines(w, cfg_id, ph, ms, hbm_peak, peak_src, n_sms, sm_max_mhz, fp64_peaks)
    n_it = max(1, g.spec.n_iters)
    # the same iterations as ONE CUDA-graph launch (sim3ba_step_graph): what launch latency costs on the small configs
    w.ba.set_poses(w.poses0)
    w.ba.step_graph(n_it)
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps = 5
    tot = 0.0
    for _ in range(reps):
        w.ba.set_poses(w.poses0)
        torch.cuda.synchronize()
        ev0.record()
        w.ba.step_graph(n_it)
        ev1.record()
        torch.cuda.synchronize()
        tot += ev0.elapsed_time(ev1)
    out = dict(workload_description(g, cfg_id), valid_per_step=w.n_valid, steps=steps, ms_per_step=ms, value=w.n_valid / (ms * 1e-3),
               ms_per_step_cuda_graph=tot / (reps * n_it),
               phases_ms={"k1_accumulate": float(ph[0]), "k2_edge_reduce_gradient": float(ph[1]), "k3_assemble": float(ph[2]),
                          "k4_factor_solve": float(ph[3]), "k5_retract": float(ph[4])},
               k1_frac_hbm_algorithmic=roof["frac"], k1_frac_hbm_dram_bytes=roof["frac_dram_bytes"], k1_frac_hbm_stream=roof["frac_stream_accounting"],
               k1_frac_fp32_alu=alu["frac"], solve_ms=float(ph[3]) + float(ph[2]), solve_plan_flops=solve["plan_flops"],
               solve_frac_fp64=solve["frac"], solver=solver,
               solve_phases_us=dict(zip(("assemble", "segments", "barrier", "schur", "border_system", "back_substitution"), map(float, sp))))
    w.close()
    return out


def run_ours(args):
    import numpy as np
    import torch
    from sim3ba_inputs import make_config, make_depth_inputs
    from paper_2605_30488_b200 import build, make_params, optimize_host, probe_fp64, refine_host

    rank, world, local = dist_setup(args.gpus)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (libsim3ba has no CPU fallback)")
    build.build()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    st = torch.cuda.current_stream().cuda_stream
    fp64_peaks = probe_fp64(st)

    g = make_config(args.config)                 # replicas only: every rank owns an independent graph
    # The oracle leg runs FIRST, on pageable memory: its worker processes are forked, and forking a process that holds
    # gigabytes of page-locked memory makes the kernel copy those pages for every child.
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        from sim3ba_inputs import config_params
        cpu = cpu_baseline(g, config_params(args.config), budget_s=8.0)
    # inputs start in pinned host memory; the graph upload is the one-off part of the end-to-end job
    w = Workload(g, dev, pinned=True, cfg_id=args.config)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)   # > 126 MB L2

    sampler = ClockSampler(local)
    sampler.start()                               # nvidia-smi needs a few hundred ms to come up: started before the warm-up
    w.steps(args.warmup, flush, timed=False)
    t_up = time.perf_counter()
    while sampler.proc is not None and len(sampler.rows) < 2 and time.perf_counter() - t_up < 5.0:
        w.steps(20, flush, timed=False)           # same load, untimed, until the sampler delivers
    barrier()
    torch.cuda.synchronize()
    t_begin = sampler.mark()
    l0 = w.ba.launch_count()
    total_ms = w.steps(args.steps, flush)
    l1 = w.ba.launch_count()
    torch.cuda.synchronize()
    t_end = sampler.mark()
    barrier()
    clocks = sampler.stop(t_begin, t_end)
    ms_per_step = total_ms / args.steps
    ph, sp = w.phases(min(args.steps, 50), flush)
    # a config that runs with the Eq. (7) damping (C5): the same iterations undamped, for the record -- same work per step,
    # plus the retried factorisation on the iteration where H has lost definiteness
    undamped = None
    if w.preset.get("lm_lambda", 0.0) != 0.0 and world == 1:
        n_u = 2 * max(1, g.spec.n_iters)
        w.ba.set_params(make_params(**dict(w.preset, lm_lambda=0.0)))
        w.steps(max(1, g.spec.n_iters), flush, timed=False)
        undamped = {"lm_lambda": 0.0, "steps": n_u, "ms_per_step": w.steps(n_u, flush) / n_u,
                    "note": "undamped GN leaves the basin on this chain (cost rises from the third iteration); not the reported configuration"}
        w.ba.set_params(make_params(**w.preset))

    # ---- end to end through the C ABI with HOST buffers (pinned).  Pose-only job: sim3ba_optimize_host = device allocation
    # + upload of the whole graph + create (pack, bookkeeping, solve plan) + n_iters GN steps + poses and costs back + free.
    n_it = max(1, g.spec.n_iters)
    prm = make_params(**w.preset)
    h_in = torch.from_numpy(g.poses_init.copy()).pin_memory()
    h_out = torch.empty((g.n_kf, 8), dtype=torch.float64).pin_memory()
    h_cost = torch.empty((n_it,), dtype=torch.float64).pin_memory()

    def timed_jobs(job, n_jobs):
        job()                                         # two warm-up jobs (the library's pool, page tables)
        job()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        torch.cuda.synchronize()
        w0 = time.perf_counter()
        ev0.record()
        for _ in range(n_jobs):
            job()
        ev1.record()
        torch.cuda.synchronize()
        wall = (time.perf_counter() - w0) * 1e3
        return max(ev0.elapsed_time(ev1), wall) / n_jobs

    n_jobs = max(1, min(args.steps // n_it, 10))
    pose_job_ms = timed_jobs(lambda: optimize_host(w.h_pts, w.h_cf, w.h_ed, w.h_mt, g.fixed_kf, prm, g.spec.height, g.spec.width,
                                                   h_in, n_it, h_out, h_cost, st), n_jobs)
    e2e_ms = pose_job_ms / n_it
    e2e = {"ms_per_step": None, "h2d_bytes_per_step": (w.upload_bytes + g.n_kf * 64) / n_it, "d2h_bytes_per_step": (g.n_kf * 64 + 8 * n_it) / n_it,
           "jobs": n_jobs, "steps_per_job": n_it,
           "what": "sim3ba_optimize_host: device allocation + upload of the whole graph from pinned host memory "
                   "+ create + n_iters GN steps + poses and costs back + free; per step = job / n_iters"}

    # ---- the structure pass (NEXT-1) and, on config 5, the pose-depth alternation as one host job (sim3ba_refine_host)
    depth, alternation = None, None
    if args.config == 5 or args.depth:
        depth = {"what": "sim3ba_depth_refine, 10 iterations (PAPER.md:143), poses fixed at the seeded start", "per_labelling": []}
        n_dit = 10
        for irregular in (0, 200):
            d = make_depth_inputs(g, irregular=irregular)
            labels = torch.from_numpy(d.labels).to(dev)
            eta = torch.zeros(g.n_kf * d.n_seg, dtype=torch.float64, device=dev)
            w.ba.set_poses(w.poses0)
            w.ba.depth_refine(labels, d.n_seg, d.pairs, d.delta, d.anchor_kf, eta, 1)          # warm-up (allocations)
            eta.zero_()
            torch.cuda.synchronize()
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ev0.record()
            costs = w.ba.depth_refine(labels, d.n_seg, d.pairs, d.delta, d.anchor_kf, eta, n_dit)
            ev1.record()
            torch.cuda.synchronize()
            pass_ms = ev0.elapsed_time(ev1)
            it_ms = pass_ms / n_dit
            # the same pass with twice the iterations: the difference is the cost of an iteration proper, the rest the
            # once-per-pass part (k_depth_prep, the label tables)
            eta.zero_()
            torch.cuda.synchronize()
            ev0.record()
            w.ba.depth_refine(labels, d.n_seg, d.pairs, d.delta, d.anchor_kf, eta, 2 * n_dit)
            ev1.record()
            torch.cuda.synchronize()
            marginal_ms = (ev0.elapsed_time(ev1) - pass_ms) / n_dit
            dbytes = 20.0 * g.n_edges * g.hw + 20.0 * g.n_kf * g.hw      # per iteration: record + label per candidate, X_i + label per pixel
            depth["per_labelling"].append({
                "labels": "4x8 grid (BASELINE config 5: 32 segments per keyframe)" if irregular == 0 else
                          "jittered superpixels (the paper's M_k ~ 200, PAPER.md:126)",
                "segments_per_kf": d.n_seg, "ms_per_iteration": it_ms,
                "ms_per_iteration_marginal": marginal_ms, "ms_once_per_pass": pass_ms - n_dit * marginal_ms,
                "roofline": {"bound": "hbm", "kernel": "k_depth_edge", "algorithmic_bytes_per_iteration": dbytes,
                             "achieved": dbytes / (it_ms * 1e-3) / 1e9, "peak": load_peaks()[0], "unit": "GB/s",
                             "frac": dbytes / (it_ms * 1e-3) / 1e9 / load_peaks()[0],
                             "note": "time = the whole iteration (k_depth_edge + objective + update kernels) plus a tenth of the "
                                     "once-per-pass k_depth_prep"},
                "objective_first_last": [float(costs[0]), float(costs[-1])]})
            if irregular == 0 and args.config == 5:
                h_lab = torch.from_numpy(d.labels).pin_memory()
                h_eta = torch.zeros(g.n_kf * d.n_seg, dtype=torch.float64).pin_memory()

                def alt_job():
                    h_eta.zero_()
                    refine_host(w.h_pts, w.h_cf, w.h_ed, w.h_mt, g.fixed_kf, prm, g.spec.height, g.spec.width, h_lab, d.n_seg, d.pairs,
                                d.delta, None, 1, n_dit, n_it, h_in, h_out, h_eta, None, None, st)

                alt_ms = timed_jobs(alt_job, max(1, n_jobs // 2))
                alternation = {
                    "ms_per_job": alt_ms, "ms_per_step": alt_ms / n_it, "value": w.n_valid * n_it / (alt_ms * 1e-3), "unit": UNIT,
                    "h2d_bytes_per_step": (w.upload_bytes + d.labels.nbytes + h_eta.numel() * 8 + g.n_kf * 64) / n_it,
                    "d2h_bytes_per_step": (g.n_kf * 64 + h_eta.numel() * 8) / n_it,
                    "what": f"sim3ba_refine_host, BASELINE config 5's whole job: upload of the graph and the labels from pinned host "
                            f"memory + create + one pose-depth round ({n_dit} structure iterations on {d.n_seg} segments per "
                            f"keyframe, apply, {n_it} GN iterations) + poses and eta back + free; value counts the GN iterations' "
                            f"valid correspondences over the whole job time"}
            del labels, eta

    job_ms, job_units = aggregate_over_ranks(ms_per_step, float(w.n_valid), dev)
    e2e_job_ms, _ = aggregate_over_ranks(e2e_ms, float(w.n_valid), dev)
    hbm_peak, peak_src = load_peaks()
    n_sms = torch.cuda.get_device_properties(dev).multi_processor_count
    sm_max_mhz = float(clocks.get("sm_max_mhz") or 1965.0)
    roof, alu, solve, solver = rooflines(w, args.config, ph, ms_per_step, hbm_peak, peak_src, n_sms, sm_max_mhz, fp64_peaks)
    upload_ms, upload_bytes, n_valid = w.upload_ms, w.upload_bytes, w.n_valid
    cand = g.n_edges * g.hw
    launches = int(l1 - l0)

    per_config = {}
    if rank == 0 and world == 1 and not args.no_per_config:
        w.close()
        for k in (1, 2, 3, 4, 5):
            if k == args.config:
                continue
            gk = make_config(k)
            per_config[f"C{k}"] = per_config_entry(k, gk, dev, flush, 30 if k < 5 else 10, hbm_peak, peak_src, n_sms, sm_max_mhz, fp64_peaks)
            del gk
        per_config["tracker"] = per_config_entry(0, tracker_graph(), dev, flush, 30, hbm_peak, peak_src, n_sms, sm_max_mhz, fp64_peaks)
    if rank != 0:
        return
    e2e.update(value=job_units / (e2e_job_ms * 1e-3), unit=UNIT, ms_per_step=e2e_job_ms)
    out = {
        "metric": METRIC, "value": job_units / (job_ms * 1e-3), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": job_ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32 per-match, f64 reduce/solve", "data": "synthetic",
        "config": dict(workload_description(g, args.config), l2="flushed between timed steps (256 MB write)",
                       valid_per_step=n_valid, graph_upload_ms=upload_ms, graph_upload_bytes=upload_bytes,
                       multi_gpu="replicas only (independent graph per rank, no collective)"),
        "clocks": clocks,
        "e2e": e2e,
        "gpu_launches": launches,
        "phases_ms": {"k1_accumulate": float(ph[0]), "k2_edge_reduce_gradient": float(ph[1]),
                      "k3_assemble": float(ph[2]), "k4_factor_solve": float(ph[3]), "k5_retract": float(ph[4]),
                      "note": "from a second loop with event records between the kernels: their sum exceeds ms_per_step by the event gaps"},
        "solve_phases_us": dict(zip(("assemble", "segments", "barrier", "schur", "border_system", "back_substitution"), map(float, sp))),
        "candidates_per_s": cand * world / (job_ms * 1e-3),
        "roofline": roof, "roofline_alu": alu, "roofline_solve": solve, "solver": solver,
        "fp64_peak_probe": {"dfma_tflops": fp64_peaks[0], "dmma_tflops": fp64_peaks[1]},
    }
    if undamped is not None:
        out["undamped"] = undamped
    if depth is not None:
        out["depth_refine"] = depth
    if alternation is not None:
        out["e2e_alternation"] = alternation
    if per_config:
        out["per_config"] = per_config
    assert clocks.get("samples_in_timed_region", 0) > 0 or clocks.get("sm_mhz") is None or total_ms < 200.0, \
        "no nvidia-smi sample landed inside the timed region"
    if cpu is not None:
        out["cpu_baseline"] = cpu
    print(json.dumps(out))


# ------------------------------------------------------------------------------------------------
def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_assemble(g, preset, edges_sample, n_workers, px_limit=None):
    """The oracle's normal-equation assembly over a sample of edges on n_workers cores; (seconds, valid matches, system)."""
    from oracle import sim3_gn_oracle as orc
    from oracle.edge_pool import build_system_parallel
    prm = orc.Params(**preset)
    match = g.match
    if px_limit is not None:
        match = g.match[:max(edges_sample) + 1].copy()
        match[:, px_limit:] = -1
    t0 = time.perf_counter()
    sysm = build_system_parallel(g.poses_init, g.points, g.conf, g.edges, match, prm, edge_subset=edges_sample, n_workers=n_workers, dense=False)
    return time.perf_counter() - t0, int(sysm.n_valid.sum()), sysm


def oracle_rate_1core(g, preset):
    """Valid matches per second of the oracle on one core, from a short probe (the first pixels of edge 0)."""
    px = min(g.hw, 16384)
    oracle_assemble(g, preset, [0], 1, px)
    dt, nv, _ = oracle_assemble(g, preset, [0], 1, px)
    return max(nv, 1) / max(dt, 1e-6), px / max(dt, 1e-6)


def oracle_sample(g, budget_s, cand_rate, n_workers):
    """Bounded sample of the workload for the CPU oracle: the first edges whose work fits budget_s on n_workers cores, or --
    when not even one edge fits -- the first pixels of edge 0.  Returns (edge list, pixel limit or None)."""
    per_edge_s = g.hw / cand_rate
    n = int(budget_s * n_workers / per_edge_s)
    if n >= 1:
        return list(range(max(1, min(g.n_edges, n)))), None
    return [0], max(1024, int(budget_s * cand_rate))


def oracle_solve_seconds(g, preset, sysm_sample, threads):
    """The oracle's Eq. (7) solve and retraction at the workload's FULL system size.  The system is the sampled edges' sum plus
    1e-3 I (a partial graph is rank-deficient); a dense Cholesky does the same n^3/3 flops whatever the entries."""
    import numpy as np
    from threadpoolctl import threadpool_limits
    from oracle import sim3_gn_oracle as orc
    prm = orc.Params(**preset)
    n = 7 * g.n_kf
    H = np.zeros((n, n))
    for e in np.flatnonzero(sysm_sample.n_valid > 0):
        i, j = int(g.edges[e, 0]), int(g.edges[e, 1])
        A = sysm_sample.edge_A[e]
        si, sj = slice(7 * i, 7 * i + 7), slice(7 * j, 7 * j + 7)
        H[si, si] += A
        H[sj, sj] += A
        H[si, sj] -= A
        H[sj, si] -= A
    H[np.diag_indices(n)] += 1e-3
    with threadpool_limits(limits=threads):
        t0 = time.perf_counter()
        sol = orc.solve(H, sysm_sample.g, g.fixed_kf, prm)
        orc.retract(g.poses_init, sol.tau)
        return time.perf_counter() - t0


def cpu_baseline(g, preset, budget_s=8.0, with_solve=True):
    """The oracle as it stands on the host cores: assembly rate on 1 core and on every core (edge-parallel pool over a bounded
    sample of edges), the full-size solve + retraction, and the whole GN iteration they add up to for this workload."""
    from oracle.edge_pool import host_cores
    cores = host_cores()
    valid_rate1, cand_rate1 = oracle_rate_1core(g, preset)
    s1, px1 = oracle_sample(g, budget_s, cand_rate1, 1)
    dt1, nv1, _ = oracle_assemble(g, preset, s1, 1, px1)
    sN, pxN = oracle_sample(g, budget_s, cand_rate1, cores)
    dtN, nvN, sysm = oracle_assemble(g, preset, sN, cores, pxN)
    rate1, rateN = nv1 / dt1, nvN / dtN
    solve_s = oracle_solve_seconds(g, preset, sysm, cores) if with_solve else 0.0
    # valid matches of the whole workload, extrapolated from the sample's valid fraction
    n_valid_total = nvN / (len(sN) * (pxN or g.hw)) * g.n_edges * g.hw
    it_1 = n_valid_total / rate1 + solve_s
    it_N = n_valid_total / rateN + solve_s
    return {"value": n_valid_total / it_N, "unit": UNIT, "cores": cores, "kind": "oracle", "cpu_model": cpu_model(),
            "value_1core": n_valid_total / it_1, "assemble_corr_per_s_1core": rate1, "assemble_corr_per_s_all_cores": rateN,
            "solve_retract_seconds_full_size": solve_s, "seconds_spent": dt1 + dtN + solve_s,
            "sample": f"oracle/sim3_gn_oracle.py as it stands (NumPy float64): assembly timed on edges 0..{len(s1) - 1} with 1 core and on "
                      f"edges 0..{len(sN) - 1} of {g.n_edges} with {cores} worker processes (oracle/edge_pool.py"
                      + (f", first {pxN} pixels" if pxN else "") + "), BLAS 1 thread per worker; Eq. (7) solve + retraction timed once at the "
                      f"full system size n = {7 * g.n_kf} with {cores} BLAS threads; value = valid matches of the whole graph / "
                      "(assembly extrapolated to all edges + solve)"}


def run_reference(args):
    """The reference arm of this tier is the oracle, as it stands, on the host cores: each step = the oracle's assembly over a
    bounded sample of edges on every core (edge-parallel pool); the full-size solve is timed once and charged to every step in
    proportion to the sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle.edge_pool import host_cores
    from sim3ba_inputs import config_params, make_config
    g = make_config(args.config)
    preset = config_params(args.config)
    cores = host_cores()
    # bounded sample per step so that the whole --steps K --warmup W run ends within a couple of minutes
    per_step_s = min(3.0, max(0.25, 60.0 / max(1, args.steps + args.warmup)))
    _, cand_rate1 = oracle_rate_1core(g, preset)
    sample, px = oracle_sample(g, per_step_s, cand_rate1, cores)
    for _ in range(args.warmup):
        oracle_assemble(g, preset, sample, cores, px)
    tot, units, sysm = 0.0, 0, None
    for _ in range(args.steps):
        dt, nv, sysm = oracle_assemble(g, preset, sample, cores, px)
        tot += dt
        units += nv
    frac = len(sample) * (px or g.hw) / (g.n_edges * g.hw)
    solve_s = oracle_solve_seconds(g, preset, sysm, cores) if args.steps > 0 else 0.0
    tot += solve_s * frac * args.steps                 # the solve's share of a step that covers `frac` of the graph
    val = units / tot
    desc = (f"oracle/sim3_gn_oracle.py as it stands, each step = assembly over edges 0..{len(sample) - 1} of {g.n_edges}"
            + (f", first {px} pixels" if px is not None else "") + f" on {cores} worker processes (oracle/edge_pool.py, BLAS 1 thread each) "
            f"+ that fraction ({frac:.3g}) of the full-size solve + retraction ({solve_s:.2f} s with {cores} BLAS threads)")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": tot / max(1, args.steps) * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": workload_description(g, args.config),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "cpu_model": cpu_model(), "sample": desc},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_probe_fp64():
    import torch
    from paper_2605_30488_b200 import build, probe_fp64
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --probe-fp64: no CUDA device")
    build.build()
    dfma, dmma = probe_fp64(torch.cuda.current_stream().cuda_stream)
    print(json.dumps({"probe": "fp64", "gpu": torch.cuda.get_device_name(0), "dfma_tflops": dfma, "dmma_m8n8k4_tflops": dmma,
                      "how": "sim3ba_probe_fp64: register-resident chains, 8 per thread, 256 threads x 8 CTAs per SM, best of 5, CUDA events"}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--depth", action="store_true", help="also time the segment log-depth refinement on configs other than 5")
    ap.add_argument("--probe-fp64", action="store_true", help="only measure the FP64 peaks (DFMA, DMMA) of this device")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config entries of the other configs")
    ap.add_argument("--no-cpu-baseline", action="store_true",
                    help="skip the oracle timing leg (profiling runs under ncu; never for a reported line)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.probe_fp64:
        run_probe_fp64()
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
