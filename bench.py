#!/usr/bin/env python
"""bench.py - throughput of the Sim(3) Gauss-Newton step (libsim3ba) on synthetic graphs shaped like
BASELINE.json's configs.  One "step" = one pass of the whole hot path (a1-a8: per-match residual /
Jacobian, block reduction, assembly, Cholesky solve, retraction) over the workload's graph.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]

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
        """Statistics over the samples that arrived in [t0, t1] (all samples if none did: a region shorter than the period)."""
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
    s = g.spec
    return {"workload": f"BASELINE configs[{cfg_id - 1}] {s.name}: {g.n_kf} keyframes {s.width}x{s.height}, "
                        f"{g.n_edges} edges, {int(s.p_out * 100)}% outlier matches, preset sigma=1 kappa=0.05",
            "n_kf": g.n_kf, "hw": g.hw, "n_edges": g.n_edges, "system_n": 7 * g.n_kf,
            "candidates_per_step": int(g.n_edges) * int(g.hw), "gn_iters_per_pose_reset": s.n_iters}


def run_ours(args):
    import numpy as np
    import torch
    from sim3ba_inputs import PRESETS, make_config
    from paper_2605_30488_b200 import Sim3BA, build, make_params

    rank, world, local = dist_setup(args.gpus)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (libsim3ba has no CPU fallback)")
    build.build()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)

    g = make_config(args.config)                 # replicas only: every rank owns an independent graph
    preset = PRESETS["config"]
    # inputs start in pinned host memory; the graph upload is the one-off part of the end-to-end job
    h_pts, h_cf = torch.from_numpy(g.points).pin_memory(), torch.from_numpy(g.conf).pin_memory()
    h_ed, h_mt = torch.from_numpy(g.edges).pin_memory(), torch.from_numpy(g.match).pin_memory()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    d_pts, d_cf = h_pts.to(dev, non_blocking=True), h_cf.to(dev, non_blocking=True)
    d_ed, d_mt = h_ed.to(dev, non_blocking=True), h_mt.to(dev, non_blocking=True)
    ba = Sim3BA(d_pts, d_cf, d_ed, d_mt, g.fixed_kf, make_params(**preset), g.spec.height, g.spec.width)
    torch.cuda.synchronize()
    upload_ms = (time.perf_counter() - t0) * 1e3
    upload_bytes = sum(t.numel() * t.element_size() for t in (h_pts, h_cf, h_ed, h_mt))

    poses0 = torch.from_numpy(g.poses_init).to(dev)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)   # > 126 MB L2
    n_reset = max(1, g.spec.n_iters)

    def one_pass(n_steps, timed):
        """n_steps GN iterations; poses reset to the seeded start every n_reset steps (untimed)."""
        total_ms = 0.0
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for s in range(n_steps):
            if s % n_reset == 0:
                ba.set_poses(poses0)
            flush.fill_(s & 0xFF)                 # L2 flush between timed iterations (untimed)
            torch.cuda.synchronize()
            ev0.record()
            ba.step()
            ev1.record()
            torch.cuda.synchronize()
            if timed:
                total_ms += ev0.elapsed_time(ev1)
        return total_ms

    # units per step: valid correspondences (counted by the library itself on the first step)
    ba.set_poses(poses0)
    ba.step()
    torch.cuda.synchronize()
    n_valid = int(ba.edge_stats()[0].sum().item())

    sampler = ClockSampler(local)
    sampler.start()                               # nvidia-smi needs a few hundred ms to come up: started before the warm-up
    one_pass(args.warmup, timed=False)
    t_up = time.perf_counter()
    while sampler.proc is not None and len(sampler.rows) < 2 and time.perf_counter() - t_up < 5.0:
        one_pass(20, timed=False)                 # same load, untimed, until the sampler delivers
    barrier()
    torch.cuda.synchronize()
    t_begin = sampler.mark()
    l0 = ba.launch_count()
    total_ms = one_pass(args.steps, timed=True)
    l1 = ba.launch_count()
    torch.cuda.synchronize()
    t_end = sampler.mark()
    barrier()
    clocks = sampler.stop(t_begin, t_end)
    ms_per_step = total_ms / args.steps

    # end to end through the C ABI with HOST buffers (pinned): sim3ba_optimize_host = device allocation + upload of the
    # whole graph (points, confidences, edges, match maps) + create (pack, bookkeeping, solve plan) + n_iters GN steps
    # + poses and costs back + free.  One job = the config's n_iters steps; per-step figures divide by n_iters.
    from paper_2605_30488_b200 import optimize_host
    n_it = max(1, g.spec.n_iters)
    h_in = torch.from_numpy(g.poses_init.copy()).pin_memory()
    h_out = torch.empty((g.n_kf, 8), dtype=torch.float64).pin_memory()
    h_cost = torch.empty((n_it,), dtype=torch.float64).pin_memory()
    st = torch.cuda.current_stream().cuda_stream

    def e2e_job():
        optimize_host(h_pts, h_cf, h_ed, h_mt, g.fixed_kf, make_params(**preset), g.spec.height, g.spec.width,
                      h_in, n_it, h_out, h_cost, st)

    e2e_job()                                         # two warm-up jobs (allocator, page tables)
    e2e_job()
    n_jobs = max(1, min(args.steps // n_it, 10))
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    torch.cuda.synchronize()
    w0 = time.perf_counter()
    ev0.record()
    for _ in range(n_jobs):
        e2e_job()
    ev1.record()
    torch.cuda.synchronize()
    e2e_wall_ms = (time.perf_counter() - w0) * 1e3
    e2e_ms = max(ev0.elapsed_time(ev1), e2e_wall_ms) / (n_jobs * n_it)
    e2e_h2d = (upload_bytes + g.n_kf * 64) / n_it
    e2e_d2h = (g.n_kf * 64 + 8 * n_it) / n_it

    # per-kernel device times (CUDA events recorded by the library on its stream), same loop
    ba.set_profiling(True)
    ph = []
    for s in range(args.steps):
        if s % n_reset == 0:
            ba.set_poses(poses0)
        flush.fill_(s & 0xFF)
        torch.cuda.synchronize()
        ba.step()
        ph.append(ba.phase_ms())
    ba.set_profiling(False)
    ph = np.asarray(ph)[:, :5].mean(axis=0)

    depth = None
    if args.depth:   # NEXT-1: one structure pass (segment log-depth refinement, poses fixed) timed beside the pose step
        from sim3ba_inputs import make_depth_inputs
        d = make_depth_inputs(g)
        labels = torch.from_numpy(d.labels).to(dev)
        eta = torch.zeros(g.n_kf * d.n_seg, dtype=torch.float64, device=dev)
        ba.set_poses(poses0)
        ba.depth_refine(labels, d.n_seg, d.pairs, d.delta, d.anchor_kf, eta, 1)          # warm-up (allocations)
        n_dit = 10
        eta.zero_()
        torch.cuda.synchronize()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        costs = ba.depth_refine(labels, d.n_seg, d.pairs, d.delta, d.anchor_kf, eta, n_dit)
        ev1.record()
        torch.cuda.synchronize()
        depth = {"what": "sim3ba_depth_refine, 10 iterations (PAPER.md:143), poses fixed at the seeded start",
                 "segments_per_kf": d.n_seg, "ms_per_iteration": ev0.elapsed_time(ev1) / n_dit,
                 "objective_first_last": [float(costs[0]), float(costs[-1])]}

    job_ms, job_units = aggregate_over_ranks(ms_per_step, float(n_valid), dev)
    e2e_job_ms, _ = aggregate_over_ranks(e2e_ms, float(n_valid), dev)
    if rank != 0:
        return
    hbm_peak, peak_src = load_peaks()
    n_sms = torch.cuda.get_device_properties(dev).multi_processor_count
    sm_max_mhz = float(clocks.get("sm_max_mhz") or 1965.0)
    cand = g.n_edges * g.hw
    bytes_min = 4.0 * cand + 16.0 * g.n_kf * g.hw          # unique bytes: every index + every packed pixel once
    bytes_stream = 36.0 * cand                              # no-reuse accounting (4 idx + 16 X_i + 16 X_j)
    k1_s = float(ph[0]) * 1e-3
    out = {
        "metric": METRIC, "value": job_units / (job_ms * 1e-3), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": job_ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32 per-match, f64 reduce/solve", "data": "synthetic",
        "config": dict(workload_description(g, args.config), l2="flushed between timed steps (256 MB write)",
                       valid_per_step=n_valid, graph_upload_ms=upload_ms, graph_upload_bytes=upload_bytes,
                       multi_gpu="replicas only (independent graph per rank, no collective)"),
        "clocks": clocks,
        "e2e": {"value": job_units / (e2e_job_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_job_ms,
                "h2d_bytes_per_step": e2e_h2d, "d2h_bytes_per_step": e2e_d2h, "jobs": n_jobs, "steps_per_job": n_it,
                "what": "sim3ba_optimize_host: device allocation + upload of the whole graph from pinned host memory "
                        "+ create + n_iters GN steps + poses and costs back + free; per step = job / n_iters"},
        "gpu_launches": int(l1 - l0),
        "phases_ms": {"k1_accumulate": float(ph[0]), "k2_edge_reduce_gradient": float(ph[1]),
                      "k3_assemble": float(ph[2]), "k4_factor_solve": float(ph[3]), "k5_retract": float(ph[4])},
        "candidates_per_s": cand * world / (job_ms * 1e-3),
        "roofline": {"bound": "hbm", "kernel": "k_accumulate", "achieved": bytes_min / k1_s / 1e9,
                     "peak": hbm_peak, "unit": "GB/s", "frac": bytes_min / k1_s / 1e9 / hbm_peak,
                     "traffic": load_traffic(args.config), "peak_source": peak_src,
                     "algorithmic_bytes_per_launch": bytes_min,
                     "achieved_stream_accounting": bytes_stream / k1_s / 1e9,
                     "frac_stream_accounting": bytes_stream / k1_s / 1e9 / hbm_peak,
                     "note": "kernel 1 sits on the ridge: HBM traffic equals the unique bytes (ncu), the binding resource "
                             "is fp32 issue (see roofline_alu and profiles/)"},
        # the same kernel against the plain-ALU roof: 300 fp32 flop per valid match (FMA = 2),
        # peak = SMs x 128 fp32 lanes x 2 x max SM clock
        "roofline_alu": {"bound": "alu", "kernel": "k_accumulate", "achieved": 300.0 * n_valid / k1_s / 1e12,
                         "peak": n_sms * 128 * 2 * sm_max_mhz * 1e6 / 1e12, "unit": "TFLOP/s",
                         "frac": 300.0 * n_valid / k1_s / (n_sms * 128 * 2 * sm_max_mhz * 1e6),
                         "flop_per_valid_match": 300.0},
        "solver": dict(ba.bb_info(), mode="band + border block Cholesky (2)" if ba.bb_info()["valid"] else "tile-sparse (0)",
                       dense_equivalent_tflops=(7.0 * g.n_kf) ** 3 / 3.0 / (float(ph[3]) * 1e-3) / 1e12),
    }
    if depth is not None:
        out["depth_refine"] = depth
    if world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(g, preset, budget_s=20.0)
    print(json.dumps(out))


# ------------------------------------------------------------------------------------------------
def oracle_rate(g, preset):
    """Candidates per second of the oracle on this host, from a short probe (the first pixels of edge 0)."""
    px = min(g.hw, 16384)
    time_oracle_step(g, preset, [0], px)
    dt, _ = time_oracle_step(g, preset, [0], px)
    return px / max(dt, 1e-6)


def oracle_sample(g, budget_s, rate):
    """Bounded sample of the workload for the CPU oracle: the first edges whose work fits the budget, or -- when not even one
    edge fits -- the first pixels of edge 0.  Returns (edge list, pixel limit or None)."""
    per_edge_s = g.hw / rate
    if budget_s >= per_edge_s:
        return list(range(max(1, min(g.n_edges, int(budget_s / per_edge_s))))), None
    return [0], max(1024, int(budget_s * rate))


def time_oracle_step(g, preset, edges_sample, px_limit=None):
    """One oracle GN iteration restricted to a sample of edges (and pixels): assemble, solve, retract."""
    import numpy as np
    from oracle import sim3_gn_oracle as orc
    prm = orc.Params(**preset)
    match = g.match
    if px_limit is not None:
        match = g.match[:max(edges_sample) + 1].copy()
        match[:, px_limit:] = -1
    t0 = time.perf_counter()
    sysm = orc.build_system(g.poses_init, g.points, g.conf, g.edges, match, prm, edge_subset=edges_sample)
    partial = len(edges_sample) < g.n_edges or px_limit is not None
    sol = orc.solve(sysm.H + 1e-3 * np.eye(sysm.H.shape[0]) * partial, sysm.g, g.fixed_kf, prm)
    orc.retract(g.poses_init, sol.tau)
    dt = time.perf_counter() - t0
    return dt, int(sysm.n_valid.sum())


def cpu_baseline(g, preset, budget_s=20.0):
    from threadpoolctl import threadpool_limits
    with threadpool_limits(limits=1):
        sample, px = oracle_sample(g, budget_s, oracle_rate(g, preset))
        dt, n_valid = time_oracle_step(g, preset, sample, px)
    return {"value": n_valid / dt, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": dt,
            "sample": f"oracle/sim3_gn_oracle.py, one GN iteration over edges 0..{len(sample) - 1} of "
                      f"{g.n_edges} ({n_valid} valid correspondences), BLAS limited to 1 thread"}


def run_reference(args):
    """The reference arm of this tier is the oracle, as it stands, on the host cores."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from threadpoolctl import threadpool_limits
    from sim3ba_inputs import PRESETS, make_config
    g = make_config(args.config)
    preset = PRESETS["config"]
    # bounded sample per step so that the whole --steps K --warmup W run ends within a couple of minutes
    with threadpool_limits(limits=1):
        sample, px = oracle_sample(g, min(3.0, max(0.05, 100.0 / max(1, args.steps + args.warmup))), oracle_rate(g, preset))
        for _ in range(args.warmup):
            time_oracle_step(g, preset, sample, px)
        tot, units = 0.0, 0
        for _ in range(args.steps):
            dt, nv = time_oracle_step(g, preset, sample, px)
            tot += dt
            units += nv
    val = units / tot
    desc = (f"oracle/sim3_gn_oracle.py, each step = one GN iteration over edges 0..{len(sample) - 1} of "
            f"{g.n_edges}" + (f", first {px} pixels" if px is not None else "") + ", BLAS limited to 1 thread")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": tot / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": workload_description(g, args.config),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--depth", action="store_true", help="also time the segment log-depth refinement (NEXT-1)")
    ap.add_argument("--no-cpu-baseline", action="store_true",
                    help="skip the oracle timing leg (profiling runs under ncu; never for a reported line)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
