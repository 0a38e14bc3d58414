#!/usr/bin/env python
"""bench.py -- throughput of the fused MBS iteration (BASELINE.json metric) on N B200s of one node.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3|4|5] [--impl b200|reference]
    python bench.py --converge-config 3|4|5      (cold-start solve to the config's tol: seconds and iterations)

A "step" is one iteration of Eq. (6) of the paper over the whole grid: every row of
SURVEY.md 8(a) (scattering operator with edge-slab corrections, per-subdomain FFT propagator, difference,
second scattering operator, residual norm, alpha-update, stop flag).  The workload is one of the seeded
synthetic media of BASELINE.json (default: config 5, 1024^3, 4x2x2 subdomains).

Output: ONE JSON line (rank 0).  `value` = voxel-iterations/s with every input resident in HBM, timed with CUDA
events on the solver's stream, max over ranks; `e2e` = the same metric through the host-buffer entry point
mbs_solve_host (H2D of y and x0 and D2H of x inside the timed region); `roofline` = the dominant kernel's
algorithmic bytes per launch / its average event-timed duration against MEASURED_PEAKS.json; `cpu_baseline` =
the CPU oracle, as it stands, timed on a bounded sample on this box's host cores.  The default run (no --config)
times the two other 3-D configs of BASELINE.json as well (same K-step event timing) and reports them under
`other_configs`, each against the 112 B floor ledger and against its own sparse-source ledger.

Multi-GPU: the path does not shard in this build (BASELINE.json: "no sharding, no collectives"): --gpus N runs N
independent replicas ("replicas only"); value = N x voxels x K / max-over-ranks time.

`--impl reference` times the oracle (the only reference implementation that exists for this paper here).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "Gvoxel-iterations/s of fused MBS step"
UNIT = "Gvoxel-it/s"
# Oracle samples (cpu_baseline, --impl reference): config 3 itself; for configs 4 and 5 ONE subdomain of the workload in
# its real shape (same generator; the per-subdomain FFTs, the largest part of an oracle iteration, are exactly those of the
# full grid).  The full grids need 30 / 120 GiB of complex128 arrays and minutes per oracle iteration, outside the
# 10-30 s budget of this leg; `--cpu-baseline-full` times the oracle on the workload itself when the host has the memory.
SAMPLE_GRIDS = {3: ((256, 256, 256), (2, 1, 1), (16, 16, 16)),
                4: ((320, 320, 320), (1, 1, 1), (24, 24, 24)),
                5: ((256, 512, 512), (1, 1, 1), (32, 32, 32)),
                6: ((630, 315, 315), (2, 1, 1), (20, 20, 20))}
DEFAULT_STEPS = {3: 400, 4: 60, 5: 30, 6: 20}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--config", type=int, default=None, choices=(3, 4, 5, 6),
                    help="workload (default 5; without this flag configs 3 and 4 are timed too, under other_configs); "
                         "6 = the shape of the paper's own large run, 1260^3 voxels in two subdomains (context, not a BASELINE config)")
    ap.add_argument("--converge-config", type=int, default=None, choices=(3, 4, 5, 6),
                    help="only: cold-start mbs_solve of this config at its tol; prints seconds and iterations")
    ap.add_argument("--cpu-baseline-full", action="store_true",
                    help="time the oracle on the workload itself (3 iterations; config 5 needs ~120 GiB of host memory)")
    ap.add_argument("--impl", default="b200", choices=("b200", "reference"))
    ap.add_argument("--shape", default=None, help="override the grid, e.g. 256,512,1024 (profiling runs; not the headline)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-converge", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="default run: do not time configs 3 and 4 as well")
    ap.add_argument("--unfused", action="store_true", help="one kernel per step of P:122-128 instead of the fused sweeps")
    ap.add_argument("--opt", action="append", default=[], metavar="NAME=VALUE",
                    help="kernel option for profiling runs, e.g. LINE=2, LINE=0, TMA=0 (enum mbs_option; not the headline)")
    ap.add_argument("--batch", type=int, default=None, metavar="N",
                    help="only: time mbs_solve_batch with N sources sharing the medium of --config (P:23; NEXT-4) beside one source")
    ap.add_argument("--activation", type=float, default=None, metavar="THRESHOLD",
                    help="--converge-config only: solve with subdomain activation (P:139-141) at this relative threshold "
                         "(negative: the default tol / 10) and report it beside the plain solve")
    return ap.parse_args()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.samples, self.stop_flag, self.thread = index, [], threading.Event(), None

    def _run(self):
        while not self.stop_flag.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                f = [t.strip() for t in out.strip().split(",")]
                if len(f) >= 6:
                    self.samples.append(f)
            except Exception:
                pass
            self.stop_flag.wait(0.1)

    def __enter__(self):
        self.thread = threading.Thread(target=self._run, daemon=True)
        self.thread.start()
        return self

    def __exit__(self, *a):
        self.stop_flag.set()
        self.thread.join(timeout=10)

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        sm = sorted(float(s[0]) for s in self.samples)
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        reasons = [n for i, n in enumerate(names) if any(s[2 + i].lower().startswith("active") for s in self.samples)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.samples[0][1]), "reasons": reasons,
                "samples": len(sm)}


def oracle_sample(cfg, n_iter, budget_s=25.0, warmup=1, full=False):
    """Time the CPU oracle (oracle/mbs_oracle.py, as it stands) on a bounded sample of config `cfg` (SAMPLE_GRIDS), or on
    the workload itself (`full`), `n_iter` iterations of Eq. (6) at most `budget_s` seconds.  Returns a dict."""
    import dataclasses
    from paper_2410_02395_b200 import workloads
    from oracle import mbs_oracle
    if full:
        w = workloads.config(cfg)
        what = "the workload itself"
    else:
        shape, S, W = SAMPLE_GRIDS[cfg]
        w = dataclasses.replace(workloads.config(cfg, shape=shape, boundary_width=W), n_subdomains=S)
        what = ("the workload itself" if shape == workloads.config(cfg).shape else
                "one subdomain of the workload in its real shape (the full grid needs %d GiB of complex128 arrays and minutes "
                "per oracle iteration: outside this leg's budget)" % (workloads.config(cfg).voxels * 16 * 7 // 2 ** 30))
    n, y = w.make_medium(), w.make_source()
    o = mbs_oracle.from_workload(w, n)
    times = []
    t_last = [time.perf_counter()]

    def cb(i, eps, x):
        now = time.perf_counter()
        times.append(now - t_last[0])
        t_last[0] = now
        if sum(times) > budget_s:
            raise StopIteration

    t_last[0] = time.perf_counter()
    try:
        o.solve(y, tol=0.0, max_iter=n_iter, callback=cb)
    except StopIteration:
        pass
    # the first callback interval also holds the nu pre-pass: the warm-up iterations are dropped when there are more
    steady = times[warmup:] if len(times) > warmup else times[-1:]
    per_it = float(np.mean(steady))
    return {"value": w.voxels / per_it / 1e9, "unit": UNIT, "cores": mbs_oracle._workers(), "kind": "oracle",
            "sample": "cfg%d generator at %s with %s subdomains = %s; %d oracle iteration(s) timed (numpy complex128, scipy.fft)"
                      % (cfg, "x".join(map(str, w.shape)), "x".join(map(str, w.n_subdomains)), what, len(steady)),
            "ms_per_step": per_it * 1e3, "voxels": w.voxels}


def _workloads():
    from paper_2410_02395_b200 import workloads
    return workloads


def config_block(w, world):
    """The `config` object of the JSON line: the same on both arms (the driver compares them)."""
    return {"workload": workload_name(w),
            "l2": "inputs larger than L2 (%.1f GiB per array): no flush between iterations" % (w.voxels * 8 / 2 ** 30)
                  if w.voxels * 8 > 4 * 126e6 else "arrays comparable to L2; no flush (the step streams 4 arrays)",
            "parallelism": "replicas x%d (the path does not shard in this build)" % world}


def run_reference(args):
    """--impl reference: the oracle is the only reference implementation of this paper available here.  A step is one
    oracle iteration on the bounded sample of the workload (SAMPLE_GRIDS); the run stops early after 4 minutes."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = args.config or 5
    K = args.steps if args.steps is not None else 5
    W = args.warmup if args.warmup is not None else 1
    r = oracle_sample(cfg, K + W, budget_s=240.0, warmup=W, full=args.cpu_baseline_full)
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus, "steps": K,
            "warmup": W, "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "c128", "data": "synthetic",
            "config": config_block(_workloads().config(cfg), max(1, args.gpus)),
            "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def workload_name(w):
    return "%s: %s grid, %s subdomains, t=%d, W=%s, complex64, seeded synthetic medium (workloads.config)" % (
        w.name, "x".join(map(str, w.shape)), "x".join(map(str, w.n_subdomains)), w.n_correction,
        "x".join(map(str, w.boundary_width)))


TRAFFIC_SOURCE = ("dram__bytes_read.sum + dram__bytes_write.sum per voxel from the committed ncu --set full capture "
                  "(profiles/dram_traffic.json, measured on a smaller grid with the same line lengths), scaled to this "
                  "workload's voxel count; not measured in this run")


def dominant_kernel_traffic(name, voxels):
    """DRAM bytes per launch of kernel class `name`, scaled from profiles/dram_traffic.json (see TRAFFIC_SOURCE).
    None when the kernel is not in the capture."""
    path = os.path.join(ROOT, "profiles", "dram_traffic.json")
    if not os.path.exists(path):
        return None
    try:
        per_voxel = json.load(open(path))["kernels"][name]["dram_bytes_per_voxel"]
        return per_voxel * voxels
    except Exception:
        return None


def max_over_ranks(ms, device):
    """Device time of the timed region as the max over ranks (every rank gets it); identity without a process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms)
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(voxels, steps, ms, world):
    """Whole-job Gvoxel-iterations/s of `world` independent replicas that each did `steps` iterations in `ms`."""
    return world * voxels * steps / (ms * 1e-3) / 1e9


def time_config(cfg, K, W, dev, world, shape=None, unfused=False, options=()):
    """K timed iterations of Eq. (6) on BASELINE.json config `cfg` after W warm-up iterations, everything resident in
    HBM, CUDA events on the solver's stream, max over ranks.  Returns (solver, workload, y_dev, x_dev, result dict)."""
    import torch
    import torch.distributed as dist
    from paper_2410_02395_b200 import binding, workloads
    w = workloads.config(cfg, shape=shape)
    t0 = time.perf_counter()
    n_map, y = w.make_medium(), w.make_source()
    t_gen = time.perf_counter() - t0
    s = binding.Solver.from_workload(w, device=dev)
    s.set_option(binding.MBS_OPT_FUSED, 0 if unfused else 1)
    for opt, val in options:
        s.set_option(opt, val)
    nd = torch.from_numpy(n_map).to(dev)
    s.set_potential(nd)
    del nd, n_map
    yd = torch.from_numpy(y).to(dev)
    xd = torch.zeros(w.shape, dtype=torch.complex64, device=dev)
    torch.cuda.synchronize()

    # warm-up (also computes nu = ||Gamma^-1 y_vec||)
    s.iterate(yd, xd, W, nu=0.0, want_history=False)
    nu = s.info()["norm_rhs"]
    # Per-kernel event timing inside the timed region on grids that stream from HBM (an event pair per multi-ms launch
    # costs nothing there).  On grids of <= 32 M voxels the library replays CUDA graphs, which event pairs would switch
    # off: those get the kernel times from a second pass of the same K steps right after the timed one.
    profile_in_timed_region = w.voxels > (1 << 25)
    s.set_option(binding.MBS_OPT_PROFILE, 1 if profile_in_timed_region else 0)
    s.reset_kernel_stats()
    launches0 = s.info()["kernel_launches"]

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    with ClockSampler(dev.index) as clocks:
        ev0.record(s.stream)
        hist = s.iterate(yd, xd, K, nu=nu)
        ev1.record(s.stream)
        barrier()
    ms = ev0.elapsed_time(ev1)
    launches = s.info()["kernel_launches"] - launches0
    if not profile_in_timed_region:
        s.set_option(binding.MBS_OPT_PROFILE, 1)
        s.reset_kernel_stats()
        s.iterate(yd, xd, K, nu=nu, want_history=False)
    stats = s.kernel_stats()
    s.set_option(binding.MBS_OPT_PROFILE, 0)
    ms = max_over_ranks(ms, dev)
    value = aggregate_throughput(w.voxels, K, ms, world)

    peak, peak_kind = peaks()
    stats = [k for k in stats if k["launches"] > 0]
    stats.sort(key=lambda k: -k["total_ms"])
    info = s.info()
    floor_bytes = info["algorithmic_bytes_per_iteration"]            # 112 B/voxel in 3-D: the quoted denominator
    sparse_bytes = info["sparse_source_bytes_per_iteration"]          # minus the all-zero rows of y this workload skips
    per_s = K / (ms * 1e-3) / 1e9 * world
    kernels = [{"name": k["name"], "launches_per_step": k["launches"] / K, "avg_ms": k["total_ms"] / k["launches"],
                "GBps": k["algorithmic_bytes"] / max(k["total_ms"], 1e-9) / 1e6} for k in stats]
    res = {"cfg": cfg, "workload": workload_name(w), "value": value, "unit": UNIT, "steps": K, "warmup": W,
           "ms_per_step": ms / K, "gpu_launches": int(launches), "clocks": clocks.summary(),
           "residual_last": float(hist[-1]) if len(hist) else None, "medium_generation_s": t_gen,
           "whole_step": {"floor_ledger_bytes_per_voxel_iteration": floor_bytes / w.voxels,
                          "achieved": floor_bytes * per_s / world, "frac": floor_bytes * per_s / world / peak,
                          "sparse_source_ledger_bytes_per_voxel_iteration": sparse_bytes / w.voxels,
                          "achieved_sparse_source": sparse_bytes * per_s / world,
                          "frac_sparse_source": sparse_bytes * per_s / world / peak,
                          "note": "frac = floor ledger (SURVEY 8(d), the quoted denominator); frac_sparse_source = the bytes "
                                  "this workload must move (all-zero rows of y are skipped); peak = " + peak_kind},
           "kernels": kernels, "kernels_above_peak": [k["name"] for k in kernels if k["GBps"] > peak],
           "kernel_times": "CUDA events around every launch, " + ("inside the timed region" if profile_in_timed_region
                           else "second pass of the same K steps (the timed region replays CUDA graphs)"),
           "_stats": stats, "_peak": (peak, peak_kind)}
    return s, w, yd, xd, res


def primary_line(res, w, world, unfused):
    """The contract's JSON line from the result of the primary workload."""
    stats, (peak, peak_kind) = res.pop("_stats"), res.pop("_peak")
    top = stats[0]
    top_ms = top["total_ms"] / top["launches"]
    top_bytes = top["algorithmic_bytes"] / top["launches"]
    achieved = top_bytes / (top_ms * 1e-3) / 1e9
    total_kernel_ms = sum(k["total_ms"] for k in stats)
    roofline = {"bound": "hbm", "kernel": top["name"], "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": dominant_kernel_traffic(top["name"], w.voxels),
                "traffic_source": TRAFFIC_SOURCE, "peak_kind": peak_kind,
                "algorithmic_bytes_per_launch": top_bytes, "avg_launch_ms": top_ms,
                "share_of_step": top["total_ms"] / total_kernel_ms, "kernel_times": res["kernel_times"],
                "whole_step": res["whole_step"], "kernels": res["kernels"], "kernels_above_peak": res["kernels_above_peak"]}
    return {"metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": world, "steps": res["steps"],
            "warmup": res["warmup"], "ms_per_step": res["ms_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "c64", "data": "synthetic", "config": config_block(w, world),
            "run": {"fused": not unfused, "residual_last": res["residual_last"], "medium_generation_s": res["medium_generation_s"]},
            "clocks": res["clocks"], "gpu_launches": res["gpu_launches"], "roofline": roofline}


def add_e2e(s, w, y, line, K):
    """Same metric through the host-buffer entry point: H2D of y and x0, K iterations, D2H of x, every step."""
    import torch
    yh = torch.from_numpy(y).pin_memory()
    xh = torch.zeros(w.shape, dtype=torch.complex64).pin_memory()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    ev0.record(s.stream)
    s.solve_host(yh, xh, 0.0, K)
    ev1.record(s.stream)
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    ms = max(ev0.elapsed_time(ev1), wall * 1e3)
    nbytes = w.voxels * 8
    line["e2e"] = {"value": w.voxels * K / (ms * 1e-3) / 1e9, "unit": UNIT, "h2d_bytes_per_step": 2 * nbytes / K,
                   "d2h_bytes_per_step": nbytes / K, "ms_total": ms,
                   "note": "mbs_solve_host: one call = H2D(y, x0) + nu pre-pass + %d iterations + D2H(x); bytes are per iteration" % K}
    del yh, xh


def batched(cfg, n_batch, K, W, dev):
    """Throughput of mbs_solve_batch (n_batch sources, one medium) against the same solver with one source: device time of
    the iteration loop (mbs_info.last_solve_ms; the nu pre-pass is outside it), K updates after W warm-up updates."""
    import torch
    from paper_2410_02395_b200 import binding, workloads
    w = workloads.config(cfg)
    n_map, y = w.make_medium(), w.make_source()
    s = binding.Solver.from_workload(w, device=dev)
    s.set_potential(torch.from_numpy(n_map).to(dev))
    del n_map
    peak, peak_kind = peaks()
    out = {"workload": workload_name(w), "steps": K, "warmup": W, "peak": peak, "runs": []}
    for nb in (1, n_batch):
        # the sources: the config's own source shifted along axis 0 (distinct right-hand sides, same sparsity)
        ys = torch.stack([torch.from_numpy(np.roll(y, 7 * b, axis=0)) for b in range(nb)]).to(dev)
        xs = torch.zeros_like(ys)
        binding.mbs_solve_batch(s.ctx, nb, ys.data_ptr(), xs.data_ptr(), -1.0, W, want_history=False)
        rc, hist, _ = binding.mbs_solve_batch(s.ctx, nb, ys.data_ptr(), xs.data_ptr(), -1.0, K)
        ms = s.info()["last_solve_ms"]
        ledger = (96.0 + 16.0 / nb) * w.voxels * nb                 # bytes per iteration of the batch
        out["runs"].append({"n_batch": nb, "ms_per_iteration": ms / K, "Gvoxel_it_per_s": nb * w.voxels * K / (ms * 1e-3) / 1e9,
                            "ledger_bytes_per_voxel_iteration_and_source": 96.0 + 16.0 / nb,
                            "frac_of_own_ledger": ledger * K / (ms * 1e-3) / 1e9 / peak,
                            "frac_of_112B_roofline": 112.0 * w.voxels * nb * K / (ms * 1e-3) / 1e9 / peak,
                            "residual_last": float(hist[-1])})
        del ys, xs
    s.close()
    return out


def converge(cfg, dev, with_floor=True, activation=None):
    """Seconds to converge (BASELINE.json metric, second part): cold-start mbs_solve of config `cfg` at its tol, and the
    complex64 residual floor of that case (minimum eps when iterating on without a stop test)."""
    import torch
    from paper_2410_02395_b200 import binding, workloads
    w = workloads.config(cfg)
    n_map, y = w.make_medium(), w.make_source()
    s = binding.Solver.from_workload(w, device=dev)
    s.set_potential(torch.from_numpy(n_map).to(dev))
    del n_map
    if activation is not None:
        s.set_activation(True, activation)
    yd = torch.from_numpy(y).to(dev)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    x, hist, rc = s.solve(yd, tol=w.tol, max_iter=w.max_iter)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    loop_ms = s.info()["last_solve_ms"]
    out = {"workload": workload_name(w), "tol": w.tol, "seconds": dt, "iterations": int(len(hist)),
           "status": binding.STATUS_NAMES[rc], "device_loop_ms": loop_ms,
           "Gvoxel_it_per_s_over_the_solve": w.voxels * len(hist) / (loop_ms * 1e-3) / 1e9,
           "monotone": bool(np.all(np.diff(hist) <= 0.0)), "residual_final": float(hist[-1])}
    if activation is not None:
        act = s.activation()
        out["activation"] = {"threshold": activation if activation >= 0 else 0.1 * w.tol, "activated_at": act,
                             "work_fraction": sum(len(hist) - a for a in act if a >= 0) / (len(act) * len(hist)),
                             "reading": "R17 (DESIGN.md section 3); P:139-141 reports 12 % on 100^3 wavelengths, 3x1x1"}
    if with_floor:
        # complex64 floor: keep iterating without a stop test until eps stops falling (chunks of 500, at most 20 000 more)
        nu, floor, extra = s.info()["norm_rhs"], float(hist.min()), 0
        while extra < 20000:
            chunk_min = float(s.iterate(yd, x, 500, nu=nu).min())
            extra += 500
            stalled = chunk_min > 0.98 * floor
            floor = min(floor, chunk_min)
            if stalled:
                break
        out["complex64_floor"] = floor
        out["floor_iterations_after_stop"] = extra
    s.close()
    return out


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if args.batch is not None:
        if rank == 0:
            cfgb = args.config or 3
            print(json.dumps({"batched": batched(cfgb, args.batch, args.steps or DEFAULT_STEPS[cfgb], max(args.warmup or 3, 3), dev)}))
        return
    if args.converge_config is not None:
        if rank == 0:
            out = {}
            if not (args.no_converge and args.activation is not None):      # --no-converge + --activation: the activated solve only
                out["time_to_converge"] = converge(args.converge_config, dev, with_floor=args.converge_config == 3)
            if args.activation is not None:
                out["time_to_converge_with_activation"] = converge(args.converge_config, dev, with_floor=False,
                                                                   activation=args.activation)
            print(json.dumps(out))
        return
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    cfg = args.config or 5
    K = args.steps if args.steps is not None else DEFAULT_STEPS[cfg]
    W = max(args.warmup if args.warmup is not None else 3, 3)
    shape = tuple(int(v) for v in args.shape.split(",")) if args.shape else None
    from paper_2410_02395_b200 import binding as _b
    options = [(getattr(_b, "MBS_OPT_" + kv.split("=")[0].upper()), int(kv.split("=")[1])) for kv in args.opt]
    s, w, yd, xd, res = time_config(cfg, K, W, dev, world, shape=shape, unfused=args.unfused, options=options)
    line = primary_line(res, w, world, args.unfused)
    if rank == 0 and not args.no_e2e:
        y = yd.cpu().numpy()
        del xd
        xd = None
        add_e2e(s, w, y, line, K)
    s.close()
    del s, yd, xd
    torch.cuda.empty_cache()
    # the two other 3-D configs of BASELINE.json ("... >= 70 % of B200 HBM bandwidth on the 3D configs"), same timing
    if args.config is None and shape is None and not args.no_other_configs:
        others = []
        for oc in (3, 4):
            # their own window (at least 50 iterations where an iteration is short), not the primary's K
            so, wo, yo, xo, ro = time_config(oc, DEFAULT_STEPS[oc], W, dev, world)
            so.close()
            del so, yo, xo
            torch.cuda.empty_cache()
            ro.pop("_stats"), ro.pop("_peak")
            others.append(ro)
        line["other_configs"] = others
    if rank == 0:
        if not args.no_converge:
            line["time_to_converge"] = converge(3, dev)
        if not args.no_cpu_baseline and world == 1:
            r = oracle_sample(cfg, 3, full=args.cpu_baseline_full, budget_s=3600.0 if args.cpu_baseline_full else 25.0)
            line["cpu_baseline"] = {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")}
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
