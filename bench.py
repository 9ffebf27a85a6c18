#!/usr/bin/env python
"""bench.py - throughput of the SPD hot path (arXiv:1910.08324) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload 3]

One "step" = one pass of the whole hot path over one
synthetic plane: spd_run (stage, mean removal, partial-sum tree, SNR, max/arg-max, store)
followed by spd_find_candidates (threshold + peak list).  The default workload is
BASELINE.json configs[2] ("SKA-MID-like", 4096 x 1,048,576 float32, widths {2^i <= 8192}),
the configuration north_star's target is quoted on.  Prints ONE JSON line on rank 0.

Multi-GPU: the path needs no exchange; under torchrun every rank
runs the same per-GPU workload on its own DM trials (weak scaling, no data-path collective).

--impl reference times the CPU oracle (oracle/, as it stands) on the host cores on a bounded
sample of the same workload; it is a deliberately slow program, reported for context.
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

METRIC = "dm_time_samples_per_s"
UNIT = "samples/s"
BYTES_PER_SAMPLE = 12  # 4 read x + 4 write SNR + 4 write int32 width index
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback
PAPER_SKA_SAMPLES_PER_S = 6000 * 15625  # "SKA-like" real-time load: 6000 DM trials/s at 64 us


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", type=int, default=3, help="BASELINE.json config number (1-based)")
    ap.add_argument("--n-dm", type=int, default=0, help="override the number of DM trials (debugging)")
    ap.add_argument("--width-set", default="", help="override the workload's width set, e.g. IGRID:1 "
                    "(widths 2^k and 3*2^m, the paper's IG(1) set) - not the BASELINE configuration")
    ap.add_argument("--grid", default="", help="boxcar separation per width (SURVEY.md sec. 8(f2)): BOXDIT:<L_max>, "
                    "DIT or IGRID:<layers>; the width set is then evaluated on the paper's decimated grid")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config legs (the other BASELINE "
                    "configs and the IG(1) width set, measured in the same run at N = 1)")
    ap.add_argument("--per-config-steps", type=int, default=5)
    ap.add_argument("--width-u8", action="store_true", help="uint8 width index (SPD_FLAG_WIDTH_U8): 9 B per sample")
    ap.add_argument("--no-aux", action="store_true", help="skip the timings outside the step (row statistics, sigma "
                    "per width, 2-D peak stage): a short launch list for profiling")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target duration of the oracle sample")
    return ap.parse_args()


def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), \
        int(os.environ.get("WORLD_SIZE", "1"))


def rank_workload(w, rank):
    """Weak scaling: every rank holds its own n_dm DM trials of the same recipe (its own seed);
    DM trials are independent, so there is no data-path exchange."""
    from dataclasses import replace
    return replace(w, seed=w.seed + 1000003 * rank)


def max_over_ranks(ms, device=None):
    """Device-timed milliseconds -> max over the ranks of the job (identity without a process group)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms)
    t = torch.tensor([ms], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world, samples_per_rank, ms_per_step):
    """DM-time samples/s of the whole job: all ranks' samples over the slowest rank's step time."""
    return world * samples_per_rank / (ms_per_step * 1e-3)


def workload_config(w, widths, extra=None):
    cfg = {
        "workload": f"configs[{w.index - 1}] {w.name}: {w.n_dm} DM trials x {w.n_t} samples float32 per GPU",
        "n_dm": w.n_dm, "n_t": w.n_t,
        "width_set": f"{w.width_kind}<= {w.max_width} ({len(widths)} widths, every sample)",
        "max_width": w.max_width, "sampling_time_s": w.sampling_time_s,
        "n_pulses": w.n_pulses, "seed": w.seed,
        "l2": "inputs larger than L2 (plane and outputs are each >= 8 GiB; no flush needed)"
        if w.n_samples * 4 > (1 << 30) else "plane fits L2: rotating buffers larger than L2",
    }
    if extra:
        cfg.update(extra)
    if cfg.get("grid"):
        cfg["width_set"] = cfg["width_set"].replace("every sample", "on the grid below")
    return cfg


# ----------------------------------------------------------------------------------------
# CPU oracle legs (cpu_baseline of the b200 arm; the whole of --impl reference)
# ----------------------------------------------------------------------------------------
def oracle_sample_plan(w, widths, target_s):
    """Pick rows x samples of the workload so that the direct-summation oracle takes about
    target_s seconds: calibrate on a small window first."""
    import numpy as np
    import oracle
    from workloads import make_plane_numpy
    oracle.build()
    cores = oracle.num_threads()
    n_t = min(w.n_t, 1 << 20)
    rows = max(1, min(w.n_dm, cores))
    sub = w.scaled(rows, n_t, max(1, min(w.n_pulses, rows)))
    x, _ = make_plane_numpy(sub)
    cal = min(n_t - w.max_width, 4096 * max(1, 64 // max(1, len(widths))))
    cal = max(256, min(cal, 1 << 16))
    t = time.perf_counter()
    oracle.spd_direct(x, 0.0, 1.0, widths, 0, cal)
    dt = max(time.perf_counter() - t, 1e-4)
    rate = rows * cal / dt
    span = int(min(n_t, max(cal, rate * target_s / rows)))
    return x, rows, span, cores


def time_oracle(w, widths, target_s, steps=1, warmup=0, seps=None):
    import numpy as np
    import oracle
    if seps is not None:
        return time_oracle_grid(w, widths, seps, target_s, steps, warmup)
    x, rows, span, cores = oracle_sample_plan(w, widths, target_s / max(1, steps + warmup))
    times = []
    for i in range(warmup + steps):
        t = time.perf_counter()
        oracle.spd_direct(x, 0.0, 1.0, widths, 0, span)
        dt = time.perf_counter() - t
        if i >= warmup:
            times.append(dt)
    n = rows * span
    direct = n * len(times) / sum(times)
    t = time.perf_counter()
    oracle.spd_prefix(x, 0.0, 1.0, widths)
    prefix = x.size / (time.perf_counter() - t)
    sample = (f"oracle_spd_direct (double, direct summation, OpenMP) on the first {span} samples of {rows} rows "
              f"of the same recipe ({n} samples per step); prefix_value = oracle_spd_prefix on {rows} x {x.shape[1]}")
    return {"value": direct, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
            "prefix_value": prefix, "ms_per_step": 1e3 * sum(times) / len(times), "samples_per_step": n}


def time_oracle_grid(w, widths, seps, target_s, steps, warmup):
    """cpu_baseline / reference arm of a --grid run: oracle_spd_grid on a bounded sample."""
    import oracle
    from workloads import make_plane_numpy
    oracle.build()
    cores = oracle.num_threads()
    n_t = min(w.n_t, 1 << 18)
    rows = max(1, min(w.n_dm, cores))
    x, _ = make_plane_numpy(w.scaled(rows, n_t, max(1, min(w.n_pulses, rows))))
    cal = 4096
    t = time.perf_counter()
    oracle.spd_grid(x, 0.0, 1.0, widths, seps, 0, cal)
    rate = rows * cal / max(time.perf_counter() - t, 1e-4)
    span = int(min(n_t - w.max_width, max(cal, rate * target_s / max(1, steps + warmup) / rows))) // 4096 * 4096
    times = []
    for i in range(warmup + steps):
        t = time.perf_counter()
        oracle.spd_grid(x, 0.0, 1.0, widths, seps, 0, span)
        if i >= warmup:
            times.append(time.perf_counter() - t)
    n = rows * span
    return {"value": n * len(times) / sum(times), "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"oracle_spd_grid (double, direct summation on the grid, OpenMP) on the first {span} samples of "
                      f"{rows} rows of the same recipe ({n} samples per step)",
            "ms_per_step": 1e3 * sum(times) / len(times), "samples_per_step": n}


def grid_separations(args, widths):
    """Separations of --grid from the oracle's formula module (CPU legs only)."""
    if not args.grid:
        return None
    from oracle import formulas
    kind, _, param = args.grid.partition(":")
    kind, param = kind.upper(), int(param or 0)
    sep = {"BOXDIT": lambda: formulas.boxdit_separation(param), "DIT": lambda: (lambda L: L),
           "IGRID": lambda: formulas.igrid_separation(param)}[kind]()
    return [sep(int(L)) for L in widths]


def oracle_widths(w):
    from oracle import formulas
    return formulas.width_set(w.width_kind, w.width_param, w.max_width)


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    from workloads import get_workload
    w = apply_overrides(get_workload(args.workload), args)
    widths = oracle_widths(w)
    # bounded: the whole --steps/--warmup run is sized to about 4 * cpu_seconds
    res = time_oracle(w, widths, 4.0 * args.cpu_seconds, steps=args.steps, warmup=args.warmup,
                      seps=grid_separations(args, widths))
    line = {
        "impl": "reference", "metric": METRIC, "value": res["value"], "unit": UNIT,
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": res["ms_per_step"], "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(w, widths, {"sample_per_step": res["sample"],
                                              **({"grid": args.grid} if args.grid else {})}),
        "cpu_baseline": {"value": res["value"], "unit": UNIT, "cores": res["cores"], "kind": "oracle",
                         "sample": res["sample"]},
        "e2e": {"value": res["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
        "real_time_factor_ska_like": res["value"] / PAPER_SKA_SAMPLES_PER_S,
    }
    print(json.dumps(line), flush=True)
    return 0


# ----------------------------------------------------------------------------------------
# clocks sampling (the profiling recipe's clocks line) during the timed region
# ----------------------------------------------------------------------------------------
class ClockSampler:
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.rows = []
        self.proc = None
        self.gpu_index = gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.gpu_index), f"--query-gpu={self.QUERY}",
                 "--format=csv,noheader,nounits", "-lms", "50"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        inside = [r for (t, r) in self.rows if t0 <= t <= t1 + 0.06] or [r for (_, r) in self.rows[-3:]]
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in inside:
            f = [v.strip() for v in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
                pw.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def measured_sm_mhz():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["sm_max_mhz"])
    except (OSError, KeyError, ValueError):
        return 1965.0


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
    except (OSError, KeyError, ValueError):
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ----------------------------------------------------------------------------------------
# the B200 arm
# ----------------------------------------------------------------------------------------
KERNEL_NAMES = {"tree_ws": "spd_tree_ws_kernel", "tree_block": "spd_tree_kernel", "tree_ig": "spd_tree_ig_kernel",
                "tree_ws_ig": "spd_tree_ws_kernel (IGRID depth-1 widths)",
                "grid_ws": "spd_tree_ws_kernel (grid)", "grid_tile": "grid_tile_kernel", "generic": "generic_tile_kernel",
                "dense": "spd_dense_kernel (max_width <= 64)",
                "boxdit": "spd_boxdit_kernel (Alg. 1, all iterations in one block)"}


def kernel_key(spd, info):
    if info["path"] == spd.SPD_PATH_DYADIC_TREE:
        return "tree_ws" if info["tree_kernel"] == 2 else "tree_block"
    if info["path"] == spd.SPD_PATH_IGRID_TREE:
        return "tree_ws_ig" if info["tree_kernel"] == 2 else "tree_ig"
    if info["path"] == spd.SPD_PATH_GRID:
        if info["tree_kernel"] == 2:
            return "grid_ws"
        return "boxdit" if info["threads_per_block"] == 256 else "grid_tile"   # the tile kernel runs 1024 threads
    return "dense" if info["threads_per_block"] == 256 else "generic"   # the tile kernel runs 1024 threads


class Workbench:
    """One workload resident on the device: plane, statistics, outputs, plan; step() runs the hot path once."""

    def __init__(self, spd, torch, w, dev, grid="", width_u8=False):
        from workloads import make_plane_torch
        self.spd, self.torch, self.w, self.dev = spd, torch, w, dev
        self.widths = spd.spd_width_set_generate(w.width_kind, w.width_param, w.max_width)
        self.n = w.n_samples
        self.plane, self.pulses = make_plane_torch(w, dev)
        self.mean = torch.zeros(w.n_dm, dtype=torch.float32, device=dev)
        self.sigma = torch.ones(w.n_dm, dtype=torch.float32, device=dev)
        self.thr = w.candidate_threshold if w.candidate_threshold is not None else 6.0
        self.cap = 1 << 22
        seps = None
        if grid:
            gkind, _, gparam = grid.partition(":")
            seps = spd.spd_separation_generate(gkind, int(gparam or 0), self.widths)
        flags = spd.SPD_FLAG_WIDTH_U8 if width_u8 else 0
        self.plan = spd.Plan(w.n_dm, w.n_t, self.widths, w.max_width, flags=flags, separations=seps)
        self.info = self.plan.info
        self.bytes_per_sample = 8 + self.info["width_bytes"]
        self.out_snr = torch.empty((w.n_dm, w.n_t), dtype=torch.float32, device=dev)
        self.out_width = torch.empty((w.n_dm, w.n_t), dtype=torch.uint8 if width_u8 else torch.int32, device=dev)
        # Per-DM mu, sigma: supplied (0, 1) by the config, or measured (reading A6) by spd_row_stats.
        if w.stats == "measured":
            self.plan.row_stats(self.plane, 0.0, 0, self.mean, self.sigma)
        self.activity = torch.empty(self.info["activity_bytes"], dtype=torch.uint8, device=dev)
        self.cand_list = torch.empty(self.cap * 16, dtype=torch.uint8, device=dev)
        self.cand_count = torch.zeros(1, dtype=torch.int64, device=dev)
        # planes smaller than L2 would be re-read from cache: flush between steps
        self.flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if 3 * self.n * 4 <= (512 << 20) else None
        self.stream = torch.cuda.current_stream()

    def step(self, ev=None):
        if self.flush is not None:
            self.flush.fill_(1)
        if ev is not None:
            ev[0].record(self.stream)
        self.plan.run_flagged(self.plane, self.mean, self.sigma, self.thr, self.out_snr, self.out_width, self.activity)
        if ev is not None:
            ev[1].record(self.stream)
        lst, n_found = self.plan.find_candidates_flagged(self.out_snr, self.out_width, self.activity, self.thr,
                                                         self.cap, lst=self.cand_list, n_found=self.cand_count)
        if ev is not None:
            ev[2].record(self.stream)
        return lst, n_found

    def timed(self, fn, reps=1):
        """Device time of fn() in ms (CUDA events on the launching stream, one untimed call first)."""
        torch = self.torch
        fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(self.stream)
        for _ in range(reps):
            fn()
        e1.record(self.stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    def run_steps(self, steps, warmup, barrier=None, sampler=None):
        """W warm-up steps, then exactly `steps` timed ones between barriers; returns the step record."""
        torch = self.torch
        barrier = barrier or torch.cuda.synchronize
        for _ in range(max(warmup, 0)):
            self.step()
        barrier()
        if sampler is not None:
            sampler.start()
            time.sleep(0.15)
        evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
        e_beg, e_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        t0 = time.perf_counter()
        e_beg.record(self.stream)
        n_found = None
        for i in range(steps):
            _, n_found = self.step(evs[i])
        e_end.record(self.stream)
        barrier()
        t1 = time.perf_counter()
        clocks = sampler.stop(t0, t1) if sampler is not None else None
        total_ms = e_beg.elapsed_time(e_end)
        run_ms = [e[0].elapsed_time(e[1]) for e in evs]
        cand_ms = [e[1].elapsed_time(e[2]) for e in evs]
        flush_ms = 0.0
        if self.flush is not None:  # the flush is not part of the path: take it out of the step time
            flush_ms = (total_ms - sum(run_ms) - sum(cand_ms)) / steps
            total_ms = sum(run_ms) + sum(cand_ms)
        return {"total_ms": total_ms, "run_ms": run_ms, "cand_ms": cand_ms, "flush_ms": flush_ms, "clocks": clocks,
                "n_cand": int(n_found.item())}

    def roofline(self, rec, peak, peak_src):
        k_ms = sum(rec["run_ms"]) / len(rec["run_ms"])
        achieved = self.bytes_per_sample * self.n / (k_ms * 1e-3) / 1e9
        key = kernel_key(self.spd, self.info)
        traffic, traffic_src, cap = ncu_traffic_bytes(key, self.w, self.info["width_bytes"])
        alu = None
        if cap:
            # The tree kernels are bound by their half-rate ALU-pipe instructions (width tags, 3-input maxima):
            # busy time of that pipe per sample from the committed capture, scaled to this launch; `ceiling` is
            # what the kernels' instruction mix reaches in a register-only microbenchmark
            # (profiles/r02_lane_rates.md: 12 of 15.7 clocks).
            busy_ms = cap["alu_pipe_pct"] / 100.0 * cap["kernel_ms"] * self.n / cap["samples"]
            alu = {"bound": "alu", "what": "half-rate ALU pipe (LOP3 width tags, FMNMX3 running maxima)",
                   "alu_pipe_busy_ms_per_launch": busy_ms, "frac": busy_ms / k_ms, "ceiling": 0.76,
                   "fma_pipe_busy_frac_in_capture": cap["fma_pipe_pct"] / 100.0, "source": traffic_src}
        return {
            "bound": "hbm", "kernel": KERNEL_NAMES[key], "achieved": achieved, "peak": peak, "unit": "GB/s",
            "frac": achieved / peak, "peak_source": peak_src, "traffic": traffic, "traffic_source": traffic_src,
            "algorithmic_bytes_per_launch": self.bytes_per_sample * self.n, "bytes_per_sample": self.bytes_per_sample,
            "kernel_ms": k_ms, "kernel_ms_min": min(rec["run_ms"]),
            "kernel_ms_each": [round(v, 3) for v in rec["run_ms"]],
            "candidates_ms": sum(rec["cand_ms"]) / len(rec["cand_ms"]),
            "kernel_share_of_step": sum(rec["run_ms"]) / (sum(rec["run_ms"]) + sum(rec["cand_ms"])),
            "co_bound": alu,
        }

    def close(self):
        self.plan.close()
        for name in ("plane", "out_snr", "out_width", "activity", "cand_list", "flush"):
            setattr(self, name, None)
        self.torch.cuda.empty_cache()


def per_config_legs(args, spd, torch, dev, peak, peak_src, uuid, local_rank):
    """The other BASELINE configs and the paper's IG(1) width set, measured in this same run (N = 1):
    the same step, fewer repetitions, each with its own clock record."""
    from dataclasses import replace
    from workloads import get_workload
    legs = [(f"configs[{c - 1}]", get_workload(c), "") for c in (1, 2, 3, 4, 5) if c != args.workload]
    ig = replace(get_workload(3), width_kind="IGRID", width_param=1)
    legs.append(("configs[2] with the IG(1) width set (26 widths 2^k and 3*2^m, PAPER.md:364-387)", ig, ""))
    legs.append(("configs[2] on the DIT grid (Alg. 3, PAPER.md:311)", get_workload(3), "DIT"))
    legs.append(("configs[2], IG(1) widths on 4 layers (PAPER.md:356)", ig, "IGRID:4"))
    legs.append(("configs[2], BoxDIT L_max = 8 (Alg. 1, eq. 14)",
                 replace(get_workload(3), width_kind="BOXDIT", width_param=8), "BOXDIT:8"))
    out = []
    for name, w, grid in legs:
        free, _ = torch.cuda.mem_get_info(dev)
        if free < 13 * w.n_samples + (4 << 30):
            out.append({"workload": name, "skipped": f"needs {(13 * w.n_samples) >> 30} GiB of device memory"})
            continue
        wb = Workbench(spd, torch, w, dev, grid=grid)
        rec = wb.run_steps(args.per_config_steps, 3, sampler=ClockSampler(uuid if uuid else local_rank))
        rf = wb.roofline(rec, peak, peak_src)
        ms = rec["total_ms"] / args.per_config_steps
        out.append({"workload": name, "n_dm": w.n_dm, "n_t": w.n_t, "n_widths": len(wb.widths),
                    "width_set": f"{w.width_kind}<= {w.max_width}", "grid": grid or "every sample",
                    "steps": args.per_config_steps, "ms_per_step": ms, "value": wb.n / (ms * 1e-3), "unit": UNIT,
                    "kernel": rf["kernel"], "kernel_ms": rf["kernel_ms"], "kernel_ms_min": rf["kernel_ms_min"],
                    "frac": rf["frac"], "achieved_gbs": rf["achieved"], "candidates_ms": rf["candidates_ms"],
                    "candidates_found": rec["n_cand"], "clocks": rec["clocks"],
                    **({"l2_flush_ms_per_step_excluded": rec["flush_ms"]} if wb.flush is not None else {})})
        wb.close()
        del wb
    return out


def run_b200(args):
    import torch
    import paper_1910_08324_b200 as spd
    from workloads import get_workload

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device - the SPD path has no CPU fallback (use --impl reference "
                         "for the oracle timing)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    distributed = world > 1
    if distributed:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    spd.build()
    w = apply_overrides(get_workload(args.workload), args)
    if args.n_dm:
        w = w.scaled(args.n_dm, w.n_t)
    # weak scaling: every rank holds its own n_dm DM trials (different seed per rank)
    wb = Workbench(spd, torch, rank_workload(w, rank), dev, grid=args.grid, width_u8=args.width_u8)
    plan, info, widths, n = wb.plan, wb.info, wb.widths, wb.n

    # The step before the hot path: timed on its own, outside the step.
    stats_ms = conv_ms = conv_passes = wsig_ms = run_sw_ms = None
    if not args.no_aux:
        s_mean, s_sigma = torch.empty_like(wb.mean), torch.empty_like(wb.sigma)
        stats_ms = wb.timed(lambda: plan.row_stats(wb.plane, 2.0, 2, s_mean, s_sigma))
        n_pass = torch.empty(w.n_dm, dtype=torch.int32, device=dev)
        conv_ms = wb.timed(lambda: plan.row_stats_converge(wb.plane, 2.0, 32, 1e-4, s_mean, s_sigma, n_pass))
        conv_passes = float(n_pass.float().mean().item())
        plan.row_stats(wb.plane, 2.0, 2, s_mean, s_sigma)
        # sigma per width from power-of-two decimations (row f1): one more read of the plane
        sw = plan.width_sigma(wb.plane, s_mean)
        wsig_ms = wb.timed(lambda: plan.width_sigma(wb.plane, s_mean, sw))
        # the same pass with the measured sigma per width in place of eq. (5) (where the plan's kernels take it)
        if not args.width_u8:
            try:
                run_sw_ms = wb.timed(lambda: plan.run_sigma_w(wb.plane, s_mean, sw, wb.out_snr, wb.out_width))
            except spd.SpdError:
                run_sw_ms = None
        del sw

    def barrier():
        if distributed:
            dist.barrier()
        torch.cuda.synchronize()

    uuid = None
    try:
        uuid = "GPU-" + str(torch.cuda.get_device_properties(dev).uuid)
    except Exception:
        pass
    rec = wb.run_steps(args.steps, args.warmup, barrier=barrier, sampler=ClockSampler(uuid if uuid else local_rank))
    total_ms = max_over_ranks(rec["total_ms"], dev)
    ms_per_step = total_ms / args.steps
    value = whole_job_value(world, n, ms_per_step)

    # ---- roofline of the dominant kernel (the spd_run kernel) ---------------------------
    peak, peak_src = measured_peak()
    roofline = wb.roofline(rec, peak, peak_src)

    # ---- row f4: the 2-D (DM x time) peak stage over the step's 1-D list (reading A18) -----
    cluster = None
    try:
        if args.no_aux:
            raise spd.SpdError(0, "skipped (--no-aux)")
        lst2 = torch.empty(wb.cap * 16, dtype=torch.uint8, device=dev)
        n2 = torch.zeros(1, dtype=torch.int64, device=dev)
        c_ms = wb.timed(lambda: plan.cluster_candidates(wb.out_snr, wb.cand_list, wb.cand_count, wb.cap, 1, wb.cap,
                                                        lst_out=lst2, n_out=n2))
        cluster = {"what": "spd_cluster_candidates, dm_radius 1, over the step's 1-D list; not part of the step",
                   "ms": c_ms, "candidates_in": min(rec["n_cand"], wb.cap), "kept": int(n2.item()),
                   "injected_pulses": len(wb.pulses)}
        del lst2
    except spd.SpdError as e:
        cluster = {"error": str(e)}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": workload_config(w, widths, {
            **({"grid": args.grid + " (a boxcar separation per width: widths of later iterations only at "
                                    "every 2^i-th sample; one merged plane)"} if args.grid else {}),
            "parallelism": f"dm-rows x{world} (independent DM trials per GPU, no collective)",
            "path": {spd.SPD_PATH_DYADIC_TREE: "dyadic_tree", spd.SPD_PATH_IGRID_TREE: "igrid_tree",
                     spd.SPD_PATH_GRID: "grid"}.get(info["path"], "generic"),
            "width_index_bytes": info["width_bytes"],
            "blocks": info["blocks"], "threads_per_block": info["threads_per_block"],
            "segments_per_row": info["segments_per_row"], "piece_chunks": info["piece_chunks"], "chunk": info["chunk"], "smem_bytes": info["smem_bytes"],
            "candidate_threshold": wb.thr, "candidates_found": rec["n_cand"]}),
        "roofline": roofline,
        "clocks": rec["clocks"],
        "gpu_launches": args.steps * (info["launches_per_run"] + 1),
        "real_time_factor_plane": (w.n_t * w.sampling_time_s) / (ms_per_step * 1e-3),
        "real_time_factor_ska_like": value / PAPER_SKA_SAMPLES_PER_S,
        "n_dm_real_time": value * w.sampling_time_s,
        "row_stats": None if stats_ms is None else {
                      "what": "spd_row_stats, 3 passes (plain + 2 rejection passes at 2 sigma), not part of the step",
                      "ms": stats_ms, "gbs": 3 * 4 * n / (stats_ms * 1e-3) / 1e9, "bytes_per_sample_per_pass": 4,
                      "until_convergence": {"what": "spd_row_stats_converge, clip 2 sigma, rel_tol 1e-4, limit 32 passes "
                                                    "(converged rows are skipped by later passes)",
                                            "ms": conv_ms, "mean_rejection_passes": conv_passes}},
        "width_sigma": None if wsig_ms is None else {
                        "what": "spd_width_sigma: sigma per width from power-of-two decimations, interpolated; "
                                "one pass, not part of the step",
                        "ms": wsig_ms, "gbs": 4 * n / (wsig_ms * 1e-3) / 1e9, "bytes_per_sample": 4,
                        "run_sigma_w_ms": run_sw_ms},
        "cluster_stage": cluster,
    }
    if wb.flush is not None:
        line["config"]["l2_flush_ms_per_step_excluded"] = rec["flush_ms"]

    # ---- end to end through the C ABI with HOST buffers ---------------------------------
    if not args.no_e2e:
        line["e2e"] = run_e2e(args, spd, w, widths, wb.plane, wb.mean, wb.sigma, world, distributed, dev, wb.thr)
    else:
        line["e2e"] = None

    wb.close()
    del wb

    # ---- the other configs, in the same run (rank 0, N = 1 only) --------------------------
    if rank == 0 and world == 1 and not args.no_per_config and not args.n_dm and not args.grid and \
            not args.width_set and not args.width_u8:
        line["per_config"] = per_config_legs(args, spd, torch, dev, peak, peak_src, uuid, local_rank)

    # ---- CPU oracle on the same box (rank 0, N=1 only) ----------------------------------
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        res = time_oracle(w, oracle_widths(w), args.cpu_seconds, seps=grid_separations(args, oracle_widths(w)))
        line["cpu_baseline"] = {k: res[k] for k in ("value", "unit", "cores", "kind", "sample", "prefix_value") if k in res}
    else:
        line["cpu_baseline"] = None

    if rank == 0:
        print(json.dumps(line), flush=True)
    if distributed:
        dist.barrier()
        dist.destroy_process_group()
    return 0


# DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) of the dominant kernel come from the committed
# `ncu --set full` captures listed in profiles/dram_traffic.csv (one row per kernel and workload: samples of the
# captured launch, bytes read and written, the capture's summary file and commit, and the sha256 of the kernel's
# source files at capture time).  The kernels stream rows independently, so the per-sample figure of the
# captured launch scales to this launch.  If the kernel's sources have changed since the capture the figure is
# stale: traffic is null and traffic_source says which capture is outdated.
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "dram_traffic.csv")
KERNEL_SOURCES = {
    "tree_ws": ["spd_tree_ws.cuh", "spd_tree_common.cuh"],
    "tree_ws_ig": ["spd_tree_ws.cuh", "spd_tree_common.cuh"],
    "tree_block": ["spd_tree.cu", "spd_tree_common.cuh"],
    "grid_ws": ["spd_tree_ws.cuh", "spd_tree_common.cuh"],
    "tree_ig": ["spd_tree_ig.cu", "spd_tree_common.cuh"],
}


def kernel_source_hash(key):
    import hashlib
    h = hashlib.sha256()
    for name in KERNEL_SOURCES.get(key, []):
        with open(os.path.join(ROOT, "paper_1910_08324_b200", "csrc", name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def ncu_traffic_bytes(key, w, width_bytes):
    import csv
    if key not in KERNEL_SOURCES or not os.path.exists(TRAFFIC_CSV):
        return None, None, None
    with open(TRAFFIC_CSV) as f:
        rows = [r for r in csv.DictReader(f) if r["kernel"] == key and int(r["workload"]) == w.index and
                r["width_set"] == f"{w.width_kind}:{w.width_param}" and int(r["width_bytes"]) == width_bytes]
    if not rows:
        return None, None, None
    r = rows[-1]
    src = {"measured_in_run": False, "capture": r["capture"], "commit": r["commit"]}
    if r["source_sha256_16"] != kernel_source_hash(key):
        src["stale"] = "the kernel's sources have changed since this capture"
        return None, src, None
    per_sample = (float(r["dram_bytes_read"]) + float(r["dram_bytes_write"])) / float(r["samples"])
    cap = {"samples": float(r["samples"]), "kernel_ms": float(r["kernel_ms"]),
           "alu_pipe_pct": float(r["alu_pipe_pct"]), "fma_pipe_pct": float(r["fma_pipe_pct"])}
    return per_sample * w.n_samples, src, cap


def host_mem_available_bytes():
    try:
        with open("/proc/meminfo") as f:
            for ln in f:
                if ln.startswith("MemAvailable:"):
                    return int(ln.split()[1]) * 1024
    except OSError:
        pass
    return 8 << 30


def run_e2e(args, spd, w, widths, plane, mean, sigma, world, distributed, dev, thr):
    """Same metric end to end through the C ABI on HOST buffers, every copy inside the timed region (wall clock
    around the blocking call, max over ranks).  The headline call is spd_run_host_candidates: pinned HOST plane
    in, rows a1-a8 per row block and the 2-D peak stage (row f4) on the device, the candidate list out - what a
    pipeline consumes.  `planes` adds spd_run_host, which also ships Y and W back (12 B per sample over the link)."""
    import torch
    # rows: the whole plane when host memory allows 12 B/sample of pinned buffers per rank
    budget = host_mem_available_bytes() // (3 * max(1, world))
    rows = int(max(1, min(w.n_dm, budget // (BYTES_PER_SAMPLE * w.n_t))))
    n = rows * w.n_t
    h_plane = torch.empty((rows, w.n_t), dtype=torch.float32, pin_memory=True)
    h_plane.copy_(plane[:rows])
    h_mean = mean[:rows].cpu()
    h_sigma = sigma[:rows].cpu()
    cap = 1 << 20
    h_list = torch.empty(cap * 16, dtype=torch.uint8, pin_memory=True)
    torch.cuda.synchronize()
    seps = None
    if args.grid:
        gkind, _, gparam = args.grid.partition(":")
        seps = spd.spd_separation_generate(gkind, int(gparam or 0), widths)

    def timed_calls(fn):
        times = []
        for i in range(1 + max(1, args.e2e_steps)):
            if distributed:
                torch.distributed.barrier()
            torch.cuda.synchronize()
            t = time.perf_counter()
            out = fn()
            dt = time.perf_counter() - t
            if i > 0:
                times.append(dt)
        return max_over_ranks(sum(times) / len(times), dev), len(times), out

    note = "whole plane" if rows == w.n_dm else f"first {rows} of {w.n_dm} DM trials (host memory bound)"
    with spd.Plan(rows, w.n_t, widths, w.max_width, separations=seps) as plan:
        dt, k, (n_found, n_1d, cands) = timed_calls(
            lambda: plan.run_host_candidates(h_plane, h_mean, h_sigma, thr, 1, cap, out_list=h_list))
        res = {"value": world * n / dt, "unit": UNIT, "h2d_bytes_per_step": 4 * n + 8 * rows,
               "d2h_bytes_per_step": 16 + 16 * min(n_found, cap), "ms_per_step": 1e3 * dt, "steps": k, "rows": rows,
               "api": "spd_run_host_candidates (pinned host plane in; H2D, rows a1-a8 and the 2-D peak stage on the "
                      "device; D2H of the candidate list)",
               "note": note, "candidates_1d": n_1d, "candidates_2d": n_found,
               "checksum": float(cands["snr"].astype("float64").sum()) if len(cands) else 0.0}
    del h_list
    h_snr = torch.empty((rows, w.n_t), dtype=torch.float32, pin_memory=True)
    h_width = torch.empty((rows, w.n_t), dtype=torch.int32, pin_memory=True)
    with spd.Plan(rows, w.n_t, widths, w.max_width, separations=seps) as plan:
        dt, k, _ = timed_calls(lambda: plan.run_host(h_plane, h_mean, h_sigma, h_snr, h_width))
        res["planes"] = {"value": world * n / dt, "unit": UNIT, "h2d_bytes_per_step": 4 * n + 8 * rows,
                         "d2h_bytes_per_step": 8 * n, "ms_per_step": 1e3 * dt, "steps": k,
                         "api": "spd_run_host (Y and W planes back to pinned host buffers)",
                         "checksum": float(h_snr[0, :1024].double().sum().item())}
    return res


def apply_overrides(w, args):
    from dataclasses import replace
    if args.width_set:
        kind, _, param = args.width_set.partition(":")
        w = replace(w, width_kind=kind.upper(), width_param=int(param or 0))
    return w


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_b200(args)


if __name__ == "__main__":
    sys.exit(main())
