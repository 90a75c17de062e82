#!/usr/bin/env python
"""bench.py -- pair counts in Gpairs/s (DD + DR + RR) on the 1M x 1M full-sky configuration.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME] [--scale S]

A "step" is one pass of the whole hot path over one batch of synthetic input: the three
pair-count calls DD, DR, RR (weighted u64 counts + f64 weighted sums) of BASELINE.json's
full-sky configuration, catalogues already resident in HBM, including the on-device
preparation (validate, sort, gather, caps, work list).  One JSON line is printed by rank 0.

--impl reference times the CPU oracle (oracle/), as it stands, on the host cores on a bounded
row sample of the same workload (this tier has no reference implementation to install).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from workloads import make_config  # noqa: E402

METRIC = "pair counts Gpairs/s (DD+DR+RR)"
UNIT = "Gpairs/s"
# SURVEY.md 8(d) / DESIGN.md "Roofline": algorithmic thread-instructions per pair
I_ALG_UNWEIGHTED = 11
I_ALG_WEIGHTED = 14
# From the committed ncu capture of the dominant kernel on the default workload (one launch: the weighted DR
# count, 1.0e12 pairs); not measured by this script.  See profiles/r1_v5_pair_win_kernel_ncu.md.
NCU_FULL_SKY = {"profile": "profiles/r1_v5_pair_win_kernel_ncu.md", "launch": "weighted DR count, 1.0e12 pairs",
                "dram_bytes": 2298431496, "sass_thread_inst_per_pair": 7.23, "issue_active_pct": 60.8}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="full_sky")
    ap.add_argument("--scale", type=float, default=1.0)
    ap.add_argument("--cpu-rows", type=int, default=0, help="rows of the oracle sample (0 = auto)")
    ap.add_argument("--kernel", default="auto", choices=["auto", "table", "window"], help="pair kernel (ACF_OPT_KERNEL)")
    ap.add_argument("--bulk", action="store_true", help="ACF_OPT_BULK: count single-bin groups of points as a whole (not the default path)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


# --------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples nvidia-smi SM clocks and throttle reasons while the timed region runs."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.FIELDS, "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            p = [x.strip() for x in ln.split(",")]
            if len(p) < 8:
                continue
            try:
                sm.append(float(p[0]))
                smax.append(float(p[1]))
                power.append(float(p[2]))
            except ValueError:
                continue
            for name, v in zip(names, p[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "power_w_max": float(max(power)),
                "samples": len(sm), "reasons": sorted(reasons)}


def workload_label(args, w) -> str:
    """The same workload name on both arms."""
    return "%s x%g: %d data + %d random, %d log bins, %s; DD+DR+RR per step" % (
        args.workload, args.scale, w.n_d, w.n_r, w.nbins, "weighted (u64 counts + f64 sums)" if w.w_d is not None else "unweighted")


# --------------------------------------------------------------------------- oracle legs
def oracle_sample(w, n_rows: int):
    """Times the CPU oracle on DR rows [0, n_rows) x all randoms (weighted when the workload is).
    Returns (pairs, seconds, cores)."""
    from oracle import oracle as O
    # all the box's cores, also under torchrun (which sets OMP_NUM_THREADS=1 for its workers)
    O.set_num_threads(len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1))
    xd = O.radec_to_xyz(w.ra_d, w.dec_d)
    xr = O.radec_to_xyz(w.ra_r, w.dec_r)
    n_rows = min(n_rows, w.n_d)
    t0 = time.perf_counter()
    O.pair_count(xd, xr, w.cos_edges, False, w_a=w.w_d, w_b=w.w_r, rows=(0, n_rows))
    dt = time.perf_counter() - t0
    return n_rows * w.n_r, dt, O.num_threads()


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; each step a bounded row sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w = make_config(args.workload, args.scale)
    from oracle import oracle as O
    O.set_num_threads(len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1))
    cores = O.num_threads()
    # ~2 s of work per step at ~25 Mpairs/s/core
    n_rows = args.cpu_rows or max(1, min(w.n_d, int(2.0 * 25e6 * cores / max(1, w.n_r))))
    for _ in range(args.warmup):
        oracle_sample(w, max(1, n_rows // 8))
    pairs = secs = 0.0
    for _ in range(args.steps):
        p, dt, _ = oracle_sample(w, n_rows)
        pairs += p
        secs += dt
    value = pairs / secs / 1e9
    sample = "DR rows [0,%d) x %d randoms per step (%s)" % (n_rows, w.n_r, "weighted" if w.w_d is not None else "unweighted")
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_label(args, w), "pairs_per_step": w.nominal_pairs,
                   "reference_step": "a bounded sample of the workload: " + sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out), flush=True)
    return 0


# --------------------------------------------------------------------------- our arm
def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import paper_1208_3658_b200 as P

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libacf has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    # weak scaling: every rank counts its own realisation of the workload (independent catalogues,
    # e.g. the many random catalogues of a Monte-Carlo error estimate); no collective
    # on the data path
    w = make_config(args.workload, args.scale, seed_offset=1000 * rank)
    weighted = w.w_d is not None
    ctx = P.acf_create(local_rank)
    P.acf_set_option(ctx, P.ACF_OPT_KERNEL, {"auto": P.ACF_KERNEL_AUTO, "table": P.ACF_KERNEL_TABLE, "window": P.ACF_KERNEL_WINDOW}[args.kernel])
    if args.bulk:
        P.acf_set_option(ctx, P.ACF_OPT_BULK, 1)
    dev = torch.device("cuda", local_rank)
    h_xd = P.acf_radec_to_xyz(w.ra_d, w.dec_d)
    h_xr = P.acf_radec_to_xyz(w.ra_r, w.dec_r)
    xd = torch.from_numpy(h_xd).to(dev)
    xr = torch.from_numpy(h_xr).to(dev)
    wd = torch.from_numpy(w.w_d).to(dev) if weighted else None
    wr = torch.from_numpy(w.w_r).to(dev) if weighted else None
    nb = w.nbins
    counts = [torch.empty(nb, dtype=torch.int64, device=dev) for _ in range(3)]
    wsums = [torch.empty(nb, dtype=torch.float64, device=dev) for _ in range(3)] if weighted else [None] * 3
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2
    stream = torch.cuda.current_stream(dev)

    stats_acc = {"launches": 0, "pair_ms": 0.0, "device_ms": 0.0, "evaluated": 0, "fp64": 0, "window": 0}

    def step(collect: bool):
        calls = [(xd, wd, None, None, True, 0), (xd, wd, xr, wr, False, 1), (xr, wr, None, None, True, 2)]
        for a, wa, b, wb, auto, k in calls:
            if weighted:
                P.acf_pair_count_weighted(ctx, a, wa, b, wb, w.cos_edges, auto, counts[k], wsums[k])
            else:
                P.acf_pair_count(ctx, a, b, w.cos_edges, auto, counts[k])
            if collect:
                st = P.acf_get_stats(ctx)  # synchronises; only outside the timed steps
                stats_acc["launches"] += st["kernel_launches"]
                stats_acc["pair_ms"] += st["pair_kernel_ms"]
                stats_acc["device_ms"] += st["device_ms"]
                stats_acc["evaluated"] += st["pairs_evaluated"]
                stats_acc["fp64"] += st["pairs_fp64"]
                stats_acc["window"] += st["pairs_window"]

    for _ in range(args.warmup):
        step(False)
        flush_buf.fill_(1)
    # one instrumented step (not timed) for per-kernel shares and launch counts
    step(True)
    flush_buf.fill_(2)
    launches_per_step = stats_acc["launches"]
    pair_ms_per_step = stats_acc["pair_ms"]
    evaluated_per_step = stats_acc["evaluated"]

    torch.cuda.synchronize(dev)
    if dist is not None:
        dist.barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    torch.cuda.synchronize(dev)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    t_wall0 = time.perf_counter()
    for k in range(args.steps):
        ev[k][0].record(stream)
        step(False)
        ev[k][1].record(stream)
        flush_buf.fill_(k)  # L2 flush between timed steps, outside the per-step events
    torch.cuda.synchronize(dev)
    t_wall = time.perf_counter() - t_wall0
    if dist is not None:
        dist.barrier()
    clocks = sampler.stop()
    ms_steps = [a.elapsed_time(b) for a, b in ev]
    ms_total = float(sum(ms_steps))
    if dist is not None:
        t = torch.tensor([ms_total], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    pairs_per_step = w.nominal_pairs
    value = world * pairs_per_step * args.steps / (ms_total * 1e-3) / 1e9

    # ---- end to end through the C ABI with host buffers (canonicalise + H2D + count + D2H + Eq. 2)
    e2e = None
    if not args.no_e2e:
        e2e_steps = max(1, min(args.steps, 2))
        P.acf_correlate_host(ctx, w.ra_d, w.dec_d, w.w_d, w.ra_r, w.dec_r, w.w_r, w.cos_edges)  # warm the staging buffers
        torch.cuda.synchronize(dev)
        if dist is not None:
            dist.barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            res = P.acf_correlate_host(ctx, w.ra_d, w.dec_d, w.w_d, w.ra_r, w.dec_r, w.w_r, w.cos_edges)
        dt = time.perf_counter() - t0
        if dist is not None:
            t = torch.tensor([dt], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        h2d = 24 * (w.n_d + w.n_r) + (4 * (w.n_d + w.n_r) if weighted else 0) + 8 * (nb + 1)
        d2h = 3 * nb * (8 + (8 if weighted else 0))
        e2e = {"value": world * pairs_per_step * e2e_steps / dt / 1e9, "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "steps": e2e_steps,
               "includes": "host canonicalisation (glibc sin/cos), H2D, DD+DR+RR, D2H, Eq. 2"}
        assert int(res["dd"].sum()) > 0

    # ---- roofline of the dominant kernel (pair kernel): issue-slot bound
    props = torch.cuda.get_device_properties(dev)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except (OSError, ValueError):
        pass
    sm_max_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    i_alg = I_ALG_WEIGHTED if weighted else I_ALG_UNWEIGHTED
    peak_tinst = props.multi_processor_count * 4 * 32 * sm_max_mhz * 1e6 / 1e12  # thread-instructions/s (T)
    pair_kernel_share = pair_ms_per_step / max(1e-9, stats_acc["device_ms"])
    pair_s = pair_ms_per_step * 1e-3
    achieved = evaluated_per_step * i_alg / pair_s / 1e12 if pair_s > 0 else 0.0
    roofline = {
        "bound": "alu", "kernel": "pair_win_kernel" if (weighted or args.kernel == "window") and args.kernel != "table" else "pair_kernel", "achieved": achieved, "peak": peak_tinst, "unit": "Tinst/s",
        "frac": achieved / peak_tinst,
        "traffic": NCU_FULL_SKY["dram_bytes"] if (args.workload == "full_sky" and args.scale == 1.0 and args.kernel == "auto") else None,
        "traffic_is": "dram__bytes_read.sum + dram__bytes_write.sum of one launch (%s), %s" % (NCU_FULL_SKY["launch"], NCU_FULL_SKY["profile"]),
        "ncu": NCU_FULL_SKY if (args.workload == "full_sky" and args.scale == 1.0 and args.kernel == "auto") else None,
        "algorithmic_inst_per_pair": i_alg,
        "algorithmic_inst_is": "SURVEY.md 8(d): 3 cosine + ~5 locate + 2 certify + 1 update (+3 weighted); the window kernel's "
                               "single-edge loop issues 5.5 per weighted pair, so frac may exceed 1: see ncu.issue_active_pct for the "
                               "issue-slot utilisation itself",
        "frac_of_fma_floor": (evaluated_per_step * 3 / pair_s / 1e12 / peak_tinst) if pair_s > 0 else 0.0, "pairs_per_step": evaluated_per_step, "kernel_ms_per_step": pair_ms_per_step,
        "kernel_share_of_step": pair_kernel_share,
        "peak_is": "%d SMs x 4 schedulers x 32 lanes x %.0f MHz (max SM clock, MEASURED_PEAKS.json / fallback 1965)"
                   % (props.multi_processor_count, sm_max_mhz),
        "frac_at_observed_clock": (achieved / (peak_tinst * clocks["sm_mhz"] / sm_max_mhz)) if clocks.get("sm_mhz") else None,
    }

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import oracle as O
        O.set_num_threads(len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1))
        cores = O.num_threads()
        n_rows = args.cpu_rows or max(1, min(w.n_d, int(12.0 * 25e6 * cores / max(1, w.n_r))))
        pairs, dt, cores = oracle_sample(w, n_rows)
        cpu_baseline = {"value": pairs / dt / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": "DR rows [0,%d) x %d randoms, %s, %.1f s" % (n_rows, w.n_r, "weighted" if weighted else "unweighted", dt)}

    if rank == 0:
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_label(args, w), "pairs_per_step": pairs_per_step, "l2": "flushed between timed steps (256 MB write)",
                "per_rank": "independent realisation per rank (seeds + 1000*rank)",
                "bulk_windows": bool(args.bulk)},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches_per_step * args.steps, "roofline": roofline,
            "cpu_baseline": cpu_baseline,
            "detail": {"ms_steps": ms_steps, "wall_s_timed_region": t_wall, "pairs_fp64_per_step": stats_acc["fp64"],
                       "pairs_evaluated_per_step": evaluated_per_step, "pairs_single_edge_window_per_step": stats_acc["window"], "launches_per_step": launches_per_step,
                       "version": P.acf_version()},
        }
        print(json.dumps(out), flush=True)
    P.acf_destroy(ctx)
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
