#!/usr/bin/env python
"""bench.py -- pair counts in Gpairs/s (DD + DR + RR) on the 1M x 1M full-sky configuration.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME] [--scale S]
                    [--sharded] [--no-configs] [--no-e2e] [--no-cpu-baseline]

A "step" is one pass of the whole hot path over one batch of synthetic input: both catalogues
(already resident in HBM as canonical fp64 vectors) are prepared on the device -- validate, sort,
gather, caps: acf_prepare_again on two handles -- and DD, DR, RR are counted on the handles
(weighted u64 counts + f64 weighted sums for BASELINE.json's full-sky configuration).  One JSON line
is printed by rank 0.  `detail.configs` adds one short measurement of each of the five
configurations of BASELINE.json (same step, default kernel), `detail.jackknife` one of acf_jackknife.

--gpus N: every rank counts its own realisation (weak scaling, no collective on the data path);
with --sharded all ranks hold ONE realisation and rank r counts slice r of N of every count
(acf_pair_count_prepared part / n_parts), the histograms are all-reduced (strong scaling).

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
# The committed ncu capture of the dominant kernel on the default workload (one launch: the weighted DR count,
# 1.0e12 pairs).  Its figures are read from the file at run time and dropped when the kernel sources have changed
# since the capture (the file records their hash).
NCU_PROFILE = "profiles/r2_pair_win_kernel_ncu.md"
ALL_CONFIGS = ["tiny", "clustered_patch", "survey_scale", "full_sky", "pruning_stress"]


def source_hash() -> str:
    """sha256 (16 hex digits) of the library's sources: what an ncu capture must have been made of to describe this build."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_1208_3658_b200", "csrc")
    for name in sorted(os.listdir(d)):
        if name.endswith((".cu", ".cuh", ".h", ".cpp")):
            h.update(name.encode())
            h.update(open(os.path.join(d, name), "rb").read())
    return h.hexdigest()[:16]


def read_ncu_profile():
    """-> dict of the figures in NCU_PROFILE (lines `key: value` of its `bench.py reads` block), or None."""
    try:
        text = open(os.path.join(ROOT, NCU_PROFILE)).read()
    except OSError:
        return None
    out = {"profile": NCU_PROFILE}
    for line in text.splitlines():
        line = line.strip().lstrip("-").strip()
        for key in ("source_sha16", "launch", "dram_bytes", "sass_thread_inst_per_pair", "issue_active_pct", "kernel_ms"):
            if line.startswith(key + ":"):
                v = line.split(":", 1)[1].strip().strip("`")
                out[key] = v if key in ("source_sha16", "launch") else (int(v) if key == "dram_bytes" else float(v))
    if "source_sha16" not in out or "sass_thread_inst_per_pair" not in out:
        return None
    out["stale"] = out["source_sha16"] != source_hash()
    return out


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="full_sky")
    ap.add_argument("--scale", type=float, default=1.0)
    ap.add_argument("--cpu-rows", type=int, default=0, help="rows of the oracle sample (0 = auto)")
    ap.add_argument("--cpu-full", action="store_true", help="cpu_baseline also times clustered_patch in full (about two minutes on 16 cores)")
    ap.add_argument("--kernel", default="auto", choices=["auto", "table", "window"], help="pair kernel (ACF_OPT_KERNEL)")
    ap.add_argument("--bulk", action="store_true", help="ACF_OPT_BULK: count single-bin groups of points as a whole (not the default path)")
    ap.add_argument("--sharded", action="store_true", help="one realisation, rank r counts slice r of N of every count (strong scaling)")
    ap.add_argument("--no-configs", action="store_true", help="skip detail.configs (the five configurations) and detail.jackknife")
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
def host_cores() -> int:
    return len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)


def oracle_rows_for(w, cores: int, seconds: float = 4.0) -> int:
    """Rows of the DR sample that take the oracle about `seconds` on `cores` cores (about 50 Mpairs/s and core);
    the reference arm and the cpu_baseline leg time the same sample."""
    return max(1, min(w.n_d, int(seconds * 50e6 * cores / max(1, w.n_r))))


def oracle_sample(w, n_rows: int, threads: int, xyz=None):
    """Times the CPU oracle, as it stands, on DR rows [0, n_rows) x all randoms (weighted when the workload is).
    Returns (pairs, seconds, threads used)."""
    from oracle import oracle as O
    O.set_num_threads(threads)  # (torchrun sets OMP_NUM_THREADS=1 for its workers: say what is wanted)
    xd, xr = xyz if xyz is not None else (O.radec_to_xyz(w.ra_d, w.dec_d), O.radec_to_xyz(w.ra_r, w.dec_r))
    n_rows = min(n_rows, w.n_d)
    t0 = time.perf_counter()
    O.pair_count(xd, xr, w.cos_edges, False, w_a=w.w_d, w_b=w.w_r, rows=(0, n_rows))
    dt = time.perf_counter() - t0
    return n_rows * w.n_r, dt, O.num_threads()


def cpu_baseline_block(args, w):
    """The oracle on the box's host cores: all cores and one core (the paper's CPU figure is one core)
    on a bounded DR sample of the workload, and the `tiny` configuration in full (DD + DR + RR)."""
    from oracle import oracle as O
    cores = host_cores()
    xyz = (O.radec_to_xyz(w.ra_d, w.dec_d), O.radec_to_xyz(w.ra_r, w.dec_r))
    n_rows = args.cpu_rows or oracle_rows_for(w, cores)
    pairs, dt, used = oracle_sample(w, n_rows, cores, xyz)
    n1 = max(1, n_rows // cores)
    p1, dt1, _ = oracle_sample(w, n1, 1, xyz)
    kind = "weighted" if w.w_d is not None else "unweighted"
    out = {"value": pairs / dt / 1e9, "unit": UNIT, "cores": used, "kind": "oracle",
           "sample": "DR rows [0,%d) x %d randoms, %s, %.1f s" % (n_rows, w.n_r, kind, dt),
           "single_thread": {"value": p1 / dt1 / 1e9, "unit": UNIT, "cores": 1,
                             "sample": "DR rows [0,%d) x %d randoms, %s, %.1f s" % (n1, w.n_r, kind, dt1)}}
    t = make_config("tiny", 1.0)
    O.set_num_threads(cores)
    xd, xr = O.radec_to_xyz(t.ra_d, t.dec_d), O.radec_to_xyz(t.ra_r, t.dec_r)
    t0 = time.perf_counter()
    O.pair_count(xd, None, t.cos_edges, True)
    O.pair_count(xd, xr, t.cos_edges, False)
    O.pair_count(xr, None, t.cos_edges, True)
    dtt = time.perf_counter() - t0
    out["tiny_in_full"] = {"value": t.nominal_pairs / dtt / 1e9, "unit": UNIT, "cores": cores, "seconds": dtt,
                           "sample": "tiny x1: DD + DR + RR, all %d pairs" % t.nominal_pairs}
    if args.cpu_full:
        c = make_config("clustered_patch", 1.0)
        xd, xr = O.radec_to_xyz(c.ra_d, c.dec_d), O.radec_to_xyz(c.ra_r, c.dec_r)
        t0 = time.perf_counter()
        O.pair_count(xd, None, c.cos_edges, True)
        O.pair_count(xd, xr, c.cos_edges, False)
        O.pair_count(xr, None, c.cos_edges, True)
        dtc = time.perf_counter() - t0
        out["clustered_patch_in_full"] = {"value": c.nominal_pairs / dtc / 1e9, "unit": UNIT, "cores": cores, "seconds": dtc,
                                          "sample": "clustered_patch x1: DD + DR + RR, all %d pairs" % c.nominal_pairs}
    return out


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; each step a bounded row sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w = make_config(args.workload, args.scale)
    from oracle import oracle as O
    cores = host_cores()
    xyz = (O.radec_to_xyz(w.ra_d, w.dec_d), O.radec_to_xyz(w.ra_r, w.dec_r))
    n_rows = args.cpu_rows or oracle_rows_for(w, cores)
    for _ in range(args.warmup):
        oracle_sample(w, max(1, n_rows // 8), cores, xyz)
    pairs = secs = 0.0
    used = cores
    for _ in range(args.steps):
        p, dt, used = oracle_sample(w, n_rows, cores, xyz)
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
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": used, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out), flush=True)
    return 0


# --------------------------------------------------------------------------- our arm
class Runner:
    """One workload on one device: the canonical vectors and weights in HBM, two catalogue handles, and the step."""

    def __init__(self, P, ctx, dev, w):
        import torch
        self.P, self.ctx, self.dev, self.w = P, ctx, dev, w
        self.weighted = w.w_d is not None
        self.xd = torch.from_numpy(P.acf_radec_to_xyz(w.ra_d, w.dec_d)).to(dev)
        self.xr = torch.from_numpy(P.acf_radec_to_xyz(w.ra_r, w.dec_r)).to(dev)
        self.wd = torch.from_numpy(w.w_d).to(dev) if self.weighted else None
        self.wr = torch.from_numpy(w.w_r).to(dev) if self.weighted else None
        nb = w.nbins
        self.counts = [torch.empty(nb, dtype=torch.int64, device=dev) for _ in range(3)]
        self.wsums = [torch.empty(nb, dtype=torch.float64, device=dev) for _ in range(3)] if self.weighted else [None] * 3
        self.cd = P.acf_prepare(ctx, self.xd, self.wd)
        self.cr = P.acf_prepare(ctx, self.xr, self.wr)

    def close(self):
        self.P.acf_release(self.ctx, self.cd)
        self.P.acf_release(self.ctx, self.cr)

    def step(self, acc=None, part=0, n_parts=1):
        """Prepare both catalogues (validate, sort, gather, caps), count DD, DR, RR on the handles."""
        P, ctx, e = self.P, self.ctx, self.w.cos_edges
        for cat, x, wt in ((self.cd, self.xd, self.wd), (self.cr, self.xr, self.wr)):
            P.acf_prepare_again(ctx, cat, x, wt)
            if acc is not None:
                acc["launches"] += P.acf_get_stats(ctx)["kernel_launches"]
        for k, (a, b) in enumerate(((self.cd, None), (self.cd, self.cr), (self.cr, None))):
            P.acf_pair_count_prepared(ctx, a, b, e, part=part, n_parts=n_parts, weighted=self.weighted,
                                      d_counts=self.counts[k], d_wsums=self.wsums[k])
            if acc is not None:
                st = P.acf_get_stats(ctx)  # synchronises; only outside the timed steps
                acc["launches"] += st["kernel_launches"]
                for key, name in (("pair_ms", "pair_kernel_ms"), ("evaluated", "pairs_evaluated"), ("fp64", "pairs_fp64"),
                                  ("window", "pairs_window"), ("chord", "pairs_chord")):
                    acc[key] += st[name]


def new_acc():
    return {"launches": 0, "pair_ms": 0.0, "evaluated": 0, "fp64": 0, "window": 0, "chord": 0}


def timed_steps(runner, steps, warmup, flush_buf, stream, part=0, n_parts=1, barrier=None):
    """W warm-up steps, one instrumented step (statistics, not timed), K timed steps with CUDA events on the
    context's stream, L2 flushed between steps.  -> (ms per step list, wall seconds, statistics of one step)."""
    import torch
    for _ in range(warmup):
        runner.step(part=part, n_parts=n_parts)
        flush_buf.fill_(1)
    acc = new_acc()
    runner.step(acc, part=part, n_parts=n_parts)
    flush_buf.fill_(2)
    torch.cuda.synchronize(runner.dev)
    if barrier is not None:
        barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    t0 = time.perf_counter()
    for k in range(steps):
        ev[k][0].record(stream)
        runner.step(part=part, n_parts=n_parts)
        ev[k][1].record(stream)
        flush_buf.fill_(k)  # L2 flush between timed steps, outside the per-step events
    torch.cuda.synchronize(runner.dev)
    wall = time.perf_counter() - t0
    return [a.elapsed_time(b) for a, b in ev], wall, acc


def e2e_measure(P, ctx, w, steps):
    """The same metric end to end through acf_correlate_host: host canonicalisation, H2D from pinned staging, the
    three counts, D2H, the estimator.  -> dict."""
    P.acf_correlate_host(ctx, w.ra_d, w.dec_d, w.w_d, w.ra_r, w.dec_r, w.w_r, w.cos_edges)  # warm the staging buffers
    t0 = time.perf_counter()
    for _ in range(steps):
        res = P.acf_correlate_host(ctx, w.ra_d, w.dec_d, w.w_d, w.ra_r, w.dec_r, w.w_r, w.cos_edges)
    dt = time.perf_counter() - t0
    weighted = w.w_d is not None
    nb = w.nbins
    assert int(res["dd"].sum()) > 0
    return {"seconds": dt, "steps": steps,
            "h2d": 24 * (w.n_d + w.n_r) + (4 * (w.n_d + w.n_r) if weighted else 0) + 8 * (nb + 1),
            "d2h": 3 * nb * (8 + (8 if weighted else 0))}


def config_line(P, ctx, dev, name, flush_buf, stream, peak_tinst, runner=None, e2e=False):
    """One short measurement of a configuration of BASELINE.json at full size (detail.configs)."""
    w = runner.w if runner is not None else make_config(name, 1.0)
    own = runner is None
    if own:
        runner = Runner(P, ctx, dev, w)
    ms, _, acc = timed_steps(runner, 3, 3, flush_buf, stream)
    if own:
        runner.close()
    t = float(np.median(ms)) * 1e-3
    i_alg = I_ALG_WEIGHTED if w.w_d is not None else I_ALG_UNWEIGHTED
    line = {"ms_per_step": 1e3 * t, "nominal_gpairs_s": w.nominal_pairs / t / 1e9, "evaluated_gpairs_s": acc["evaluated"] / t / 1e9,
            "pairs_nominal": w.nominal_pairs, "pairs_evaluated": acc["evaluated"], "pair_kernel_ms": acc["pair_ms"],
            "prep_share": max(0.0, 1.0 - acc["pair_ms"] / (1e3 * t)), "launches_per_step": acc["launches"],
            "frac_algorithmic": acc["evaluated"] * i_alg / (acc["pair_ms"] * 1e-3) / 1e12 / peak_tinst if acc["pair_ms"] > 0 else None,
            "kernel": "pair_win_kernel", "pairs_fp64": acc["fp64"], "pairs_single_edge": acc["window"], "pairs_on_chord": acc["chord"]}
    if e2e:
        r = e2e_measure(P, ctx, w, 3)
        line["e2e_gpairs_s"] = w.nominal_pairs * r["steps"] / r["seconds"] / 1e9
        line["e2e_over_device"] = line["e2e_gpairs_s"] / line["nominal_gpairs_s"]
    return line


def jackknife_line(P, ctx, dev):
    """acf_jackknife on the clustered patch, 16 regions in RA: wall time of the whole call (detail.jackknife)."""
    import torch
    w = make_config("clustered_patch", 1.0)
    n_reg = 16
    out = {}
    xs = []
    for ra, dec in ((w.ra_d, w.dec_d), (w.ra_r, w.dec_r)):
        reg = np.minimum((ra / 20.0 * n_reg).astype(int), n_reg - 1)
        order = np.argsort(reg, kind="stable")
        xs.append((torch.from_numpy(P.acf_radec_to_xyz(ra[order], dec[order])).to(dev), np.searchsorted(reg[order], np.arange(n_reg + 1))))
    P.acf_jackknife(ctx, xs[0][0], xs[0][1], xs[1][0], xs[1][1], w.cos_edges)
    torch.cuda.synchronize(dev)
    t0 = time.perf_counter()
    res = P.acf_jackknife(ctx, xs[0][0], xs[0][1], xs[1][0], xs[1][1], w.cos_edges)
    dt = time.perf_counter() - t0
    out = {"workload": "clustered_patch x1, %d regions in RA, Landy-Szalay" % n_reg, "seconds": dt,
           "launches": P.acf_get_stats(ctx)["kernel_launches"], "gpairs_s_nominal": w.nominal_pairs / dt / 1e9,
           "finite_bins": int(np.isfinite(res["w"]).sum())}
    return out


def ensemble_line(P, ctx, dev):
    """acf_random_ensemble: the clustered patch's data against 8 random catalogues (detail.mc_randoms)."""
    import torch
    w = make_config("clustered_patch", 1.0)
    K = 8
    xd = torch.from_numpy(P.acf_radec_to_xyz(w.ra_d, w.dec_d)).to(dev)
    rands = []
    for k in range(K):
        r = make_config("clustered_patch", 1.0, seed_offset=100 + k)
        rands.append(torch.from_numpy(P.acf_radec_to_xyz(r.ra_r, r.dec_r)).to(dev))
    cat = P.acf_prepare(ctx, xd)
    P.acf_random_ensemble(ctx, cat, rands[:2], w.cos_edges)
    torch.cuda.synchronize(dev)
    t0 = time.perf_counter()
    res = P.acf_random_ensemble(ctx, cat, rands, w.cos_edges)
    dt = time.perf_counter() - t0
    launches = P.acf_get_stats(ctx)["kernel_launches"]
    P.acf_release(ctx, cat)
    pairs = w.n_d * (w.n_d - 1) // 2 + K * (w.n_d * w.n_r + w.n_r * (w.n_r - 1) // 2)
    sd = np.sqrt(np.diag(res["cov"]))
    return {"workload": "clustered_patch x1 data, %d random catalogues of %d points, Landy-Szalay" % (K, w.n_r), "seconds": dt,
            "launches": launches, "gpairs_s_nominal": pairs / dt / 1e9, "median_sigma_w": float(np.nanmedian(sd))}


# PAPER.md:117-124 (Table 1): the DR component, n^2 pairs, 254 logarithmic bins; whole-program wall time on a Tesla
# M2070 and on one core of a Xeon E5540, its own catalogue.  Context for detail.paper_shaped, not a
# target: another machine, another dataset, a timed region that there included reading a text file.
PAPER_TABLE1 = {"n": [10 ** 4, 10 ** 5, 10 ** 6], "gpu_seconds": [0.2, 16.0, 1254.0], "cpu_seconds": [23.9, 2305.0, 231225.0]}


def paper_shaped_line(P, ctx, dev):
    """The shape of the paper's own timing test: the DR count of n clustered galaxies against n
    "flat" randoms on the octant 0 < RA, Dec < 90 deg, 254 logarithmic bins over a wide range (1 arcmin - 90 deg), n =
    1e4, 1e5, 1e6.  Timed from host coordinates to host histogram: canonicalisation, H2D, the count, D2H
    (detail.paper_shaped)."""
    import torch
    from workloads import cos_edges_from_theta_deg, log_theta_edges_deg, neyman_scott, uniform_patch
    edges = cos_edges_from_theta_deg(log_theta_edges_deg(1.0 / 60.0, 90.0, 254))
    octant = ((0.0, 90.0), (0.0, 90.0))
    seconds, in_range = [], []
    for k, n in enumerate(PAPER_TABLE1["n"]):
        ra_d, dec_d = neyman_scott(n, max(1, n // 20), 5.0, octant[0], octant[1], 51 + k, children="poisson")
        ra_r, dec_r = uniform_patch(n, octant[0], octant[1], 61 + k)
        for rep in range(2 if n < 10 ** 6 else 1):  # (the small ones once more, warm)
            torch.cuda.synchronize(dev)
            t0 = time.perf_counter()
            xa = torch.from_numpy(P.acf_radec_to_xyz(ra_d, dec_d)).to(dev)
            xb = torch.from_numpy(P.acf_radec_to_xyz(ra_r, dec_r)).to(dev)
            counts = P.counts_to_numpy(P.acf_pair_count(ctx, xa, xb, edges, False))
            dt = time.perf_counter() - t0
        seconds.append(dt)
        in_range.append(int(counts.sum()))
    return {"workload": "DR of n clustered points x n flat randoms on the octant 0 < RA, Dec < 90 deg, 254 log bins 1 arcmin - 90 deg, unweighted; "
                        "host coordinates -> host histogram (canonicalise, H2D, prepare, count, D2H)",
            "n": PAPER_TABLE1["n"], "seconds": seconds, "pairs_in_range": in_range,
            "gpairs_s": [n * n / t / 1e9 for n, t in zip(PAPER_TABLE1["n"], seconds)],
            "paper_table1": dict(PAPER_TABLE1, cite="PAPER.md:117-124", note="context only: Tesla M2070 / one Xeon E5540 core, the paper's "
                                 "catalogue, whole-program wall time including the text file")}


def binning_sweep_line(P, ctx, dev):
    """The paper's binning sweep (the DR count of the 1e5 sample over bin counts, ranges and even or
    logarithmic spacing took between 11 and 57 s there, "users should be aware that depending on their choice of
    binning, timing results may vary"): the same kind of sweep on the octant catalogue of paper_shaped_line, n = 1e5,
    catalogues resident and prepared once, each count timed on its own after one warm call (detail.binning_sweep)."""
    import torch
    from workloads import neyman_scott, uniform_patch
    n = 10 ** 5
    octant = ((0.0, 90.0), (0.0, 90.0))
    ra_d, dec_d = neyman_scott(n, n // 20, 5.0, octant[0], octant[1], 52, children="poisson")
    ra_r, dec_r = uniform_patch(n, octant[0], octant[1], 62)
    cd = P.acf_prepare(ctx, torch.from_numpy(P.acf_radec_to_xyz(ra_d, dec_d)).to(dev))
    cr = P.acf_prepare(ctx, torch.from_numpy(P.acf_radec_to_xyz(ra_r, dec_r)).to(dev))
    cases = [("log", 1.0 / 60.0, 90.0, 254), ("log", 1.0 / 60.0, 90.0, 20), ("log", 1.0 / 60.0, 90.0, 1024),
             ("even", 0.0, 90.0, 254), ("even", 0.0, 90.0, 20), ("even", 0.0, 90.0, 1024),
             ("log", 1.0 / 60.0, 1.0, 254), ("even", 0.0, 10.0, 100)]
    rows = []
    for kind, lo, hi, nb in cases:
        edges = P.acf_cos_edges(P.acf_theta_edges(P.ACF_BINS_LOG if kind == "log" else P.ACF_BINS_EVEN, lo, hi, nb))
        out = torch.empty(nb, dtype=torch.int64, device=dev)
        P.acf_pair_count_prepared(ctx, cd, cr, edges, d_counts=out)
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        P.acf_pair_count_prepared(ctx, cd, cr, edges, d_counts=out)
        torch.cuda.synchronize(dev)
        dt = time.perf_counter() - t0
        st = P.acf_get_stats(ctx)
        rows.append({"bins": "%s, %d bins, %.4g - %.4g deg" % (kind, nb, lo, hi), "ms": 1e3 * dt, "gpairs_s_nominal": n * n / dt / 1e9,
                     "pairs_evaluated": st["pairs_evaluated"], "pairs_in_range": int(P.counts_to_numpy(out).sum())})
    P.acf_release(ctx, cd)
    P.acf_release(ctx, cr)
    ms = [r["ms"] for r in rows]
    return {"workload": "DR of 1e5 clustered points x 1e5 flat randoms on the octant, unweighted, prepared catalogues; one count per binning",
            "cases": rows, "ms_min": min(ms), "ms_max": max(ms),
            "paper": {"seconds_min": 11.0, "seconds_max": 57.0, "cite": "PAPER.md:126",
                      "note": "context only: Tesla M2070, the paper's catalogue and its own choice of binnings"}}


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
    barrier = dist.barrier if dist is not None else None
    sharded = bool(args.sharded) and world > 1

    # replicas (default): every rank counts its own realisation of the workload (independent catalogues, e.g. the
    # many random catalogues of a Monte-Carlo error estimate), no collective on the data path.
    # --sharded: one realisation on every rank, rank r counts slice r of `world` of every count (PAPER.md:201:
    # "division of the dataset into sub-sets"), the histograms are summed with one all-reduce per step.
    w = make_config(args.workload, args.scale, seed_offset=0 if sharded else 1000 * rank)
    weighted = w.w_d is not None
    dev = torch.device("cuda", local_rank)
    ctx = P.acf_create(local_rank)
    P.acf_set_option(ctx, P.ACF_OPT_KERNEL, {"auto": P.ACF_KERNEL_AUTO, "table": P.ACF_KERNEL_TABLE, "window": P.ACF_KERNEL_WINDOW}[args.kernel])
    if args.bulk:
        P.acf_set_option(ctx, P.ACF_OPT_BULK, 1)
    stream = torch.cuda.current_stream(dev)
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2
    runner = Runner(P, ctx, dev, w)
    part, n_parts = (rank, world) if sharded else (0, 1)

    if sharded:
        from paper_1208_3658_b200.sharding import all_reduce_counts
        plain_step = runner.step

        def step_and_reduce(acc=None, part=0, n_parts=1):
            plain_step(acc, part=part, n_parts=n_parts)
            for k in range(3):
                all_reduce_counts(runner.counts[k], runner.wsums[k])
        runner.step = step_and_reduce

    sampler = ClockSampler(local_rank)
    sampler.start()
    ms_steps, t_wall, acc = timed_steps(runner, args.steps, args.warmup, flush_buf, stream, part, n_parts, barrier)
    if dist is not None:
        dist.barrier()
    clocks = sampler.stop()
    ms_total = float(sum(ms_steps))
    if dist is not None:
        t = torch.tensor([ms_total], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    pairs_per_step = w.nominal_pairs
    jobs = 1 if sharded else world
    value = jobs * pairs_per_step * args.steps / (ms_total * 1e-3) / 1e9
    launches_per_step, pair_ms_per_step, evaluated_per_step = acc["launches"], acc["pair_ms"], acc["evaluated"]

    # ---- end to end through the C ABI with host buffers (canonicalise + H2D + count + D2H + Eq. 2)
    e2e = None
    if not args.no_e2e and not sharded:
        e2e_steps = max(1, min(args.steps, 2))
        torch.cuda.synchronize(dev)
        if dist is not None:
            dist.barrier()
        r = e2e_measure(P, ctx, w, e2e_steps)
        dt = r["seconds"]
        if dist is not None:
            t = torch.tensor([dt], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        e2e = {"value": world * pairs_per_step * e2e_steps / dt / 1e9, "unit": UNIT, "h2d_bytes_per_step": r["h2d"],
               "d2h_bytes_per_step": r["d2h"], "steps": e2e_steps,
               "includes": "host canonicalisation (glibc sin/cos), H2D from pinned staging (the randoms' on a second stream under "
                           "the DD count), prepare + DD + DR + RR, D2H, Eq. 2"}

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
    pair_s = pair_ms_per_step * 1e-3
    step_ms = ms_total / args.steps
    achieved = evaluated_per_step * i_alg / pair_s / 1e12 if pair_s > 0 else 0.0
    headline = args.workload == "full_sky" and args.scale == 1.0 and args.kernel == "auto" and not args.bulk and not sharded
    ncu = read_ncu_profile() if headline else None
    if ncu is not None and ncu["stale"]:
        ncu = {"profile": ncu["profile"], "stale": True, "note": "the kernel sources have changed since this capture: its figures are not quoted"}
    issued = None
    if ncu is not None and not ncu.get("stale"):
        # what the kernel actually issues: SASS thread-instructions per pair (ncu) x pairs per second, against the peak issue rate
        issued = ncu["sass_thread_inst_per_pair"] * evaluated_per_step / pair_s / 1e12 / peak_tinst
    roofline = {
        "bound": "alu", "kernel": "pair_kernel" if args.kernel == "table" else "pair_win_kernel", "achieved": achieved, "peak": peak_tinst,
        "unit": "Tinst/s", "frac": achieved / peak_tinst,
        "frac_is": "ALGORITHMIC thread-instructions per pair (SURVEY.md 8(d): 3 cosine + ~5 locate + 2 certify + 1 update, +3 weighted) x "
                   "pairs evaluated / pair-kernel time / peak issue rate.  The kernel issues fewer instructions per pair than that "
                   "(FFMA2, register tallies), so this can exceed 1: it is a speed relative to a kernel that spends the algorithmic "
                   "instructions at full issue rate, NOT the issue-slot utilisation -- that is issue_frac",
        "issue_frac": issued,
        "issue_frac_is": "SASS thread-instructions per pair of the committed ncu capture x pairs evaluated / pair-kernel time of THIS run / "
                         "peak issue rate: the share of the issue slots the kernel fills (null when the capture is stale or absent)",
        "traffic": (ncu or {}).get("dram_bytes"), "traffic_is": "dram__bytes_read.sum + dram__bytes_write.sum of one launch (%s), %s"
                                                                 % ((ncu or {}).get("launch"), NCU_PROFILE),
        "ncu": ncu, "algorithmic_inst_per_pair": i_alg,
        "frac_of_fma_floor": (evaluated_per_step * 3 / pair_s / 1e12 / peak_tinst) if pair_s > 0 else 0.0,
        "pairs_per_step": evaluated_per_step, "kernel_ms_per_step": pair_ms_per_step,
        "kernel_share_of_step": pair_ms_per_step / step_ms if step_ms > 0 else None,
        "peak_is": "%d SMs x 4 schedulers x 32 lanes x %.0f MHz (max SM clock, MEASURED_PEAKS.json / fallback 1965)"
                   % (props.multi_processor_count, sm_max_mhz),
        "frac_at_observed_clock": (achieved / (peak_tinst * clocks["sm_mhz"] / sm_max_mhz)) if clocks.get("sm_mhz") else None,
    }

    # ---- the five configurations and the jackknife, one short measurement each (one GPU, rank 0's box only)
    configs = jk = mc = paper = sweep = None
    if world == 1 and not args.no_configs:
        configs = {}
        for name in ALL_CONFIGS:
            same = name == args.workload and args.scale == 1.0
            configs[name] = config_line(P, ctx, dev, name, flush_buf, stream, peak_tinst, runner=runner if same else None,
                                        e2e=name in ("tiny", "clustered_patch"))
        jk = jackknife_line(P, ctx, dev)
        mc = ensemble_line(P, ctx, dev)
        paper = paper_shaped_line(P, ctx, dev)
        sweep = binning_sweep_line(P, ctx, dev)

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu_baseline = cpu_baseline_block(args, w)

    if rank == 0:
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": step_ms, "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_label(args, w), "pairs_per_step": pairs_per_step, "l2": "flushed between timed steps (256 MB write)",
                       "per_rank": ("slice r of %d of every count of one realisation; one all-reduce of the histograms per step" % world) if sharded
                                   else "independent realisation per rank (seeds + 1000*rank)",
                       "step": "acf_prepare_again x2 (validate, sort, gather, caps) + DD + DR + RR on the handles",
                       "bulk_windows": bool(args.bulk)},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches_per_step * args.steps, "roofline": roofline,
            "cpu_baseline": cpu_baseline,
            "detail": {"ms_steps": ms_steps, "wall_s_timed_region": t_wall, "pairs_fp64_per_step": acc["fp64"],
                       "pairs_evaluated_per_step": evaluated_per_step, "pairs_single_edge_window_per_step": acc["window"],
                       "pairs_on_chord_per_step": acc["chord"], "launches_per_step": launches_per_step,
                       "source_sha16": source_hash(), "version": P.acf_version(), "configs": configs, "jackknife": jk, "mc_randoms": mc,
                       "paper_shaped": paper, "binning_sweep": sweep},
        }
        print(json.dumps(out), flush=True)
    runner.close()
    P.acf_destroy(ctx)
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
