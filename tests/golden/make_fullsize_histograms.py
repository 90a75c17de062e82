#!/usr/bin/env python
"""Writes tests/golden/fullsize_<config>.txt: the whole DD / DR / RR histograms of BASELINE.json's five
configurations at full size (scale 1), computed by the CPU oracle alone.

    python tests/golden/make_fullsize_histograms.py [config ...]      (default: all five)

This script calls only oracle/ (the checker) and workloads/ (the seeded input generators); nothing of the
CUDA path is imported, so no stored value comes from the code under test.  tests/test_gpu_fullsize.py
compares the library's full-size histograms with these files bin for bin (u64 equal; weighted sums to
1e-12), after checking -- by the hashes stored here -- that it counts the very same canonical vectors,
weights and edges.  This is the one-off whole-histogram CPU/GPU comparison of PAPER.md:115 (sect. 2.2:
the paper compares its CPU and GPU histograms bin by bin), with exact parity as the bar.

Oracle function per configuration (acf_oracle.c): the plain O(N^2) loop `oracle_pair_count_rows` for tiny,
clustered_patch and full_sky (weighted: long-double row sums); the Dec + RA window variant
`oracle_pair_count_cellwindow` for survey_scale and pruning_stress (theta_max of 3 and 1 degrees: the plain
loop would need 4.5e12 and 1.28e14 pairs), which tests/test_oracle_pins.py pins to the plain loop.
Wall time on the 8-core build box: seconds (tiny), minutes (clustered_patch, survey_scale,
pruning_stress), about an hour and a half (full_sky, 2.0e12 weighted pairs).
"""
import hashlib
import os
import sys
import time

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from oracle import oracle as O  # noqa: E402
from workloads import make_config  # noqa: E402

CELLWINDOW = {"survey_scale", "pruning_stress"}
ALL = ["tiny", "clustered_patch", "survey_scale", "full_sky", "pruning_stress"]


def sha(a) -> str:
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()


def run(name: str) -> str:
    w = make_config(name, 1.0)
    O.set_num_threads(len(os.sched_getaffinity(0)))
    xd, xr = O.radec_to_xyz(w.ra_d, w.dec_d), O.radec_to_xyz(w.ra_r, w.dec_r)
    weighted = w.w_d is not None
    lines = [
        "# Whole-catalogue histograms of the `%s` configuration at scale 1 (BASELINE.json), by the CPU oracle." % name,
        "# Written by tests/golden/make_fullsize_histograms.py, which calls only oracle/ and workloads/.",
        "# The sha256 lines are of the float64 canonical vectors [x|y|z] (oracle_radec_to_xyz), the float32 weights",
        "# and the float64 cosine edges the counts were made from.  Counts are u64; weighted sums are C99 hex floats.",
    ]
    rec = {"n_d": w.n_d, "n_r": w.n_r, "nbins": w.nbins}
    hashes = {"xyz_d": sha(xd), "xyz_r": sha(xr), "cos_edges": sha(w.cos_edges)}
    if weighted:
        hashes.update({"w_d": sha(w.w_d), "w_r": sha(w.w_r)})
    out = {}
    timing = []
    for key, (a, ra, da, wa, b, rb, db, wb, auto) in {
            "dd": (xd, w.ra_d, w.dec_d, w.w_d, None, None, None, None, True),
            "dr": (xd, w.ra_d, w.dec_d, w.w_d, xr, w.ra_r, w.dec_r, w.w_r, False),
            "rr": (xr, w.ra_r, w.dec_r, w.w_r, None, None, None, None, True)}.items():
        t0 = time.time()
        if name in CELLWINDOW:
            c = O.pair_count_cellwindow(a, ra, da, b, rb, db, w.cos_edges, auto)
            func = "oracle_pair_count_cellwindow"
        elif weighted:
            c, s = O.pair_count(a, b, w.cos_edges, auto, w_a=wa, w_b=wb)
            out["w" + key] = s
            func = "oracle_pair_count_rows (weighted)"
        else:
            c = O.pair_count(a, b, w.cos_edges, auto)
            func = "oracle_pair_count_rows"
        out[key] = c
        timing.append("%s %.1f s" % (key.upper(), time.time() - t0))
        print(name, key, "%.1f s" % (time.time() - t0), flush=True)
    lines.append("# %s, %d threads: %s" % (func, O.num_threads(), ", ".join(timing)))
    for k, v in rec.items():
        lines.append("%s %d" % (k, v))
    for k, v in hashes.items():
        lines.append("sha256_%s %s" % (k, v))
    for key in ("dd", "dr", "rr"):
        lines.append(key + " " + " ".join(str(int(v)) for v in out[key]))
    if weighted:
        for key in ("wdd", "wdr", "wrr"):
            lines.append(key + " " + " ".join(float(v).hex() for v in out[key]))
    path = os.path.join(HERE, "fullsize_%s.txt" % name)
    with open(path + ".tmp", "w") as f:
        f.write("\n".join(lines) + "\n")
    os.replace(path + ".tmp", path)
    return path


if __name__ == "__main__":
    for n in (sys.argv[1:] or ALL):
        if n not in ALL:
            raise SystemExit("unknown configuration %r (one of %s)" % (n, ", ".join(ALL)))
        print("wrote", run(n), flush=True)
