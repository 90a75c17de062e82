"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times
(acf_pair_count / acf_pair_count_weighted on whole catalogues):

  * the WHOLE DD / DR / RR histograms of the full calls against tests/golden/fullsize_<config>.txt, written by the
    CPU oracle alone (tests/golden/make_fullsize_histograms.py, the paper's own bin-by-bin CPU/GPU
    comparison, with exact parity as the bar), through every fast kernel;
  * sampled outputs the oracle can compute one by one: the histogram of row blocks
    (acf_pair_count_rows vs oracle rows), u64-equal -- narrow blocks (ragged tiles: the masked paths) and
    blocks of more than two whole tiles plus a ragged rest (full tiles and full groups: the unmasked loops
    that classify nearly all pairs of a full call);
  * properties that hold at any size, on the full calls: the single-edge window path and the
    table path (two different kernels paths) give identical u64 counts; DR(a, b) == DR(b, a);
    row-block additivity; totals; the closed-form expectation on the uniform sphere.

Run on the B200 box:  python -m pytest tests/test_gpu_fullsize.py -m gpu -x -q
"""
import hashlib
import os

import numpy as np
import pytest

from conftest import GOLDEN, read_golden
from workloads import make_config

pytestmark = pytest.mark.gpu

WSUM_RTOL = 1e-12


@pytest.fixture(scope="module")
def acf():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_1208_3658_b200 as P
    return P


@pytest.fixture(scope="module")
def ctx(acf):
    c = acf.acf_create(0)
    yield c
    acf.acf_destroy(c)


class Dev:
    """Device copies of one workload (uploaded once per test)."""

    def __init__(self, acf, w, by_sky_cell=False):
        import torch
        if by_sky_cell:
            w = in_sky_cell_order(w)
        self.w = w
        self.h_xd, self.h_xr = acf.acf_radec_to_xyz(w.ra_d, w.dec_d), acf.acf_radec_to_xyz(w.ra_r, w.dec_r)
        self.xd, self.xr = torch.from_numpy(self.h_xd).cuda(), torch.from_numpy(self.h_xr).cuda()
        self.wd = torch.from_numpy(w.w_d).cuda() if w.w_d is not None else None
        self.wr = torch.from_numpy(w.w_r).cuda() if w.w_r is not None else None


def in_sky_cell_order(w):
    """The same catalogues with their points listed Dec band by Dec band (2 degrees) and by RA inside a band, as
    a survey's file would: a run of consecutive rows is then a compact piece of sky, and a row block prepared
    as a catalogue of its own has the compact groups of points that a whole catalogue has after its sort."""
    import copy
    out = copy.copy(w)
    for s in ("d", "r"):
        ra, dec = getattr(w, "ra_" + s), getattr(w, "dec_" + s)
        order = np.lexsort((ra, np.floor(dec / 2.0)))
        setattr(out, "ra_" + s, ra[order].copy())
        setattr(out, "dec_" + s, dec[order].copy())
        if getattr(w, "w_" + s) is not None:
            setattr(out, "w_" + s, getattr(w, "w_" + s)[order].copy())
    return out


def count(acf, ctx, d, which, rows=None, windows=1, kernel=None, bulk=0):
    """-> (u64 counts, f64 sums or None, stats) of DD / DR / RD / RR on the device."""
    import torch
    a, wa, b, wb, auto = {"dd": (d.xd, d.wd, None, None, True), "dr": (d.xd, d.wd, d.xr, d.wr, False),
                          "rd": (d.xr, d.wr, d.xd, d.wd, False), "rr": (d.xr, d.wr, None, None, True)}[which]
    acf.acf_set_option(ctx, acf.ACF_OPT_WINDOWS, windows)
    acf.acf_set_option(ctx, acf.ACF_OPT_KERNEL, acf.ACF_KERNEL_AUTO if kernel is None else kernel)
    acf.acf_set_option(ctx, acf.ACF_OPT_BULK, bulk)
    try:
        n_a = a.numel() // 3
        lo, hi = rows if rows is not None else (0, n_a)
        out = acf.acf_pair_count_rows(ctx, a, wa, lo, hi, b, wb, d.w.cos_edges, auto)
        torch.cuda.synchronize()
        st = acf.acf_get_stats(ctx)
    finally:
        acf.acf_set_option(ctx, acf.ACF_OPT_WINDOWS, 1)
        acf.acf_set_option(ctx, acf.ACF_OPT_KERNEL, acf.ACF_KERNEL_AUTO)
        acf.acf_set_option(ctx, acf.ACF_OPT_BULK, 0)
    if wa is None:
        return acf.counts_to_numpy(out), None, st
    return acf.counts_to_numpy(out[0]), out[1].cpu().numpy(), st


# configurations whose theta_max is a few degrees: the oracle's Dec + RA window loop (pinned to the plain
# loop in tests/test_oracle_pins.py) makes wide row blocks of 2M and 8M-point catalogues affordable
CELLWINDOW = {"survey_scale", "pruning_stress"}


def oracle_rows(oracle, d, which, rows):
    w = d.w
    a, ra, da, wa, b, rb, db, wb, auto = {
        "dd": (d.h_xd, w.ra_d, w.dec_d, w.w_d, None, None, None, None, True),
        "dr": (d.h_xd, w.ra_d, w.dec_d, w.w_d, d.h_xr, w.ra_r, w.dec_r, w.w_r, False),
        "rr": (d.h_xr, w.ra_r, w.dec_r, w.w_r, None, None, None, None, True)}[which]
    if w.name in CELLWINDOW and wa is None:
        return oracle.pair_count_cellwindow(a, ra, da, b, rb, db, w.cos_edges, auto, rows=rows)
    return oracle.pair_count(a, b, w.cos_edges, auto, w_a=wa, w_b=wb, rows=rows)


def sample_blocks(n, width):
    """Row blocks at the start, around the middle (straddling a tile boundary) and at the ragged end."""
    mid = (n // 2 // 1024) * 1024
    return [(0, width), (max(0, mid - width // 2), min(n, mid + width // 2)), (n - width, n)]


def wide_blocks(n, seed):
    """Row blocks of more than two whole tiles of 1024 plus a ragged rest: as catalogues of their own they are
    full i-tiles of full groups, which the kernels run through their unmasked loops (the single-edge window
    loop in registers, the multi-edge chunks, the unmasked table path) at the full density of the j side."""
    rng = np.random.default_rng(seed)
    width = 2048 + 529
    mid = (n // 2 // 1024) * 1024 - 1300
    off = int(rng.integers(0, n - width))
    return [(0, width), (mid, mid + width + 5), (off, off + width)]


def read_fullsize_golden(name):
    """tests/golden/fullsize_<name>.txt -> dict, or None if the file is not there."""
    if not os.path.exists(os.path.join(GOLDEN, "fullsize_%s.txt" % name)):
        return None
    g = {}
    for r in read_golden("fullsize_%s.txt" % name):
        if r[0] in ("dd", "dr", "rr"):
            g[r[0]] = np.array([int(v) for v in r[1:]], dtype=np.uint64)
        elif r[0] in ("wdd", "wdr", "wrr"):
            g[r[0]] = np.array([float.fromhex(v) for v in r[1:]], dtype=np.float64)
        elif r[0].startswith("sha256_"):
            g[r[0]] = r[1]
        else:
            g[r[0]] = int(r[1])
    return g


def sha(a):
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()


@pytest.mark.parametrize("name,width", [("tiny", 256), ("clustered_patch", 192), ("survey_scale", 96),
                                        ("full_sky", 96), ("pruning_stress", 48)])
def test_fullsize_sampled_rows_and_properties(acf, ctx, oracle, name, width):
    w = make_config(name, 1.0)
    d = Dev(acf, w)
    assert d.h_xd.tobytes() == oracle.radec_to_xyz(w.ra_d, w.dec_d).tobytes()
    weighted = w.w_d is not None

    # ---- sampled outputs: row blocks against the oracle, DD / DR / RR
    for which, n in (("dd", w.n_d), ("dr", w.n_d), ("rr", w.n_r)):
        for rows in sample_blocks(n, width):
            got_c, got_w, _ = count(acf, ctx, d, which, rows=rows)
            want = oracle_rows(oracle, d, which, rows)
            if weighted:
                assert got_c.tolist() == want[0].tolist(), (which, rows)
                np.testing.assert_allclose(got_w, want[1], rtol=WSUM_RTOL, atol=0, err_msg="%s %s" % (which, rows))
            else:
                assert got_c.tolist() == want.tolist(), (which, rows)
    # ---- wide blocks (full tiles, full groups: the unmasked loops), through both fast kernels, on the
    # catalogues listed in sky order so that a block is a compact piece of sky (single-edge windows)
    ds = Dev(acf, w, by_sky_cell=True)
    for which, n in (("dd", w.n_d), ("dr", w.n_d), ("rr", w.n_r)):
        for rows in wide_blocks(n, 7 + len(name)):
            want = oracle_rows(oracle, ds, which, rows)
            for kern in (acf.ACF_KERNEL_WINDOW, acf.ACF_KERNEL_TABLE):
                got_c, got_w, st = count(acf, ctx, ds, which, rows=rows, kernel=kern)
                if weighted:
                    assert got_c.tolist() == want[0].tolist(), (which, rows, kern)
                    np.testing.assert_allclose(got_w, want[1], rtol=WSUM_RTOL, atol=0, err_msg="%s %s" % (which, rows))
                else:
                    assert got_c.tolist() == want.tolist(), (which, rows, kern)
                if name == "full_sky" and kern == acf.ACF_KERNEL_WINDOW:
                    # the unmasked single-edge loop did classify most of the block's pairs
                    assert st["pairs_window"] > 0.3 * st["pairs_evaluated"], st
    del ds

    # ---- the full calls, as bench.py makes them
    full = {k: count(acf, ctx, d, k) for k in ("dd", "dr", "rr")}
    # the whole histograms against the CPU oracle's (tests/golden/fullsize_<name>.txt)
    g = read_fullsize_golden(name)
    assert g is not None or name not in ("tiny", "clustered_patch"), "tests/golden/fullsize_%s.txt is missing" % name
    if g is not None:
        assert (g["n_d"], g["n_r"], g["nbins"]) == (w.n_d, w.n_r, w.nbins)
        assert g["sha256_xyz_d"] == sha(d.h_xd) and g["sha256_xyz_r"] == sha(d.h_xr) and g["sha256_cos_edges"] == sha(w.cos_edges)
        if weighted:
            assert g["sha256_w_d"] == sha(w.w_d) and g["sha256_w_r"] == sha(w.w_r)
        for k in ("dd", "dr", "rr"):
            assert full[k][0].tolist() == g[k].tolist(), k
            if weighted:
                np.testing.assert_allclose(full[k][1], g["w" + k], rtol=WSUM_RTOL, atol=0, err_msg=k)
    for k, (c, s, st) in full.items():
        n_a = w.n_d if k != "rr" else w.n_r
        nominal = n_a * (n_a - 1) // 2 if k != "dr" else w.n_d * w.n_r
        assert st["pairs_nominal"] == nominal and 0 < st["pairs_evaluated"] <= nominal
        assert int(c.sum()) <= nominal
    # three independent classification codes, bit for bit: the window kernel (edges of a window against
    # register tallies), the table kernel with its single-edge windows, and the table kernel's cell table alone
    for k in ("dd", "dr", "rr"):
        for kern, windows in ((acf.ACF_KERNEL_WINDOW, 1), (acf.ACF_KERNEL_TABLE, 1), (acf.ACF_KERNEL_TABLE, 0)):
            if k == "rr" and windows == 0:
                continue
            c2, s2, st2 = count(acf, ctx, d, k, windows=windows, kernel=kern)
            assert windows == 1 or st2["pairs_window"] == 0
            nominal = {"dd": w.n_d * (w.n_d - 1) // 2, "dr": w.n_d * w.n_r, "rr": w.n_r * (w.n_r - 1) // 2}[k]
            assert 0 < st2["pairs_evaluated"] <= nominal    # (the kernels prune groups of points to different depths)
            assert c2.tolist() == full[k][0].tolist(), (k, kern, windows)
            if weighted:
                np.testing.assert_allclose(s2, full[k][1], rtol=WSUM_RTOL, atol=0)
    # swapping the catalogues of a cross count changes every tile, window and work item, not the result
    c3, s3, _ = count(acf, ctx, d, "rd")
    assert c3.tolist() == full["dr"][0].tolist()
    if weighted:
        np.testing.assert_allclose(s3, full["dr"][1], rtol=WSUM_RTOL, atol=0)
    # additivity over row blocks
    cut = (w.n_d // 3 // 1000) * 1000 + 17
    parts = count(acf, ctx, d, "dd", rows=(0, cut))[0] + count(acf, ctx, d, "dd", rows=(cut, w.n_d))[0]
    assert parts.tolist() == full["dd"][0].tolist()

    if name == "full_sky":
        # groups of points counted as a whole where their caps allow it (ACF_OPT_BULK): the same histograms
        cb, sb, stb = count(acf, ctx, d, "dr", kernel=acf.ACF_KERNEL_WINDOW, bulk=1)
        assert cb.tolist() == full["dr"][0].tolist()
        np.testing.assert_allclose(sb, full["dr"][1], rtol=WSUM_RTOL, atol=0)
        assert stb["pairs_bulk"] > 0.3 * stb["pairs_nominal"] and stb["pairs_bulk"] + stb["pairs_evaluated"] == stb["pairs_nominal"]
        # uniform sphere: cos(theta) is uniform on [-1, 1] => E[count_k] = N_pairs (e_k - e_k+1) / 2
        e = w.cos_edges
        for k, npairs in (("dd", w.n_d * (w.n_d - 1) // 2), ("dr", w.n_d * w.n_r)):
            expect = npairs * (e[:-1] - e[1:]) / 2.0
            assert np.all(np.abs(full[k][0].astype(np.float64) - expect) <= 6.0 * np.sqrt(expect) + 1.0)
            # the range starts at 1 arcmin: the pairs closer than that are the only ones missing
            assert npairs - int(full[k][0].sum()) <= 12 * npairs * (1.0 - e[0]) / 2.0 + 50
        # weighted: E[w_i w_j] = exp(sigma^2) for independent lognormal(0, sigma) weights
        ratio = full["dr"][1] / np.maximum(1, full["dr"][0])
        big = full["dr"][0] > 10 ** 8
        assert np.all(np.abs(ratio[big] / np.exp(0.09) - 1.0) < 5e-3)
    # the estimator through the library and the oracle on the same counts
    wt = acf.acf_wtheta(full["dd"][0], full["dr"][0], full["rr"][0], w.n_d, w.n_r)
    wo = oracle.wtheta(full["dd"][0], full["dr"][0], full["rr"][0], w.n_d, w.n_r)
    np.testing.assert_allclose(wt, wo, rtol=0, atol=1e-10, equal_nan=True)


def test_two_million_points_mid_kernel_flush(acf, ctx):
    """2M x 2M weighted DR (4e12 pairs): every CTA walks more j-tiles than a u32 histogram row may take,
    so the rows are flushed to global memory in mid-kernel.  The two fast kernels (independent codes) must
    agree bit for bit; the counts must follow the uniform-sphere law and add up to all pairs beyond 1'."""
    import torch
    w = make_config("full_sky", 2.0)
    d = Dev(acf, w)
    res = {}
    for kern in (acf.ACF_KERNEL_WINDOW, acf.ACF_KERNEL_TABLE):
        res[kern] = count(acf, ctx, d, "dr", kernel=kern)
    c, s, st = res[acf.ACF_KERNEL_WINDOW]
    c2, s2, _ = res[acf.ACF_KERNEL_TABLE]
    assert c.tolist() == c2.tolist()
    np.testing.assert_allclose(s, s2, rtol=WSUM_RTOL, atol=0)
    npairs = w.n_d * w.n_r
    e = w.cos_edges
    expect = npairs * (e[:-1] - e[1:]) / 2.0
    assert np.all(np.abs(c.astype(np.float64) - expect) <= 6.0 * np.sqrt(expect) + 1.0)
    assert 0 <= npairs - int(c.sum()) <= 12 * npairs * (1.0 - e[0]) / 2.0 + 50
    assert st["pairs_evaluated"] == npairs
