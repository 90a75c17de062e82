"""GPU parity: the CUDA path (through the C ABI via the thin binding) against the CPU oracle,
element by element on the same seeded inputs.  Counts must be equal as u64 integers; weighted
sums within 1e-12 relative; w(theta) within 1e-10 absolute (north_star tolerances).

Run on the B200 box:  python -m pytest tests -m gpu -x -q
"""
import math

import numpy as np
import pytest

from workloads import cos_edges_from_theta_deg, full_sky, linear_theta_edges_deg, log_theta_edges_deg, make_config
from workloads.catalogs import lognormal_weights, uniform_patch

pytestmark = pytest.mark.gpu

WSUM_RTOL = 1e-12   # north_star: weighted sums agree to <= 1e-12 relative
WTHETA_ATOL = 1e-10  # north_star: w(theta) agrees to <= 1e-10 absolute


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


def dev(x, dtype=None):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(x))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


def gpu_counts(acf, ctx, xa, xb, edges, auto, wa=None, wb=None, rows=None, kernel=None):
    """Run one pair count on the device and bring the result back as numpy."""
    import torch
    if kernel is not None:
        acf.acf_set_option(ctx, acf.ACF_OPT_KERNEL, kernel)
    try:
        da = dev(xa)
        db = None if auto else dev(xb)
        n_a = xa.size // 3
        i0, i1 = (0, n_a) if rows is None else rows
        if wa is None:
            if rows is None:
                out = acf.acf_pair_count(ctx, da, db, edges, auto)
            else:
                out = acf.acf_pair_count_rows(ctx, da, None, i0, i1, db, None, edges, auto)
            torch.cuda.synchronize()
            return acf.counts_to_numpy(out)
        dwa = dev(wa)
        dwb = None if auto else dev(wb)
        c, w = acf.acf_pair_count_rows(ctx, da, dwa, i0, i1, db, dwb, edges, auto)
        torch.cuda.synchronize()
        return acf.counts_to_numpy(c), w.cpu().numpy()
    finally:
        if kernel is not None:
            acf.acf_set_option(ctx, acf.ACF_OPT_KERNEL, acf.ACF_KERNEL_AUTO)


def soa(v):
    v = np.asarray(v, dtype=np.float64)
    return np.concatenate([v[:, 0], v[:, 1], v[:, 2]])


def test_canonical_vectors_bit_equal(acf, oracle):
    # both sides call glibc sin/cos on the same doubles: the arrays must be identical bit for bit
    ra, dec = full_sky(20000, 3)
    a = acf.acf_radec_to_xyz(ra, dec)
    b = oracle.radec_to_xyz(ra, dec)
    assert a.tobytes() == b.tobytes()


@pytest.mark.parametrize("kernel", ["auto", "fp64", "table", "window"])
@pytest.mark.parametrize("name,scale", [("tiny", 0.5), ("clustered_patch", 0.03), ("survey_scale", 0.006),
                                        ("full_sky", 0.008), ("pruning_stress", 0.0012)])
def test_config_parity(acf, ctx, oracle, name, scale, kernel):
    """All five BASELINE configurations at a size the oracle finishes in seconds: several tiles
    and ragged tails on both catalogues; DD, DR, RR and the estimator."""
    kern = {"auto": acf.ACF_KERNEL_AUTO, "fp64": acf.ACF_KERNEL_FP64, "table": acf.ACF_KERNEL_TABLE, "window": acf.ACF_KERNEL_WINDOW}[kernel]
    w = make_config(name, scale)
    xd, xr = acf.acf_radec_to_xyz(w.ra_d, w.dec_d), acf.acf_radec_to_xyz(w.ra_r, w.dec_r)
    assert xd.tobytes() == oracle.radec_to_xyz(w.ra_d, w.dec_d).tobytes()
    res = {}
    for key, (a, b, auto, wa, wb) in {"dd": (xd, None, True, w.w_d, None), "dr": (xd, xr, False, w.w_d, w.w_r),
                                      "rr": (xr, None, True, w.w_r, None)}.items():
        want = oracle.pair_count(a, b, w.cos_edges, auto, w_a=wa, w_b=wb)
        got = gpu_counts(acf, ctx, a, b, w.cos_edges, auto, wa=wa, wb=wb, kernel=kern)
        if wa is None:
            assert got.tolist() == want.tolist(), key
            res[key] = got
        else:
            assert got[0].tolist() == want[0].tolist(), key
            np.testing.assert_allclose(got[1], want[1], rtol=WSUM_RTOL, atol=0, err_msg=key)
            res[key] = got[0]
            res["w" + key] = got[1]
        st = acf.acf_get_stats(ctx)
        n_a = a.size // 3
        assert st["pairs_nominal"] == (n_a * (n_a - 1) // 2 if auto else n_a * (b.size // 3))
        assert st["kernel_launches"] >= 1
    assert int(res["dd"].sum()) > 0 and int(res["rr"].sum()) > 0
    wt = acf.acf_wtheta(res["dd"], res["dr"], res["rr"], w.n_d, w.n_r)
    wo = oracle.wtheta(res["dd"], res["dr"], res["rr"], w.n_d, w.n_r)
    assert np.array_equal(np.isnan(wt), np.isnan(wo))
    np.testing.assert_allclose(wt[~np.isnan(wt)], wo[~np.isnan(wo)], rtol=0, atol=WTHETA_ATOL)
    if w.w_d is not None:
        ww = acf.acf_wtheta_weighted(res["wdd"], res["wdr"], res["wrr"], w.w_d, w.w_r)
        wwo = oracle.wtheta_weighted(res["wdd"], res["wdr"], res["wrr"], w.w_d, w.w_r)
        np.testing.assert_allclose(ww, wwo, rtol=0, atol=WTHETA_ATOL, equal_nan=True)


def test_polyhedra_and_full_range(acf, ctx, oracle):
    phi = (1 + 5 ** 0.5) / 2
    ico = []
    for s1 in (-1, 1):
        for s2 in (-1, 1):
            ico += [(0, s1, s2 * phi), (s1, s2 * phi, 0), (s2 * phi, 0, s1)]
    ico = np.array(ico, dtype=np.float64)
    ico /= np.linalg.norm(ico, axis=1, keepdims=True)
    xyz = soa(ico)
    edges = np.array([1.0, 0.0, -0.9, -1.0])
    assert gpu_counts(acf, ctx, xyz, None, edges, True).tolist() == [30, 30, 6]
    assert gpu_counts(acf, ctx, xyz, xyz, edges, False).tolist() == [72, 60, 12]   # + 12 self pairs at c = 1
    # totals when the bins cover [0, 180] deg: n(n-1)/2 and n_a n_b
    ra, dec = full_sky(3000, 41)
    rb, db_ = full_sky(2500, 42)
    a, b = acf.acf_radec_to_xyz(ra, dec), acf.acf_radec_to_xyz(rb, db_)
    full = cos_edges_from_theta_deg(np.array([0.0, 0.01, 1.0, 30.0, 90.0, 179.0, 180.0]))
    ca = gpu_counts(acf, ctx, a, None, full, True)
    cb = gpu_counts(acf, ctx, a, b, full, False)
    assert int(ca.sum()) == 3000 * 2999 // 2 and int(cb.sum()) == 3000 * 2500
    assert ca.tolist() == oracle.pair_count(a, None, full, True).tolist()
    assert cb.tolist() == oracle.pair_count(a, b, full, False).tolist()
    assert cb.tolist() == gpu_counts(acf, ctx, b, a, full, False).tolist()       # swap symmetry


@pytest.mark.parametrize("kernel", ["auto", "fp64", "table", "window"])
def test_edge_inclusivity_adversarial(acf, ctx, oracle, kernel):
    """Pairs whose cosine is exactly an edge, or one ulp either side, through the xyz entry point:
    a = (1,0,0), b = (c, sqrt(1-c^2), 0) makes the defined pair cosine equal c exactly."""
    kern = {"auto": acf.ACF_KERNEL_AUTO, "fp64": acf.ACF_KERNEL_FP64, "table": acf.ACF_KERNEL_TABLE, "window": acf.ACF_KERNEL_WINDOW}[kernel]
    edges = cos_edges_from_theta_deg(log_theta_edges_deg(0.05, 170.0, 12))
    cs = []
    for e in edges:
        cs += [e, np.nextafter(e, 2.0), np.nextafter(e, -2.0), e + 3e-7, e - 3e-7, e + 1e-8, e - 1e-8]
    cs += [1.0, -1.0, 0.0, 0.5]
    cs = np.clip(np.array(cs), -1.0, 1.0)
    b = np.stack([cs, np.sqrt(np.maximum(0.0, 1.0 - cs * cs)), np.zeros_like(cs)], axis=1)
    # renormalising would move c; instead keep norms within the validator's 1e-6 (they are ~1e-16 off)
    xa = soa([(1.0, 0.0, 0.0)])
    xb = soa(b)
    want = oracle.pair_count(xa, xb, edges, False)
    got = gpu_counts(acf, ctx, xa, xb, edges, False, kernel=kern)
    assert got.tolist() == want.tolist()
    got = gpu_counts(acf, ctx, xb, xa, edges, False, kernel=kern)
    assert got.tolist() == want.tolist()
    # and one pair at a time, so that a compensating double error cannot hide
    for c, row in zip(cs[:21], b[:21]):
        one = soa([row])
        assert gpu_counts(acf, ctx, xa, one, edges, False, kernel=kern).tolist() == oracle.pair_count(xa, one, edges, False).tolist(), c


def great_circle_grid(n, first, step_rad, jitter=None):
    """n points on the great circle z = 0 at longitudes (first + k) * step_rad (+ jitter[k]): pairs of such points
    have separations that are whole multiples of the step (plus the jitter), whatever their position."""
    phi = (first + np.arange(n)) * step_rad
    if jitter is not None:
        phi = phi + jitter
    return soa(np.stack([np.cos(phi), np.sin(phi), np.zeros(n)], axis=1))


@pytest.mark.parametrize("nb_arcsec,what", [(600, "single-edge windows"), (47, "windows of several edges")])
@pytest.mark.parametrize("kernel", ["auto", "table", "window"])
def test_near_edge_pairs_on_the_unmasked_paths(acf, ctx, oracle, kernel, nb_arcsec, what):
    """Adversarial pairs at full tiles and full groups, i.e. through the unmasked loops that classify nearly
    every pair of a full-size call (the one-point catalogues of test_edge_inclusivity_adversarial reach the
    masked variants only).  3 tiles of i-points and 2 tiles + a ragged rest of j-points sit on a 1-arcsec grid
    along a great circle; the bin edges are whole multiples of the grid step, so every j-point makes a pair
    with several i-points whose separation is an edge up to a chosen offset: 0, a few ulps, and offsets of the
    cosine around the guard bands of the kernels (3.0e-7 / 7.0e-7 window kernel, 4.5e-7 / 6.7e-7 table kernel).
    Counts must equal the oracle's, cross and auto."""
    kern = {"auto": acf.ACF_KERNEL_AUTO, "table": acf.ACF_KERNEL_TABLE, "window": acf.ACF_KERNEL_WINDOW}[kernel]
    h = math.radians(1.0 / 3600.0)
    n_i, n_j = 3 * 1024, 2 * 1024 + 300
    sep0 = 2 * 3600                                  # the j arc starts 2 degrees after the i arc
    m_edges = np.arange(sep0 - n_i - nb_arcsec, sep0 + n_j + 2 * nb_arcsec, nb_arcsec)   # edges, in grid steps
    m_edges = m_edges[m_edges > 0]
    edges = np.cos(m_edges * h)
    assert np.all(np.diff(edges) < 0)
    # offsets of the pair cosine from the edge; d(cos) = -sin(theta) d(theta), theta ~ 2 degrees
    offs = np.array([0.0, 1e-16, -1e-16, 1e-13, -1e-13, 1e-8, -1e-8, 1e-7, -1e-7, 2.5e-7, -2.5e-7, 2.7e-7, -2.7e-7,
                     2.9e-7, -2.9e-7, 3.0e-7, -3.0e-7, 3.1e-7, -3.1e-7, 4.4e-7, -4.6e-7, 6.6e-7, -6.8e-7, 7.1e-7, -6.9e-7])
    jit = -offs[np.arange(n_j) % offs.size] / math.sin(sep0 * h)
    xa = great_circle_grid(n_i, 0, h)
    xb = great_circle_grid(n_j, sep0, h, jit)
    want = oracle.pair_count(xa, xb, edges, False)
    got = gpu_counts(acf, ctx, xa, xb, edges, False, kernel=kern)
    st = acf.acf_get_stats(ctx)
    assert got.tolist() == want.tolist(), what
    assert st["pairs_fp64"] + st["pairs_chord"] > n_j, st        # the near-edge pairs were seen as such
    if kernel == "window" and nb_arcsec == 600:
        assert st["pairs_window"] > 0.4 * n_i * n_j, st          # the unmasked single-edge loop ran
    got = gpu_counts(acf, ctx, xb, xa, edges, False, kernel=kern)
    assert got.tolist() == want.tolist(), what
    # weighted, through the packed accumulators of the window kernel (and pair by pair in the table kernel)
    rng = np.random.default_rng(5)
    wa, wb = rng.uniform(0.5, 2.0, n_i).astype(np.float32), rng.uniform(0.5, 2.0, n_j).astype(np.float32)
    got = gpu_counts(acf, ctx, xa, xb, edges, False, wa=wa, wb=wb, kernel=kern)
    want_w = oracle.pair_count(xa, xb, edges, False, w_a=wa, w_b=wb)
    assert got[0].tolist() == want_w[0].tolist() == want.tolist()
    np.testing.assert_allclose(got[1], want_w[1], rtol=WSUM_RTOL, atol=0)
    # auto-count of both arcs together: diagonal tiles (i < j mask) beside unmasked off-diagonal ones
    xab = np.concatenate([xa.reshape(3, -1), xb.reshape(3, -1)], axis=1).reshape(-1)
    near = np.cos(np.arange(1, 40) * 97 * h)                      # edges inside the arcs as well
    e2 = np.sort(np.concatenate([edges, near]))[::-1].copy()
    assert gpu_counts(acf, ctx, xab, None, e2, True, kernel=kern).tolist() == oracle.pair_count(xab, None, e2, True).tolist()


def test_duplicates_and_clamp(acf, ctx, oracle):
    # coincident points: c may round above 1 and is clamped; counted iff e_0 = 1
    ra, dec = full_sky(500, 7)
    ra = np.concatenate([ra, ra[:100]])
    dec = np.concatenate([dec, dec[:100]])
    a = acf.acf_radec_to_xyz(ra, dec)
    for edges in (cos_edges_from_theta_deg(np.array([0.0, 1.0, 90.0, 180.0])),
                  cos_edges_from_theta_deg(np.array([1e-6, 1.0, 90.0, 180.0]))):
        want = oracle.pair_count(a, None, edges, True).tolist()
        for kern in (acf.ACF_KERNEL_TABLE, acf.ACF_KERNEL_WINDOW):
            assert gpu_counts(acf, ctx, a, None, edges, True, kernel=kern).tolist() == want


@pytest.mark.parametrize("kernel", ["table", "window"])
def test_degenerate_sizes(acf, ctx, kernel):
    import torch
    acf.acf_set_option(ctx, acf.ACF_OPT_KERNEL, {"table": acf.ACF_KERNEL_TABLE, "window": acf.ACF_KERNEL_WINDOW}[kernel])
    edges = np.array([1.0, 0.0, -1.0])
    one = soa([(0.0, 0.0, 1.0)])
    two = soa([(0.0, 0.0, 1.0), (0.0, 1.0, 0.0)])
    empty = np.zeros(0)
    assert gpu_counts(acf, ctx, one, None, edges, True).tolist() == [0, 0]          # n = 1, auto
    assert gpu_counts(acf, ctx, two, None, edges, True).tolist() == [0, 1]          # c = 0 = e_1 -> bin 1 (c <= e_1)
    assert gpu_counts(acf, ctx, one, two, edges, False).tolist() == [1, 1]          # c = 1 -> bin 0, c = 0 -> bin 1
    out = acf.acf_pair_count(ctx, torch.zeros(0, dtype=torch.float64, device="cuda"), None, edges, True)
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [0, 0]
    assert gpu_counts(acf, ctx, two, None, edges, True, rows=(1, 1)).tolist() == [0, 0]
    ones = np.ones(2, np.float32)
    c, ws = gpu_counts(acf, ctx, two, None, edges, True, wa=ones)                   # weighted, one pair
    assert c.tolist() == [0, 1] and ws.tolist() == [0.0, 1.0]
    acf.acf_set_option(ctx, acf.ACF_OPT_KERNEL, acf.ACF_KERNEL_AUTO)


@pytest.mark.parametrize("kernel", ["table", "window"])
def test_row_ranges_add_up(acf, ctx, oracle, kernel):
    # the pair matrix cut into sub-matrices; counts are additive over row ranges
    kern = {"table": acf.ACF_KERNEL_TABLE, "window": acf.ACF_KERNEL_WINDOW}[kernel]
    w = make_config("clustered_patch", 0.02)
    xd, xr = acf.acf_radec_to_xyz(w.ra_d, w.dec_d), acf.acf_radec_to_xyz(w.ra_r, w.dec_r)
    n = w.n_d
    cuts = [0, 1, 777, 1024, 2049, n]
    for b, auto in ((None, True), (xr, False)):
        whole = gpu_counts(acf, ctx, xd, b, w.cos_edges, auto, kernel=kern)
        parts = np.zeros_like(whole)
        for lo, hi in zip(cuts[:-1], cuts[1:]):
            p = gpu_counts(acf, ctx, xd, b, w.cos_edges, auto, rows=(lo, hi), kernel=kern)
            assert p.tolist() == oracle.pair_count(xd, b, w.cos_edges, auto, rows=(lo, hi)).tolist()
            parts += p
        assert parts.tolist() == whole.tolist()


def test_linear_bins_many(acf, ctx, oracle):
    # the paper's benchmark used 254 bins; even spacing is one of its presets
    ra, dec = uniform_patch(6000, (0.0, 90.0), (0.0, 90.0), 5)   # the paper's octant footprint
    a = acf.acf_radec_to_xyz(ra, dec)
    for theta in (linear_theta_edges_deg(0.0, 120.0, 254), log_theta_edges_deg(0.01, 100.0, 254)):
        edges = cos_edges_from_theta_deg(theta)
        want = oracle.pair_count(a, None, edges, True).tolist()
        for kern in (acf.ACF_KERNEL_TABLE, acf.ACF_KERNEL_WINDOW):
            assert gpu_counts(acf, ctx, a, None, edges, True, kernel=kern).tolist() == want
    acf.acf_set_option(ctx, acf.ACF_OPT_KERNEL, acf.ACF_KERNEL_AUTO)


def test_fine_bins_dense_patch(acf, ctx, oracle):
    """Narrow bins on a dense patch: every window holds many edges, unweighted counts classify such windows pair by
    pair through the cell table of the squared chord length (64 cells per octave), weighted ones in passes of three
    edges.  Even bins put up to two edges into a cell at the far end, logarithmic ones do not."""
    ra, dec = uniform_patch(12000, (10.0, 12.0), (-1.0, 1.0), 17)
    rb, db = uniform_patch(9000, (10.0, 12.0), (-1.0, 1.0), 18)
    a, b = acf.acf_radec_to_xyz(ra, dec), acf.acf_radec_to_xyz(rb, db)
    wa = (1.0 + np.random.default_rng(19).integers(0, 16, 12000) / 16.0).astype(np.float32)
    wb = (1.0 + np.random.default_rng(20).integers(0, 16, 9000) / 16.0).astype(np.float32)
    acf.acf_set_option(ctx, acf.ACF_OPT_KERNEL, acf.ACF_KERNEL_WINDOW)
    # (the last: so many bins that the cell table gives up resolution for the rows' shared memory)
    for theta in (linear_theta_edges_deg(0.0, 1.0, 100), linear_theta_edges_deg(0.0, 1.5, 400), log_theta_edges_deg(1.0 / 3600, 2.0, 300),
                  linear_theta_edges_deg(0.0, 90.0, 640)):
        edges = cos_edges_from_theta_deg(theta)
        assert gpu_counts(acf, ctx, a, None, edges, True).tolist() == oracle.pair_count(a, None, edges, True).tolist()
        assert gpu_counts(acf, ctx, a, b, edges, False).tolist() == oracle.pair_count(a, b, edges, False).tolist()
        got = gpu_counts(acf, ctx, a, b, edges, False, wa=wa, wb=wb)
        want = oracle.pair_count(a, b, edges, False, w_a=wa, w_b=wb)
        assert got[0].tolist() == want[0].tolist()
        np.testing.assert_allclose(got[1], want[1], rtol=WSUM_RTOL, atol=0)
    st = acf.acf_get_stats(ctx)
    assert st["pairs_window"] < 0.5 * st["pairs_evaluated"]  # mostly windows of several edges
    acf.acf_set_option(ctx, acf.ACF_OPT_KERNEL, acf.ACF_KERNEL_AUTO)


@pytest.mark.parametrize("kernel", ["table", "window"])
def test_small_angles_chord_tier_and_inexact_norms(acf, ctx, oracle, kernel):
    """Bins far below the fp32 resolution of 1 - cos(theta) (0.02 arcsec to 2 arcmin): the fp32 chord
    length must decide most of what the cosine leaves open, and exactly.  Then the same points with
    norms off by up to 4e-7 (accepted by the validation): c = (|u|^2 + |v|^2 - s) / 2 moves every pair
    across several of these bins and the chord tier must step aside instead of trusting s."""
    kern = {"table": acf.ACF_KERNEL_TABLE, "window": acf.ACF_KERNEL_WINDOW}[kernel]
    rng = np.random.default_rng(71)
    # 300 tight clumps of 24 points (sigma = 10 arcsec) so that thousands of pairs fall into the bins
    ra0, dec0 = full_sky(300, 72)
    ra = (np.repeat(ra0, 24) + rng.normal(0, 10 / 3600, 7200) / np.maximum(0.05, np.cos(np.radians(np.repeat(dec0, 24))))) % 360.0
    dec = np.clip(np.repeat(dec0, 24) + rng.normal(0, 10 / 3600, 7200), -89.9, 89.9)
    a = acf.acf_radec_to_xyz(ra, dec)
    edges = cos_edges_from_theta_deg(log_theta_edges_deg(0.02 / 3600, 2.0 / 60, 36))
    want = oracle.pair_count(a, None, edges, True)
    got = gpu_counts(acf, ctx, a, None, edges, True, kernel=kern)
    st = acf.acf_get_stats(ctx)
    assert got.tolist() == want.tolist() and int(want.sum()) > 20000
    assert st["pairs_chord"] > 10 * st["pairs_fp64"] > 0, st
    scale = 1.0 + rng.uniform(-2e-7, 2e-7, 7200)
    b = (a.reshape(3, -1) * scale).reshape(-1)
    want = oracle.pair_count(b, None, edges, True)
    got = gpu_counts(acf, ctx, b, None, edges, True, kernel=kern)
    assert got.tolist() == want.tolist()


@pytest.mark.parametrize("kernel", ["auto", "window"])
def test_maximum_number_of_bins(acf, ctx, oracle, kernel):
    """ACF_MAX_BINS bins, unweighted and weighted: the window kernel then keeps one set of histogram rows per
    CTA instead of one per warp; AUTO must find a kernel whose shared memory fits."""
    kern = {"auto": acf.ACF_KERNEL_AUTO, "window": acf.ACF_KERNEL_WINDOW}[kernel]
    ra, dec = full_sky(3000, 7)
    a = acf.acf_radec_to_xyz(ra, dec)
    wa = np.random.default_rng(8).uniform(0.5, 2.0, 3000).astype(np.float32)
    edges = cos_edges_from_theta_deg(linear_theta_edges_deg(0.0, 180.0, 1024))
    assert gpu_counts(acf, ctx, a, None, edges, True, kernel=kern).tolist() == oracle.pair_count(a, None, edges, True).tolist()
    got = gpu_counts(acf, ctx, a, None, edges, True, wa=wa, kernel=kern)
    want = oracle.pair_count(a, None, edges, True, w_a=wa)
    assert got[0].tolist() == want[0].tolist()
    np.testing.assert_allclose(got[1], want[1], rtol=WSUM_RTOL, atol=0)


@pytest.mark.parametrize("kernel", ["table", "window"])
def test_weights_wide_range_and_zero(acf, ctx, oracle, kernel):
    """Weights that cannot share an fp64 accumulator with the count (range far above 2^13, zeros among them):
    the window kernel must take its unpacked variant; narrow-range weights take the packed one.  Both
    against the oracle, counts exact and sums to 1e-12."""
    kern = {"table": acf.ACF_KERNEL_TABLE, "window": acf.ACF_KERNEL_WINDOW}[kernel]
    ra, dec = full_sky(5000, 61)
    rb, db = full_sky(4100, 62)
    a, b = acf.acf_radec_to_xyz(ra, dec), acf.acf_radec_to_xyz(rb, db)
    rng = np.random.default_rng(63)
    edges = cos_edges_from_theta_deg(log_theta_edges_deg(0.5, 180.0, 24))
    for lo, hi, zeros in ((-20.0, 10.0, True), (-1.0, 1.0, False), (-6.0, 7.0, False)):
        wa = np.exp(rng.uniform(lo, hi, 5000)).astype(np.float32)
        wb = np.exp(rng.uniform(lo, hi, 4100)).astype(np.float32)
        if zeros:
            wa[::7] = 0.0
            wb[::5] = 0.0
        for xb, w_b, auto in ((None, None, True), (b, wb, False)):
            got = gpu_counts(acf, ctx, a, xb, edges, auto, wa=wa, wb=w_b, kernel=kern)
            want = oracle.pair_count(a, xb, edges, auto, w_a=wa, w_b=w_b)
            assert got[0].tolist() == want[0].tolist()
            np.testing.assert_allclose(got[1], want[1], rtol=WSUM_RTOL, atol=0)
    acf.acf_set_option(ctx, acf.ACF_OPT_KERNEL, acf.ACF_KERNEL_AUTO)


def test_weighted_dyadic_exact(acf, ctx):
    # power-of-two weights: every product and partial sum is exact, so the sums must be exact too
    ra, dec = full_sky(3000, 51)
    a = acf.acf_radec_to_xyz(ra, dec)
    rng = np.random.default_rng(52)
    wa = (2.0 ** rng.integers(-3, 4, size=3000)).astype(np.float32)
    edges = cos_edges_from_theta_deg(np.array([0.0, 40.0, 90.0, 130.0, 180.0]))
    c, ws = gpu_counts(acf, ctx, a, None, edges, True, wa=wa)
    c1, w1 = gpu_counts(acf, ctx, a, None, edges, True, wa=np.ones(3000, np.float32))
    assert c.tolist() == c1.tolist() and w1.tolist() == c1.astype(np.float64).tolist()
    assert np.all(ws * 64 == np.round(ws * 64))


def test_invalid_arguments(acf, ctx):
    import torch
    ra, dec = full_sky(100, 1)
    a = acf.acf_radec_to_xyz(ra, dec)
    da = dev(a)
    ok = np.array([1.0, 0.0, -1.0])
    for bad in (np.array([0.0, 0.5]), np.array([1.5, 0.0]), np.array([0.5]), np.array([0.5, 0.5])):
        with pytest.raises(acf.AcfError) as ei:
            acf.acf_pair_count(ctx, da, None, bad, True)
        assert ei.value.code == -1
    with pytest.raises(acf.AcfError):
        acf.acf_pair_count_rows(ctx, da, None, 5, 101, None, None, ok, True)      # row range outside
    # non-unit and non-finite vectors are rejected by the device-side check
    for poison in (2.0, float("nan"), float("inf")):
        b = a.copy()
        b[17] = poison
        with pytest.raises(acf.AcfError) as ei:
            acf.acf_pair_count(ctx, dev(b), None, ok, True)
        assert ei.value.code == -1 and "unit" in str(ei.value)
    with pytest.raises(acf.AcfError):
        acf.acf_pair_count_rows(ctx, da, dev(-np.ones(100, np.float32)), 0, 100, None, None, ok, True)
    # the context still works afterwards
    out = acf.acf_pair_count(ctx, da, None, ok, True)
    torch.cuda.synchronize()
    assert int(out.sum()) == 100 * 99 // 2


def test_bulk_windows_option(acf, ctx, oracle):
    """ACF_OPT_BULK: groups of points whose bounding caps put all their pairs into one bin are counted as
    a whole.  Same integers as the oracle, weighted sums to 1e-12, and the statistics say how many pairs
    were never evaluated."""
    w = make_config("full_sky", 0.02)
    xd, xr = acf.acf_radec_to_xyz(w.ra_d, w.dec_d), acf.acf_radec_to_xyz(w.ra_r, w.dec_r)
    acf.acf_set_option(ctx, acf.ACF_OPT_BULK, 1)
    try:
        for a, b, auto, wa, wb in ((xd, None, True, w.w_d, None), (xd, xr, False, w.w_d, w.w_r)):
            want = oracle.pair_count(a, b, w.cos_edges, auto, w_a=wa, w_b=wb)
            got = gpu_counts(acf, ctx, a, b, w.cos_edges, auto, wa=wa, wb=wb, kernel=acf.ACF_KERNEL_WINDOW)
            st = acf.acf_get_stats(ctx)
            assert got[0].tolist() == want[0].tolist()
            np.testing.assert_allclose(got[1], want[1], rtol=WSUM_RTOL, atol=0)
            assert st["pairs_bulk"] > 0 and st["pairs_bulk"] + st["pairs_evaluated"] == st["pairs_nominal"]
            want_u = oracle.pair_count(a, b, w.cos_edges, auto)
            assert gpu_counts(acf, ctx, a, b, w.cos_edges, auto, kernel=acf.ACF_KERNEL_WINDOW).tolist() == want_u.tolist()
    finally:
        acf.acf_set_option(ctx, acf.ACF_OPT_BULK, 0)
    gpu_counts(acf, ctx, xd, xr, w.cos_edges, False, wa=w.w_d, wb=w.w_r, kernel=acf.ACF_KERNEL_WINDOW)
    assert acf.acf_get_stats(ctx)["pairs_bulk"] == 0


@pytest.mark.parametrize("est", [0, 3])
def test_jackknife_against_recount(acf, ctx, oracle, est):
    """acf_jackknife (counts without region k as total minus the pairs touching k, all on the device)
    against the oracle's definition (remove the region, count afresh): same integers, so the same
    estimates; regions of unequal size, one of them empty in the randoms."""
    import torch
    w = make_config("clustered_patch", 0.012)
    n_reg = 6
    reg_d = np.minimum((w.ra_d / 20.0 * n_reg).astype(int), n_reg - 1)
    reg_r = np.minimum((w.ra_r / 20.0 * n_reg).astype(int), n_reg - 1)
    reg_r[reg_r == 4] = 5                                   # region 4 has no randoms
    od, orr = np.argsort(reg_d, kind="stable"), np.argsort(reg_r, kind="stable")
    ra_d, dec_d, reg_d = w.ra_d[od], w.dec_d[od], reg_d[od]
    ra_r, dec_r, reg_r = w.ra_r[orr], w.dec_r[orr], reg_r[orr]
    off_d = np.searchsorted(reg_d, np.arange(n_reg + 1))
    off_r = np.searchsorted(reg_r, np.arange(n_reg + 1))
    xd, xr = acf.acf_radec_to_xyz(ra_d, dec_d), acf.acf_radec_to_xyz(ra_r, dec_r)
    got = acf.acf_jackknife(ctx, torch.from_numpy(xd).cuda(), off_d, torch.from_numpy(xr).cuda(), off_r, w.cos_edges, est)
    w_full, w_jk, cov = oracle.jackknife(xd, reg_d, xr, reg_r, n_reg, w.cos_edges, est)
    np.testing.assert_allclose(got["w"], w_full, rtol=0, atol=WTHETA_ATOL, equal_nan=True)
    np.testing.assert_allclose(got["w_jk"], w_jk, rtol=0, atol=WTHETA_ATOL, equal_nan=True)
    ok = ~np.isnan(cov)
    assert np.array_equal(np.isnan(got["cov"]), np.isnan(cov))
    np.testing.assert_allclose(got["cov"][ok], cov[ok], rtol=1e-9, atol=1e-12)
    assert np.isfinite(w_jk).any()


def test_correlate_host_end_to_end(acf, ctx, oracle):
    w = make_config("full_sky", 0.004)
    res = acf.acf_correlate_host(ctx, w.ra_d, w.dec_d, w.w_d, w.ra_r, w.dec_r, w.w_r, w.cos_edges)
    xd, xr = oracle.radec_to_xyz(w.ra_d, w.dec_d), oracle.radec_to_xyz(w.ra_r, w.dec_r)
    dd, wdd = oracle.pair_count(xd, None, w.cos_edges, True, w_a=w.w_d)
    dr, wdr = oracle.pair_count(xd, xr, w.cos_edges, False, w_a=w.w_d, w_b=w.w_r)
    rr, wrr = oracle.pair_count(xr, None, w.cos_edges, True, w_a=w.w_r)
    assert res["dd"].tolist() == dd.tolist() and res["dr"].tolist() == dr.tolist() and res["rr"].tolist() == rr.tolist()
    np.testing.assert_allclose(res["wdd"], wdd, rtol=WSUM_RTOL)
    np.testing.assert_allclose(res["wdr"], wdr, rtol=WSUM_RTOL)
    np.testing.assert_allclose(res["wrr"], wrr, rtol=WSUM_RTOL)
    np.testing.assert_allclose(res["w"], oracle.wtheta_weighted(wdd, wdr, wrr, w.w_d, w.w_r), rtol=0, atol=WTHETA_ATOL,
                               equal_nan=True)
    t = make_config("tiny", 0.3)
    res = acf.acf_correlate_host(ctx, t.ra_d, t.dec_d, None, t.ra_r, t.dec_r, None, t.cos_edges)
    xd, xr = oracle.radec_to_xyz(t.ra_d, t.dec_d), oracle.radec_to_xyz(t.ra_r, t.dec_r)
    dd, dr, rr = (oracle.pair_count(xd, None, t.cos_edges, True), oracle.pair_count(xd, xr, t.cos_edges, False),
                  oracle.pair_count(xr, None, t.cos_edges, True))
    assert res["dd"].tolist() == dd.tolist() and res["dr"].tolist() == dr.tolist() and res["rr"].tolist() == rr.tolist()
    np.testing.assert_allclose(res["w"], oracle.wtheta(dd, dr, rr, t.n_d, t.n_r), rtol=0, atol=WTHETA_ATOL, equal_nan=True)


def test_prepared_catalogues(acf, ctx, oracle):
    """acf_prepare / acf_pair_count_prepared: the catalogues of an estimate prepared once, DD, DR, RR counted on
    the handles (weighted and not), the interleaved parts of a count adding up to the whole, a row range prepared
    as a catalogue of its own, bad input refused when it is prepared."""
    import torch
    w = make_config("full_sky", 0.006)
    xd, xr = acf.acf_radec_to_xyz(w.ra_d, w.dec_d), acf.acf_radec_to_xyz(w.ra_r, w.dec_r)
    dxd, dxr, dwd, dwr = dev(xd), dev(xr), dev(w.w_d), dev(w.w_r)
    cd, cr = acf.acf_prepare(ctx, dxd, dwd), acf.acf_prepare(ctx, dxr, dwr)
    try:
        for a, b, xa, xb, wa, wb, auto in ((cd, None, xd, None, w.w_d, None, True), (cd, cr, xd, xr, w.w_d, w.w_r, False),
                                           (cr, None, xr, None, w.w_r, None, True)):
            want = oracle.pair_count(xa, xb, w.cos_edges, auto, w_a=wa, w_b=wb)
            c, s = acf.acf_pair_count_prepared(ctx, a, b, w.cos_edges)
            torch.cuda.synchronize()
            assert acf.counts_to_numpy(c).tolist() == want[0].tolist()
            np.testing.assert_allclose(s.cpu().numpy(), want[1], rtol=WSUM_RTOL, atol=0)
            st = acf.acf_get_stats(ctx)
            assert st["pairs_evaluated"] == st["pairs_nominal"] == (a.n * (a.n - 1) // 2 if auto else a.n * b.n)
            # the same handles, unweighted
            cu = acf.acf_pair_count_prepared(ctx, a, b, w.cos_edges, weighted=False)
            torch.cuda.synchronize()
            assert acf.counts_to_numpy(cu).tolist() == want[0].tolist()
            # parts: the slices of the pair matrix add up, more parts than tiles included
            for n_parts in (3, 40):
                tot_c, tot_s = np.zeros_like(want[0]), np.zeros_like(want[1])
                for part in range(n_parts):
                    c, s = acf.acf_pair_count_prepared(ctx, a, b, w.cos_edges, part=part, n_parts=n_parts)
                    torch.cuda.synchronize()
                    tot_c += acf.counts_to_numpy(c)
                    tot_s += s.cpu().numpy()
                assert tot_c.tolist() == want[0].tolist()
                np.testing.assert_allclose(tot_s, want[1], rtol=WSUM_RTOL, atol=0)
        # rows of the data as a catalogue of their own against the randoms
        rows = (1000, 3500)
        ck = acf.acf_prepare_rows(ctx, dxd, None, *rows)
        c = acf.acf_pair_count_prepared(ctx, ck, cr, w.cos_edges, weighted=False)
        torch.cuda.synchronize()
        assert acf.counts_to_numpy(c).tolist() == oracle.pair_count(xd, xr, w.cos_edges, False, rows=rows).tolist()
        # the handle prepared again on other data (another, smaller catalogue): its memory reused, the counts the new data's
        w2 = make_config("full_sky", 0.004, seed_offset=7)
        x2 = acf.acf_radec_to_xyz(w2.ra_d, w2.dec_d)
        acf.acf_prepare_again(ctx, ck, dev(x2), dev(w2.w_d))
        c, s = acf.acf_pair_count_prepared(ctx, ck, None, w.cos_edges)
        torch.cuda.synchronize()
        want2 = oracle.pair_count(x2, None, w.cos_edges, True, w_a=w2.w_d)
        assert acf.counts_to_numpy(c).tolist() == want2[0].tolist()
        np.testing.assert_allclose(s.cpu().numpy(), want2[1], rtol=WSUM_RTOL, atol=0)
        acf.acf_release(ctx, ck)
        with pytest.raises(acf.AcfError):
            acf.acf_pair_count_prepared(ctx, cd, cr, w.cos_edges, part=3, n_parts=3)
    finally:
        acf.acf_release(ctx, cd)
        acf.acf_release(ctx, cr)
    bad = xd.copy()
    bad[5] = 3.0
    with pytest.raises(acf.AcfError) as ei:
        acf.acf_prepare(ctx, dev(bad))
    assert ei.value.code == -1 and "unit" in str(ei.value)
    # the context still works afterwards
    assert int(acf.counts_to_numpy(acf.acf_pair_count(ctx, dxd, None, np.array([1.0, -1.0]), True)).sum()) == w.n_d * (w.n_d - 1) // 2


@pytest.mark.parametrize("est", [0, 1])
def test_random_ensemble_against_separate_counts(acf, ctx, oracle, est):
    """acf_random_ensemble (random catalogues of unequal sizes streamed through two handles, every count enqueued
    without a host wait) against the oracle's one count per catalogue: the same integers, so the same estimates,
    mean and covariance; a bad catalogue in the ensemble is refused."""
    w = make_config("clustered_patch", 0.02)
    xd = acf.acf_radec_to_xyz(w.ra_d, w.dec_d)
    rands = []
    for k in range(5):
        r = make_config("clustered_patch", 0.02 + 0.003 * k, seed_offset=50 + k)
        rands.append(acf.acf_radec_to_xyz(r.ra_r, r.dec_r))
    dxd = dev(xd)
    cat = acf.acf_prepare(ctx, dxd)
    try:
        got = acf.acf_random_ensemble(ctx, cat, [dev(x) for x in rands], w.cos_edges, est)
        dd, dr, rr, wk, mean, cov = oracle.random_ensemble(xd, rands, w.cos_edges, est)
        assert got["dd"].tolist() == dd.tolist() and got["dr"].tolist() == dr.tolist() and got["rr"].tolist() == rr.tolist()
        np.testing.assert_allclose(got["w"], wk, rtol=0, atol=WTHETA_ATOL, equal_nan=True)
        np.testing.assert_allclose(got["mean"], mean, rtol=0, atol=WTHETA_ATOL, equal_nan=True)
        ok = np.isfinite(cov)
        assert np.array_equal(np.isfinite(got["cov"]), ok)
        np.testing.assert_allclose(got["cov"][ok], cov[ok], rtol=1e-9, atol=1e-12)
        bad = rands[2].copy()
        bad[7] = float("nan")
        with pytest.raises(acf.AcfError) as ei:
            acf.acf_random_ensemble(ctx, cat, [dev(rands[0]), dev(rands[1]), dev(bad)], w.cos_edges, est)
        assert ei.value.code == -1 and "catalogue 2" in str(ei.value)
    finally:
        acf.acf_release(ctx, cat)
