"""Pins for oracle/acf_oracle.c against things other than itself (-m "not gpu").

Each test names the part of the oracle it pins (O1..O8, see acf_oracle.c header) and
what fixes the expected value: hand-counted geometry (tests/golden), the paper's own
Appendix-A formula, pair-count identities of PAPER.md:70, closed forms, or brute
force in a different formulation.
"""
import math

import numpy as np
import pytest

from conftest import read_golden
from workloads import cos_edges_from_theta_deg, full_sky, log_theta_edges_deg, make_config, uniform_patch
from workloads.catalogs import lognormal_weights, neyman_scott

PHI = (1 + 5 ** 0.5) / 2


def _soa(v):
    """(n,3) array of vectors -> flat [x|y|z] SoA (the oracle's xyz layout)."""
    v = np.asarray(v, dtype=np.float64)
    return np.concatenate([v[:, 0], v[:, 1], v[:, 2]])


def _solids():
    octa = [(1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)]
    cube = [(a, b, c) for a in (-1, 1) for b in (-1, 1) for c in (-1, 1)]
    tetra = [(1, 1, 1), (1, -1, -1), (-1, 1, -1), (-1, -1, 1)]
    ico = []
    for s1 in (-1, 1):
        for s2 in (-1, 1):
            ico += [(0, s1, s2 * PHI), (s1, s2 * PHI, 0), (s2 * PHI, 0, s1)]

    def norm(p):
        p = np.asarray(p, dtype=np.float64)
        return p / np.linalg.norm(p, axis=1, keepdims=True)

    return {"octahedron": norm(octa), "cube": norm(cube), "tetrahedron": norm(tetra), "icosahedron": norm(ico)}


def _isolating_edges(cosines):
    """Descending cosine edges that put each expected cosine alone in a bin, every edge at
    least 0.05 away from every expected cosine; range closed at -1 so antipodal pairs
    (clamped c = -1, last bin closed) are kept."""
    cs = sorted(set(cosines), reverse=True)
    edges = [min(1.0, cs[0] + 0.1)]
    for a, b in zip(cs[:-1], cs[1:]):
        assert a - b > 0.1
        edges.append((a + b) / 2)
    edges.append(max(-1.0, cs[-1] - 0.1))
    return np.array(edges)


@pytest.mark.parametrize("solid", ["octahedron", "cube", "tetrahedron", "icosahedron", "ring12"])
def test_O2_O6_regular_point_sets(oracle, solid):
    rows = [r for r in read_golden("polyhedra_pairs.txt") if r[0] == solid]
    n = int(rows[0][1])
    cosines = [float(r[2]) for r in rows]
    expect = {float(r[2]): int(r[4]) for r in rows}
    assert sum(expect.values()) == n * (n - 1) // 2
    if solid == "ring12":
        xyz = oracle.radec_to_xyz(np.arange(12) * 30.0, np.zeros(12))  # through O1 as well
    else:
        pts = _solids()[solid]
        assert len(pts) == n
        xyz = _soa(pts)
    edges = _isolating_edges(cosines)
    counts = oracle.pair_count(xyz, None, edges, True)
    got = dict(zip(sorted(set(cosines), reverse=True), counts.tolist()))
    assert got == expect
    # same sets as a cross-count of the set with itself: every ordered pair twice, plus n
    # self pairs at c = 1 (dropped here unless the first edge reaches 1)
    cross = oracle.pair_count(xyz, xyz, edges, False)
    self_in = 1 if edges[0] >= 1.0 else 0
    exp_cross = np.array([2 * expect[c] for c in sorted(set(cosines), reverse=True)])
    exp_cross[0] += n * self_in
    assert cross.tolist() == exp_cross.tolist()


def test_O1_unit_vectors_golden(oracle):
    rows = read_golden("radec_unit_vectors.txt")
    ra = np.array([float(r[0]) for r in rows])
    dec = np.array([float(r[1]) for r in rows])
    want = np.array([[float(v) for v in r[2:5]] for r in rows])
    xyz = oracle.radec_to_xyz(ra, dec).reshape(3, -1).T
    assert np.max(np.abs(xyz - want)) < 3e-16
    assert np.max(np.abs(np.linalg.norm(xyz, axis=1) - 1)) < 3e-16


def test_O1_layout_is_soa(oracle):
    xyz = oracle.radec_to_xyz(np.array([0.0, 90.0, 0.0]), np.array([0.0, 0.0, 90.0]))
    assert xyz.shape == (9,)
    np.testing.assert_allclose(xyz[0:3], [1, 0, 0], atol=1e-16)  # x of the three points
    np.testing.assert_allclose(xyz[3:6], [0, 1, 0], atol=1e-16)  # y
    np.testing.assert_allclose(xyz[6:9], [0, 0, 1], atol=1e-16)  # z


def _pair_with_cos(c):
    """a = (1,0,0), b = (c, sqrt(1-c^2), 0): the O2 chain gives fma(1,c,fma(0,s,0*0)) = c exactly."""
    s = math.sqrt(max(0.0, 1.0 - c * c))
    return _soa([(1.0, 0.0, 0.0)]), _soa([(c, s, 0.0)])


def test_O3_O4_edge_inclusivity(oracle):
    edges = np.array([0.9, 0.5, 0.25, -0.5])  # 3 bins
    up = lambda v: np.nextafter(v, np.inf)
    dn = lambda v: np.nextafter(v, -np.inf)
    cases = [
        (0.9, 0), (up(0.9), None), (dn(0.9), 0),          # range is closed at e_0
        (0.5, 1), (up(0.5), 0), (dn(0.5), 1),             # e_{k+1} < c <= e_k
        (0.25, 2), (up(0.25), 1), (dn(0.25), 2),
        (-0.5, 2), (up(-0.5), 2), (dn(-0.5), None),       # last bin closed at e_n
        (0.0, 2), (0.7, 0), (1.0, None), (-1.0, None),
    ]
    for c, k in cases:
        a, b = _pair_with_cos(c)
        got = oracle.pair_count(a, b, edges, False)
        want = np.zeros(3, dtype=np.uint64)
        if k is not None:
            want[k] = 1
        assert got.tolist() == want.tolist(), (c, k)
        assert oracle.pair_count(b, a, edges, False).tolist() == want.tolist()


def test_O2_clamp_of_coincident_points(oracle):
    # a vector whose rounded square norm exceeds 1: c = 1 + 2^-52*k before the clamp
    v = np.array([0.6, 0.8, 1e-8])
    v = v / np.linalg.norm(v)
    v[0] = np.nextafter(np.nextafter(v[0], 2.0), 2.0)
    c_raw = math.fma(v[0], v[0], math.fma(v[1], v[1], v[2] * v[2])) if hasattr(math, "fma") else None
    xyz = _soa([v, v])
    full = np.array([1.0, 0.0, -1.0])
    assert oracle.pair_count(xyz, None, full, True).tolist() == [1, 0]      # kept: clamped to 1 <= e_0 = 1
    below = np.array([np.nextafter(1.0, 0.0), 0.0, -1.0])
    assert oracle.pair_count(xyz, None, below, True).tolist() == [0, 0]     # theta = 0 is below theta_min
    if c_raw is not None:
        assert c_raw > 1.0  # the case really exercises the clamp
    # antipodal with norm > 1: clamped to -1, kept in the closed last bin
    xyz2 = _soa([v, -v])
    assert oracle.pair_count(xyz2, None, full, True).tolist() == [0, 1]


def _random_xyz(oracle, n, seed):
    ra, dec = full_sky(n, seed)
    return oracle.radec_to_xyz(ra, dec), ra, dec


def test_O6_totals_when_bins_cover_everything(oracle):
    # n(n-1)/2 auto pairs, n n_r cross pairs
    a, _, _ = _random_xyz(oracle, 700, 5)
    b, _, _ = _random_xyz(oracle, 450, 6)
    edges = cos_edges_from_theta_deg(np.array([0.0, 1.0, 10.0, 60.0, 90.0, 150.0, 180.0]))
    assert edges[0] == 1.0 and edges[-1] == -1.0
    assert int(oracle.pair_count(a, None, edges, True).sum()) == 700 * 699 // 2
    assert int(oracle.pair_count(a, b, edges, False).sum()) == 700 * 450


def test_symmetries_and_additivity(oracle):
    a, _, _ = _random_xyz(oracle, 600, 7)
    b, _, _ = _random_xyz(oracle, 500, 8)
    edges = cos_edges_from_theta_deg(log_theta_edges_deg(0.5, 180.0, 17))
    ab = oracle.pair_count(a, b, edges, False)
    ba = oracle.pair_count(b, a, edges, False)
    assert ab.tolist() == ba.tolist()                                  # swap symmetry
    auto = oracle.pair_count(a, None, edges, True)
    aa = oracle.pair_count(a, a, edges, False)
    assert aa.tolist() == (2 * auto).tolist()                          # self pairs (theta=0) below theta_min
    full = cos_edges_from_theta_deg(np.array([0.0, 30.0, 180.0]))
    assert oracle.pair_count(a, a, full, False).tolist() == (2 * oracle.pair_count(a, None, full, True)
                                                             + np.array([600, 0], dtype=np.uint64)).tolist()
    # additivity over row blocks: the paper's sub-matrix decomposition
    parts = sum(oracle.pair_count(a, b, edges, False, rows=r) for r in [(0, 100), (100, 101), (101, 600)])
    assert parts.tolist() == ab.tolist()
    parts = sum(oracle.pair_count(a, None, edges, True, rows=r) for r in [(0, 250), (250, 600)])
    assert parts.tolist() == auto.tolist()
    # merging adjacent bins = summing the fine bins
    coarse = edges[::2] if (len(edges) - 1) % 2 == 0 else np.concatenate([edges[:-1:2], edges[-1:]])
    cc = oracle.pair_count(a, b, coarse, False)
    fine = ab.astype(np.int64)
    merged = [int(fine[i:i + 2].sum()) for i in range(0, len(fine), 2)]
    assert cc.tolist() == merged


def test_O8_appendix_A_formula_agrees(oracle):
    # theta from the paper's own trigonometric expression (atan2 form), binned in theta
    ra, dec = uniform_patch(400, (10.0, 50.0), (-20.0, 35.0), 9)
    ra2, dec2 = full_sky(300, 10)
    theta_edges = log_theta_edges_deg(0.05, 170.0, 23)
    cos_edges = cos_edges_from_theta_deg(theta_edges)
    for (r1, d1, r2, d2, auto) in [(ra, dec, None, None, True), (ra, dec, ra2, dec2, False)]:
        x1 = oracle.radec_to_xyz(r1, d1)
        x2 = None if auto else oracle.radec_to_xyz(r2, d2)
        c_cos = oracle.pair_count(x1, x2, cos_edges, auto)
        c_th, n_near, near = oracle.pair_count_theta(r1, d1, r2, d2, theta_edges, auto, rel_tol=1e-9)
        assert n_near == 0, near            # no pair sits within 1e-9 of an edge in this seed
        assert c_cos.tolist() == c_th.tolist()
        assert int(c_cos.sum()) > 0


def test_brute_force_numpy_acos_formulation(oracle):
    # an independent formulation: theta = arccos(u.v) with numpy, binned with searchsorted
    a, _, _ = _random_xyz(oracle, 300, 11)
    b, _, _ = _random_xyz(oracle, 200, 12)
    theta_edges = np.array([2.0, 5.0, 20.0, 45.0, 90.0, 120.0, 175.0])
    cos_edges = cos_edges_from_theta_deg(theta_edges)
    A = a.reshape(3, -1).T
    B = b.reshape(3, -1).T
    th = np.degrees(np.arccos(np.clip(A @ B.T, -1, 1))).ravel()
    assert np.min(np.abs(th[:, None] - theta_edges[None, :])) > 1e-7   # nothing near an edge
    k = np.searchsorted(theta_edges, th, side="right") - 1
    want = np.bincount(k[(k >= 0) & (k < 6)], minlength=6)
    got = oracle.pair_count(a, b, cos_edges, False)
    assert got.tolist() == want.tolist()


def test_uniform_sphere_closed_form(oracle):
    # c = u.v is uniform on [-1, 1] for independent uniform points: E[count_k] = N (e_k - e_{k+1}) / 2
    n = 6000
    a, _, _ = _random_xyz(oracle, n, 13)
    edges = cos_edges_from_theta_deg(log_theta_edges_deg(1.0, 180.0, 12))
    counts = oracle.pair_count(a, None, edges, True).astype(np.float64)
    npairs = n * (n - 1) / 2
    expect = npairs * (edges[:-1] - edges[1:]) / 2
    z = (counts - expect) / np.sqrt(expect)
    assert np.all(np.abs(z) < 5), z
    assert abs(counts.sum() - npairs * (edges[0] - edges[-1]) / 2) < 5 * math.sqrt(npairs)


def test_O7_estimator_golden(oracle):
    for r in read_golden("wtheta_examples.txt"):
        n_d, n_r, dd, dr, rr = (int(v) for v in r[:5])
        w = oracle.wtheta([dd], [dr], [rr], n_d, n_r)[0]
        if r[5] == "nan":
            assert math.isnan(w)
        else:
            assert abs(w - float(r[5])) < 1e-15


def _num(v):
    return float("nan") if v == "nan" else float(v)


def test_other_estimators_golden(oracle):
    # PAPER.md:65 "other estimators": hand-computed values, and kind 0 is Eq. 2 itself
    for r in read_golden("estimator_examples.txt"):
        n_d, n_r, dd, dr, rr = (int(v) for v in r[:5])
        for kind in range(4):
            w = oracle.estimator(kind, [dd], [dr], [rr], n_d, n_r)[0]
            want = _num(r[5 + kind])
            assert (math.isnan(w) and math.isnan(want)) or abs(w - want) < 1e-15, (r, kind, w)
        ls = oracle.wtheta([dd], [dr], [rr], n_d, n_r)[0]
        assert (math.isnan(ls) and r[5] == "nan") or ls == oracle.estimator(0, [dd], [dr], [rr], n_d, n_r)[0]


def test_other_estimators_identities(oracle):
    # (1 + natural) = (1 + DP) * dr/rr and (1 + Hamilton) = (1 + natural) / (1 + DP)^2 * ... : all four are
    # functions of the two ratios a = dd/rr, b = dr/rr:  LS = a - 2b + 1, nat = a - 1, DP = a/b - 1, Ham = a/b^2 - 1
    rng = np.random.default_rng(5)
    n_d, n_r = 1000, 1700
    dd = rng.integers(1, 10 ** 5, 30).astype(np.uint64)
    dr = rng.integers(1, 10 ** 5, 30).astype(np.uint64)
    rr = rng.integers(1, 10 ** 5, 30).astype(np.uint64)
    f = lambda c, n: c.astype(np.float64) / n
    a = f(dd, n_d * (n_d - 1) / 2) / f(rr, n_r * (n_r - 1) / 2)
    b = f(dr, n_d * n_r) / f(rr, n_r * (n_r - 1) / 2)
    est = [oracle.estimator(k, dd, dr, rr, n_d, n_r) for k in range(4)]
    np.testing.assert_allclose(est[0], a - 2 * b + 1, rtol=0, atol=1e-11)
    np.testing.assert_allclose(est[1], a - 1, rtol=1e-13)
    np.testing.assert_allclose(est[2], a / b - 1, rtol=0, atol=1e-11)
    np.testing.assert_allclose(est[3], a / b ** 2 - 1, rtol=0, atol=1e-10)


def test_bin_presets_golden(oracle):
    modes = {"even": 0, "log": 1, "log10": 2}
    for r in read_golden("bin_presets.txt"):
        if r[0] == "cos":
            n = (len(r) - 1) // 2
            theta = [float(v) for v in r[1:1 + n]]
            want = np.array([float(v) for v in r[1 + n:]])
            e = oracle.cos_edges(theta)
            # the radian argument is rounded twice (the constant pi/180 and the product): up to ~2 ulp of pi
            np.testing.assert_allclose(e, want, rtol=0, atol=5e-16)
            assert e[0] == 1.0 and e[-1] == -1.0
            continue
        lo, hi, nb = float(r[1]), float(r[2]), int(r[3])
        want = np.array([float(v) for v in r[4:]])
        theta = oracle.theta_edges(modes[r[0]], lo, hi, nb)
        np.testing.assert_allclose(theta, want, rtol=4e-16, atol=0)
        assert theta[0] == lo and theta[-1] == hi
    # natural-log and log10 spacing are the same edges (reading R5); the workload generator agrees
    assert oracle.theta_edges(1, 0.5 / 60, 10.0, 25).tolist() == oracle.theta_edges(2, 0.5 / 60, 10.0, 25).tolist()
    from workloads import log_theta_edges_deg, cos_edges_from_theta_deg
    np.testing.assert_allclose(oracle.theta_edges(1, 1 / 60, 180.0, 40), log_theta_edges_deg(1 / 60, 180.0, 40), rtol=1e-14)
    np.testing.assert_allclose(oracle.cos_edges(log_theta_edges_deg(1 / 60, 180.0, 40)),
                               cos_edges_from_theta_deg(log_theta_edges_deg(1 / 60, 180.0, 40)), rtol=0, atol=2e-16)


def test_jackknife_pins(oracle):
    # covariance formula on a hand example: rows (1,2),(3,4),(5,6): mean (3,4), deviations (-2,-2),(0,0),(2,2),
    # sum of outer products 8 everywhere, times (N-1)/N = 2/3
    np.testing.assert_allclose(oracle.jackknife_cov([[1, 2], [3, 4], [5, 6]]), np.full((2, 2), 16.0 / 3.0), rtol=1e-15)
    # a constant estimate has no variance; one varying bin leaves the others' rows and columns zero
    assert np.all(oracle.jackknife_cov(np.ones((7, 3))) == 0)
    c = oracle.jackknife_cov([[0, 1], [2, 1], [4, 1], [6, 1]])
    assert c[0, 0] == pytest.approx(0.75 * 20.0) and c[1, 1] == 0 and c[0, 1] == 0
    # delete-one counts: a pair between two regions is missing from two of the resampled counts, a pair inside
    # a region from one: sum_k (DD - DD_(-k)) = 2 DD - sum_k DD(inside k)
    w = make_config("tiny", scale=0.06)
    xd = oracle.radec_to_xyz(w.ra_d, w.dec_d).reshape(3, -1)
    reg = np.minimum((w.ra_d / 10.0 * 5).astype(int), 4)
    dd = oracle.pair_count(xd.reshape(-1), None, w.cos_edges, True)
    gone = sum(dd - oracle.pair_count(np.ascontiguousarray(xd[:, reg != k]).reshape(-1), None, w.cos_edges, True) for k in range(5))
    inside = sum(oracle.pair_count(np.ascontiguousarray(xd[:, reg == k]).reshape(-1), None, w.cos_edges, True) for k in range(5))
    assert gone.tolist() == (2 * dd - inside).tolist()
    # the resampled estimates of an unclustered catalogue scatter around the full one
    xr = oracle.radec_to_xyz(w.ra_r, w.dec_r)
    regr = np.minimum((w.ra_r / 10.0 * 5).astype(int), 4)
    w_full, w_jk, cov = oracle.jackknife(xd.reshape(-1), reg, xr, regr, 5, w.cos_edges, 0)
    ok = ~np.isnan(w_full) & ~np.isnan(w_jk).any(axis=0)
    assert w_jk.shape == (5, w.nbins) and np.all(np.abs(w_jk[:, ok].mean(axis=0) - w_full[ok]) < 0.5 * np.abs(w_full[ok]) + 0.2)
    assert np.all(np.diag(cov)[ok] >= 0)


def test_random_ensemble_pins(oracle):
    """Monte-Carlo errors from an ensemble of random catalogues.  The covariance formula on a hand
    example; the ensemble is one count per catalogue (identical catalogues give identical estimates and a zero
    covariance); on unclustered data the estimates scatter around zero by about their Poisson error."""
    # rows (1,2),(3,4),(5,6): mean (3,4), deviations (-2,-2),(0,0),(2,2), sum of outer products 8, / (K - 1) = 4
    np.testing.assert_allclose(oracle.ensemble_cov([[1, 2], [3, 4], [5, 6]]), np.full((2, 2), 4.0), rtol=1e-15)
    c = oracle.ensemble_cov([[0, 1], [2, 1], [4, 1], [6, 1]])      # variance of 0, 2, 4, 6 is 20 / 3
    assert c[0, 0] == pytest.approx(20.0 / 3.0) and c[1, 1] == 0 and c[0, 1] == 0
    w = make_config("tiny", scale=0.08)
    xd = oracle.radec_to_xyz(w.ra_d, w.dec_d)
    rands = []
    for k in range(5):
        r = make_config("tiny", scale=0.08, seed_offset=100 + k)
        rands.append(oracle.radec_to_xyz(r.ra_r, r.dec_r))
    dd, dr, rr, wk, mean, cov = oracle.random_ensemble(xd, rands, w.cos_edges, 0)
    assert dd.tolist() == oracle.pair_count(xd, None, w.cos_edges, True).tolist()
    for k in range(5):
        assert dr[k].tolist() == oracle.pair_count(xd, rands[k], w.cos_edges, False).tolist()
        assert rr[k].tolist() == oracle.pair_count(rands[k], None, w.cos_edges, True).tolist()
        np.testing.assert_array_equal(wk[k], oracle.wtheta(dd, dr[k], rr[k], xd.size // 3, rands[k].size // 3))
    ok = np.isfinite(wk).all(axis=0) & (rr.min(axis=0) > 200)
    assert ok.sum() >= 3
    np.testing.assert_allclose(mean[ok], wk[:, ok].mean(axis=0), rtol=1e-15)
    sd = np.sqrt(np.diag(cov)[ok])
    assert np.all(sd < 5.0 * np.sqrt(2.0 / rr[:, ok].mean(axis=0)) + 0.02) and np.all(np.abs(mean[ok]) < 5 * sd + 0.05)
    same = oracle.random_ensemble(xd, [rands[0], rands[0], rands[0]], w.cos_edges, 0)
    assert np.all(np.abs(same[5][np.isfinite(same[5])]) < 1e-30) and same[3][0].tobytes() == same[3][2].tobytes()


def test_O7_unclustered_is_zero_within_noise(oracle):
    # north_star: w(theta) ~ 0 within Poisson noise for an unclustered uniform catalogue
    w = make_config("tiny", scale=0.4)
    xd = oracle.radec_to_xyz(w.ra_d, w.dec_d)
    xr = oracle.radec_to_xyz(w.ra_r, w.dec_r)
    dd = oracle.pair_count(xd, None, w.cos_edges, True)
    dr = oracle.pair_count(xd, xr, w.cos_edges, False)
    rr = oracle.pair_count(xr, None, w.cos_edges, True)
    wt = oracle.wtheta(dd, dr, rr, w.n_d, w.n_r)
    ok = rr > 0
    sigma = np.sqrt(2.0 / np.maximum(rr[ok].astype(np.float64), 1.0))
    assert np.all(np.abs(wt[ok]) < 5 * sigma + 0.01), (wt, sigma)
    big = rr > 100000
    assert np.all(np.abs(wt[big]) < 0.02)


def test_O7_neyman_scott_closed_form(oracle):
    # flat-sky Neyman-Scott: w(theta) = F / (lambda_p 4 pi sigma^2) exp(-theta^2 / (4 sigma^2)),
    # F = (m-1)/m for exactly m children per parent.  Statistical pin of the whole chain
    # generator -> O1-O6 -> O7 (a wrong normalisation, sign or bin order fails it).
    m, n_par, sigma_am = 20, 1500, 3.0
    ra_rng, dec_rng = (0.0, 10.0), (-5.0, 5.0)
    area = 10.0 * (180 / math.pi) * (math.sin(math.radians(5)) * 2)
    ra_d, dec_d = neyman_scott(m * n_par, n_par, sigma_am, ra_rng, dec_rng, seed=101)
    ra_r, dec_r = uniform_patch(m * n_par, ra_rng, dec_rng, seed=102)
    theta = np.array([1.0, 2.0, 3.0, 4.5, 6.0, 8.0]) / 60.0
    edges = cos_edges_from_theta_deg(theta)
    xd, xr = oracle.radec_to_xyz(ra_d, dec_d), oracle.radec_to_xyz(ra_r, dec_r)
    dd = oracle.pair_count_decwindow(xd, dec_d, None, None, edges, True)
    dr = oracle.pair_count_decwindow(xd, dec_d, xr, dec_r, edges, False)
    rr = oracle.pair_count_decwindow(xr, dec_r, None, None, edges, True)
    w = oracle.wtheta(dd, dr, rr, m * n_par, m * n_par)
    sig = sigma_am / 60.0
    amp = ((m - 1) / m) / ((n_par / area) * 4 * math.pi * sig ** 2)
    # bin-averaged model, area weighting ~ theta dtheta
    model = []
    for lo, hi in zip(theta[:-1], theta[1:]):
        t = np.linspace(lo, hi, 200)
        model.append(np.sum(amp * np.exp(-t ** 2 / (4 * sig ** 2)) * t) / np.sum(t))
    model = np.array(model)
    assert amp > 1.0
    # counts per bin are O(1e4-1e5): a few per cent statistical, plus edge clipping
    np.testing.assert_allclose(w, model, rtol=0.12, atol=0.05)


def test_decwindow_equals_plain(oracle):
    w = make_config("survey_scale", scale=0.004)
    xd = oracle.radec_to_xyz(w.ra_d, w.dec_d)
    xr = oracle.radec_to_xyz(w.ra_r, w.dec_r)
    for (a, da, b, db, auto) in [(xd, w.dec_d, None, None, True), (xd, w.dec_d, xr, w.dec_r, False),
                                 (xr, w.dec_r, None, None, True)]:
        plain = oracle.pair_count(a, b, w.cos_edges, auto)
        fast = oracle.pair_count_decwindow(a, da, b, db, w.cos_edges, auto)
        assert plain.tolist() == fast.tolist()
        assert int(plain.sum()) > 0
    # range reaching theta = 0 (e_0 = 1): self pairs must still be excluded in auto mode
    e0 = cos_edges_from_theta_deg(np.array([0.0, 0.5, 2.0]))
    assert oracle.pair_count(xd, None, e0, True).tolist() == \
        oracle.pair_count_decwindow(xd, w.dec_d, None, None, e0, True).tolist()


def _weighted_golden():
    for r in read_golden("wtheta_weighted_examples.txt"):
        n_d = int(r[0])
        w_d = np.array([float(v) for v in r[1:1 + n_d]], dtype=np.float32)
        n_r = int(r[1 + n_d])
        w_r = np.array([float(v) for v in r[2 + n_d:2 + n_d + n_r]], dtype=np.float32)
        wdd, wdr, wrr = (float(v) for v in r[2 + n_d + n_r:5 + n_d + n_r])
        yield w_d, w_r, wdd, wdr, wrr, _num(r[5 + n_d + n_r])


def test_O7_weighted_estimator_golden_non_unit_weights(oracle):
    # hand-computed values with weights for which sum w^2 != sum w != n (tests/golden/wtheta_weighted_examples.txt)
    n = 0
    for w_d, w_r, wdd, wdr, wrr, want in _weighted_golden():
        assert not np.all(w_d == 1) and not np.all(w_r == 1)
        got = oracle.wtheta_weighted([wdd], [wdr], [wrr], w_d, w_r)[0]
        assert (math.isnan(got) and math.isnan(want)) or abs(got - want) < 1e-15, (w_d, w_r, got, want)
        n += 1
    assert n >= 6
    # the normalisers are the weighted pair totals: the weighted sums of ALL pairs of a catalogue, counted by
    # O2-O6 over the whole range, divided by them give fdd = fdr = frr = 1 and w = 0 (ties O7 to O5)
    a, _, _ = _random_xyz(oracle, 300, 41)
    b, _, _ = _random_xyz(oracle, 200, 42)
    wa, wb = lognormal_weights(300, 43), lognormal_weights(200, 44)
    everything = np.array([1.0, -1.0])
    _, sdd = oracle.pair_count(a, None, everything, True, w_a=wa)
    _, sdr = oracle.pair_count(a, b, everything, False, w_a=wa, w_b=wb)
    _, srr = oracle.pair_count(b, None, everything, True, w_a=wb)
    assert abs(oracle.wtheta_weighted(sdd, sdr, srr, wa, wb)[0]) < 1e-12


def test_cellwindow_equals_plain(oracle):
    # the Dec + RA window variant visits a superset of the counted pairs: same u64 histograms as the plain loop
    # on the small-angle configurations ...
    for name, scale in (("survey_scale", 0.004), ("pruning_stress", 0.002), ("clustered_patch", 0.01)):
        w = make_config(name, scale)
        xd, xr = oracle.radec_to_xyz(w.ra_d, w.dec_d), oracle.radec_to_xyz(w.ra_r, w.dec_r)
        for (a, ra, da, b, rb, db, auto) in [(xd, w.ra_d, w.dec_d, None, None, None, True),
                                             (xd, w.ra_d, w.dec_d, xr, w.ra_r, w.dec_r, False),
                                             (xr, w.ra_r, w.dec_r, None, None, None, True)]:
            plain = oracle.pair_count(a, b, w.cos_edges, auto)
            assert oracle.pair_count_cellwindow(a, ra, da, b, rb, db, w.cos_edges, auto).tolist() == plain.tolist()
            assert int(plain.sum()) > 0
    # ... and where the windows are stressed: the whole sphere with points at and near both poles (no RA bound
    # there), RA given outside [0, 360), pairs across RA = 0, theta_max from half a degree to 180 degrees
    # (bands wider than the sphere), row ranges
    rng = np.random.default_rng(91)
    ra, dec = full_sky(2500, 92)
    ra = np.concatenate([ra, rng.uniform(0, 360, 300), rng.uniform(-3, 3, 300), [0.0, 123.0, 359.999999, 10.0]])
    dec = np.concatenate([dec, np.where(rng.integers(0, 2, 300) == 0, -1, 1) * (90.0 - np.abs(rng.normal(0, 1.5, 300))),
                          rng.uniform(-4, 4, 300), [90.0, -90.0, 89.9999, -89.9999]])
    dec = np.clip(dec, -90.0, 90.0)
    ra[100:200] += 360.0     # the same directions, RA outside [0, 360)
    ra[200:300] -= 720.0
    rb, db = full_sky(1500, 93)
    a, b = oracle.radec_to_xyz(ra, dec), oracle.radec_to_xyz(rb, db)
    n_pairs_seen = 0
    for theta_max, nb in ((0.5, 5), (5.0, 9), (60.0, 6), (179.0, 4), (180.0, 3)):
        edges = cos_edges_from_theta_deg(log_theta_edges_deg(0.01, theta_max, nb))
        for (bb, rbb, dbb, auto) in ((None, None, None, True), (b, rb, db, False)):
            plain = oracle.pair_count(a, bb, edges, auto)
            assert oracle.pair_count_cellwindow(a, ra, dec, bb, rbb, dbb, edges, auto).tolist() == plain.tolist(), (theta_max, auto)
            n_pairs_seen += int(plain.sum())
        rows = (700, 1900)
        assert oracle.pair_count_cellwindow(a, ra, dec, None, None, None, edges, True, rows=rows).tolist() == \
            oracle.pair_count(a, None, edges, True, rows=rows).tolist()
    assert n_pairs_seen > 10 ** 6
    # near the poles a pair a fraction of a degree apart can be 180 degrees apart in RA: counted all the same
    pr = np.array([0.0, 180.0, 90.0, 270.0])
    pd = np.array([89.9, 89.9, -89.95, -89.95])
    px = oracle.radec_to_xyz(pr, pd)
    e = cos_edges_from_theta_deg(np.array([0.05, 0.15, 0.25]))
    assert oracle.pair_count_cellwindow(px, pr, pd, None, None, None, e, True).tolist() == [1, 1] == \
        oracle.pair_count(px, None, e, True).tolist()


def test_weighted_dyadic_exact(oracle):
    # weights that are small powers of two: every product and every partial sum is exact in fp64,
    # so the expected value can be computed in integer arithmetic
    n = 400
    a, _, _ = _random_xyz(oracle, n, 21)
    b, _, _ = _random_xyz(oracle, 300, 22)
    rng = np.random.default_rng(23)
    ea, eb = rng.integers(-3, 4, size=n), rng.integers(-3, 4, size=300)
    wa, wb = (2.0 ** ea).astype(np.float32), (2.0 ** eb).astype(np.float32)
    edges = cos_edges_from_theta_deg(np.array([0.0, 40.0, 90.0, 130.0, 180.0]))
    counts, ws = oracle.pair_count(a, b, edges, False, w_a=wa, w_b=wb)
    A, B = a.reshape(3, -1).T, b.reshape(3, -1).T
    c = A @ B.T
    assert np.min(np.abs(c[:, :, None] - edges[None, None, 1:-1])) > 1e-9
    k = np.searchsorted(-edges, -c, side="left") - 1
    k = np.clip(k, 0, 3)
    prod64 = (2 ** (ea[:, None] + eb[None, :] + 6)).astype(np.int64)  # scaled by 2^6 -> integers
    for bin_ in range(4):
        sel = k == bin_
        assert int(counts[bin_]) == int(sel.sum())
        assert ws[bin_] == prod64[sel].sum() / 64.0
    # unit weights reproduce the counts
    c1, w1 = oracle.pair_count(a, None, edges, True, w_a=np.ones(n, np.float32))
    assert w1.tolist() == c1.astype(np.float64).tolist()
    assert c1.tolist() == oracle.pair_count(a, None, edges, True).tolist()


def test_weighted_sphere_expectation(oracle):
    # E[w_i w_j] = E[w]^2 = exp(sigma^2) for independent lognormal(0, sigma) weights
    n = 5000
    a, _, _ = _random_xyz(oracle, n, 31)
    wa = lognormal_weights(n, 33)
    edges = cos_edges_from_theta_deg(np.array([0.0, 60.0, 90.0, 120.0, 180.0]))
    counts, ws = oracle.pair_count(a, None, edges, True, w_a=wa)
    ratio = ws / counts
    assert np.all(np.abs(ratio / math.exp(0.09) - 1) < 0.02), ratio
    # weighted estimator with unit weights equals the unweighted one
    b, _, _ = _random_xyz(oracle, 4000, 32)
    one_a, one_b = np.ones(n, np.float32), np.ones(4000, np.float32)
    dd, wdd = oracle.pair_count(a, None, edges, True, w_a=one_a)
    dr, wdr = oracle.pair_count(a, b, edges, False, w_a=one_a, w_b=one_b)
    rr, wrr = oracle.pair_count(b, None, edges, True, w_a=one_b)
    np.testing.assert_allclose(oracle.wtheta_weighted(wdd, wdr, wrr, one_a, one_b),
                               oracle.wtheta(dd, dr, rr, n, 4000), rtol=0, atol=1e-14)


def test_invalid_arguments(oracle):
    a, _, _ = _random_xyz(oracle, 10, 1)
    with pytest.raises(ValueError):
        oracle.pair_count(a, None, np.array([0.5, 0.6]), True)         # ascending
    with pytest.raises(ValueError):
        oracle.pair_count(a, None, np.array([1.5, 0.6]), True)         # outside [-1,1]
    with pytest.raises(ValueError):
        oracle.pair_count(a, None, np.array([0.5]), True)              # no bins
    assert oracle.pair_count(np.zeros(0), None, np.array([1.0, -1.0]), True).tolist() == [0]
    assert oracle.pair_count(a[[0, 10, 20]], None, np.array([1.0, -1.0]), True).tolist() == [0]  # n = 1
