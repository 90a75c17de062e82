"""Seeded random cases through every fast kernel against the oracle (-m gpu): catalogue sizes around the
tile and group boundaries, few to 1024 bins of both presets over random ranges, auto and cross counts,
unweighted and weighted (narrow and wide weight ranges, zeros), clustered and uniform points, row ranges.
Each case is small; the point is the variety of paths (masked groups, many-edge windows, shared rows,
packed and unpacked accumulators, pruning, the chord tier)."""
import os

import numpy as np
import pytest

from workloads import cos_edges_from_theta_deg, full_sky, linear_theta_edges_deg, log_theta_edges_deg

pytestmark = pytest.mark.gpu

WSUM_RTOL = 1e-12


@pytest.fixture(scope="module")
def acf():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1208_3658_b200 as P
    P.load_library()
    return P


@pytest.fixture(scope="module")
def oracle():
    from oracle import oracle as O
    O.build()
    return O


def make_points(rng, n, clustered):
    ra, dec = full_sky(n, int(rng.integers(1, 1 << 30)))
    if clustered:  # pull the points into a few clumps so that small separations are populated
        k = max(1, n // 40)
        ra = (ra[rng.integers(0, k, n)] + rng.normal(0, 0.05, n)) % 360.0
        dec = np.clip(dec[rng.integers(0, k, n)] + rng.normal(0, 0.05, n), -89.0, 89.0)
    return ra, dec


def random_case(rng):
    big = [9000, 20000] if os.environ.get("ACF_FUZZ_BIG") else []
    n_a = int(rng.choice([1, 2, 31, 127, 128, 129, 700, 1023, 1024, 1025, 2500, 5000] + big))
    n_b = int(rng.choice([1, 33, 128, 640, 1024, 1100, 3000] + big))
    auto = bool(rng.integers(0, 2))
    nbins = int(rng.choice([1, 2, 7, 40, 254, 1024]))
    lo = float(rng.choice([0.0, 1e-4, 0.01, 0.5]))
    hi = float(rng.choice([0.2, 5.0, 60.0, 180.0]))
    if hi <= lo:
        hi = 180.0
    if rng.integers(0, 2) and lo > 0:
        theta = log_theta_edges_deg(lo, hi, nbins)
    else:
        theta = linear_theta_edges_deg(lo, hi, nbins)
    weights = int(rng.integers(0, 4))  # 0 none, 1 narrow, 2 wide, 3 with zeros
    return n_a, n_b, auto, cos_edges_from_theta_deg(theta), weights, bool(rng.integers(0, 2))


def draw_weights(rng, n, kind):
    if kind == 0:
        return None
    w = np.exp(rng.uniform(-1, 1, n) if kind == 1 else rng.uniform(-12, 12, n)).astype(np.float32)
    if kind == 3:
        w[rng.integers(0, 3, n) == 0] = 0.0
    return w


N_SEEDS = int(os.environ.get("ACF_FUZZ_SEEDS", "48"))  # more seeds for a longer hunt


@pytest.mark.parametrize("seed", range(N_SEEDS))
def test_random_cases_all_kernels(acf, oracle, seed):
    import torch
    rng = np.random.default_rng(1000 + seed)
    n_a, n_b, auto, edges, wk, clustered = random_case(rng)
    ra, dec = make_points(rng, n_a, clustered)
    a = acf.acf_radec_to_xyz(ra, dec)
    b = None
    if not auto:
        rb, db = make_points(rng, n_b, clustered)
        b = acf.acf_radec_to_xyz(rb, db)
    wa = draw_weights(rng, n_a, wk)
    wb = None if (auto or wa is None) else draw_weights(rng, n_b, wk)
    rows = None
    if rng.integers(0, 3) == 0 and n_a > 2:
        i0 = int(rng.integers(0, n_a - 1))
        rows = (i0, int(rng.integers(i0 + 1, n_a + 1)))
    want = oracle.pair_count(a, b, edges, auto, w_a=wa, w_b=wb, rows=rows)
    ctx = acf.acf_create(0)
    try:
        for kern in (acf.ACF_KERNEL_WINDOW, acf.ACF_KERNEL_TABLE, acf.ACF_KERNEL_AUTO):
            for bulk in (0, 1):
                acf.acf_set_option(ctx, acf.ACF_OPT_KERNEL, kern)
                acf.acf_set_option(ctx, acf.ACF_OPT_BULK, bulk)
                da = torch.from_numpy(a).cuda()
                db_ = None if auto else torch.from_numpy(b).cuda()
                dwa = None if wa is None else torch.from_numpy(wa).cuda()
                dwb = None if wb is None else torch.from_numpy(wb).cuda()
                i0, i1 = rows if rows is not None else (0, n_a)
                try:
                    out = acf.acf_pair_count_rows(ctx, da, dwa, i0, i1, db_, dwb, edges, auto)
                except acf.AcfError as e:
                    # an explicit kernel choice may not fit its histograms into shared memory (include/acf.h)
                    assert kern != acf.ACF_KERNEL_AUTO and edges.size > 600, str(e)
                    continue
                torch.cuda.synchronize()
                if wa is None:
                    assert acf.counts_to_numpy(out).tolist() == want.tolist(), (seed, kern, bulk)
                else:
                    assert acf.counts_to_numpy(out[0]).tolist() == want[0].tolist(), (seed, kern, bulk)
                    np.testing.assert_allclose(out[1].cpu().numpy(), want[1], rtol=WSUM_RTOL, atol=0, err_msg=str((seed, kern, bulk)))
    finally:
        acf.acf_destroy(ctx)


@pytest.mark.parametrize("kernel", ["window", "table"])
@pytest.mark.parametrize("bulk", [0, 1])
def test_inexact_norms_and_tight_groups(acf, oracle, kernel, bulk):
    """Vectors whose norms are off 1 by what the validation accepts (| |u|^2 - 1 | <= 1e-6), in tight groups: the
    pair cosine of the definition carries the norms, so a bounding cap built from the directions alone would put a
    whole window on the wrong side of an edge (round-1 advice).  First the constructed case -- 1024 copies of
    a (1 + 4e-7) against 1024 copies of b (1 + 4e-7), 1e-3 rad apart, an edge at cos(theta) (1 + 4e-7): every pair has
    c = (1 + 8e-7) cos(theta) > e_m and lies before the edge, although the directions alone say beyond it -- then
    antipodal points with norms above 1 and e_n = -1, then seeded clumps with random norms and edges at the clumps'
    separations.  Both fast kernels, with and without ACF_OPT_BULK."""
    import torch
    kern = {"window": acf.ACF_KERNEL_WINDOW, "table": acf.ACF_KERNEL_TABLE}[kernel]
    ctx = acf.acf_create(0)
    acf.acf_set_option(ctx, acf.ACF_OPT_KERNEL, kern)
    acf.acf_set_option(ctx, acf.ACF_OPT_BULK, bulk)

    def run(a, b, edges, auto=False):
        da = torch.from_numpy(a).cuda()
        db = None if auto else torch.from_numpy(b).cuda()
        out = acf.acf_pair_count_rows(ctx, da, None, 0, a.size // 3, db, None, edges, auto)
        torch.cuda.synchronize()
        return acf.counts_to_numpy(out).tolist()

    try:
        theta = 1.0e-3
        s = 1.0 + 4.0e-7
        a = np.tile(np.array([[1.0], [0.0], [0.0]]) * s, (1, 1024)).reshape(-1)
        b = np.tile(np.array([[np.cos(theta)], [np.sin(theta)], [0.0]]) * s, (1, 1024)).reshape(-1)
        edges = np.array([1.0, np.cos(theta) * s, np.cos(2 * theta), 0.0, -1.0])
        want = oracle.pair_count(a, b, edges, False).tolist()
        assert want[0] == 1024 * 1024   # the definition puts every pair before the edge
        assert run(a, b, edges) == want
        # antipodal points a little longer than 1, last edge at the pole: c clamps to -1 and belongs to the last bin
        a2 = np.concatenate([a.reshape(3, -1), -a.reshape(3, -1)], axis=1).reshape(-1)
        assert run(a2, None, edges, auto=True) == oracle.pair_count(a2, None, edges, True).tolist()
        rng = np.random.default_rng(99)
        for trial in range(6):
            n_cl = int(rng.integers(3, 40))
            centres = rng.normal(size=(n_cl, 3))
            centres /= np.linalg.norm(centres, axis=1, keepdims=True)
            sig = float(rng.choice([1e-6, 1e-4, 1e-3]))
            def clumps(n):
                p = centres[rng.integers(0, n_cl, n)] + sig * rng.normal(size=(n, 3))
                p /= np.linalg.norm(p, axis=1, keepdims=True)
                p *= (1.0 + rng.uniform(-4.5e-7, 4.5e-7, n))[:, None]
                return np.ascontiguousarray(p.T).reshape(-1)
            a, b = clumps(int(rng.choice([1024, 1500, 2600]))), clumps(int(rng.choice([1024, 2048, 3000])))
            # edges at the cosines of the separations of the clump centres, nudged by the size of the norm effect
            c = np.unique(np.clip(centres @ centres.T, -1, 1).round(12))
            c = c[(c > -0.999) & (c < 0.999999)]
            pick = rng.choice(c, size=min(12, c.size), replace=False) * (1.0 + rng.uniform(-8e-7, 8e-7, min(12, c.size)))
            edges = np.unique(np.concatenate([[1.0, -1.0], pick]))[::-1].copy()
            assert run(a, b, edges) == oracle.pair_count(a, b, edges, False).tolist(), (trial, "cross")
            assert run(a, None, edges, auto=True) == oracle.pair_count(a, None, edges, True).tolist(), (trial, "auto")
    finally:
        acf.acf_destroy(ctx)
