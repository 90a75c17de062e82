"""acf_pair_count_static: the entry point that allocates nothing (its scratch memory is a fixed __device__ array)
against the existing path (acf_pair_count on a context) and the CPU oracle, on calls in a row that share the array.
Counts are u64 integers: they must be equal.

This file is meant to be collected last (pytest -x stops at the first failure); it passes alone and after the others.
"""
import numpy as np
import pytest

from workloads import cos_edges_from_theta_deg, linear_theta_edges_deg, log_theta_edges_deg
from workloads.catalogs import neyman_scott, uniform_patch

pytestmark = pytest.mark.gpu


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


def dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def test_static_entry_point_matches_the_existing_path_on_calls_in_a_row(acf, ctx, oracle):
    import torch
    ra, dec = neyman_scott(9000, 300, 3.0, (0.0, 8.0), (-4.0, 4.0), 71, children="poisson")
    rb, db = uniform_patch(7001, (0.0, 8.0), (-4.0, 4.0), 72)
    a, b = acf.acf_radec_to_xyz(ra, dec), acf.acf_radec_to_xyz(rb, db)
    da, db_ = dev(a), dev(b)
    # the caller's outputs, allocated once: the entry point itself allocates nothing
    out = torch.full((300,), -1, dtype=torch.int64, device="cuda")
    bad = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    # many bins and CTAs first, then fewer of both (whatever the first call left in the array must not show),
    # then the first case again
    cases = [
        (cos_edges_from_theta_deg(log_theta_edges_deg(1.0 / 60.0, 10.0, 300)), False),
        (cos_edges_from_theta_deg(linear_theta_edges_deg(0.0, 3.0, 17)), True),
        (cos_edges_from_theta_deg(log_theta_edges_deg(0.5 / 60.0, 180.0, 40)), False),
        (cos_edges_from_theta_deg(log_theta_edges_deg(1.0 / 60.0, 10.0, 300)), False),
    ]
    for edges, auto in cases:
        nb = edges.size - 1
        want = acf.counts_to_numpy(acf.acf_pair_count(ctx, da, None if auto else db_, edges, auto))
        got, gbad = acf.acf_pair_count_static(da, None if auto else db_, edges, auto, d_counts=out[:nb], d_bad=bad)
        torch.cuda.synchronize()
        assert int(gbad.item()) == 0
        assert acf.counts_to_numpy(got).tolist() == want.tolist()
        assert want.tolist() == oracle.pair_count(a, None if auto else b, edges, auto).tolist()
    # two calls enqueued back to back on one stream, read afterwards: stream order keeps them apart
    e1, e2 = cases[0][0], cases[2][0]
    o1 = torch.empty(e1.size - 1, dtype=torch.int64, device="cuda")
    o2 = torch.empty(e2.size - 1, dtype=torch.int64, device="cuda")
    acf.acf_pair_count_static(da, db_, e1, False, d_counts=o1, d_bad=bad)
    acf.acf_pair_count_static(db_, None, e2, True, d_counts=o2, d_bad=bad)
    torch.cuda.synchronize()
    assert acf.counts_to_numpy(o1).tolist() == oracle.pair_count(a, b, e1, False).tolist()
    assert acf.counts_to_numpy(o2).tolist() == oracle.pair_count(b, None, e2, True).tolist()


def test_static_entry_point_limits_and_degenerate_sizes(acf):
    import torch
    edges = cos_edges_from_theta_deg(log_theta_edges_deg(0.1, 20.0, 12))
    # one point more than the fixed array serves: a clear error, nothing enqueued
    big = torch.zeros(3 * (acf.ACF_STATIC_MAX_POINTS + 1), dtype=torch.float64, device="cuda")
    with pytest.raises(acf.AcfError) as ei:
        acf.acf_pair_count_static(big, None, edges, True)
    assert ei.value.code == -1 and "ACF_STATIC_MAX_POINTS" in str(ei.value)
    with pytest.raises(acf.AcfError):
        acf.acf_pair_count_static(big[:30], None, edges[::-1].copy(), True)  # ascending edges
    # empty and one-point catalogues: all-zero counts
    for n in (0, 1):
        got, bad = acf.acf_pair_count_static(torch.tensor([1.0, 0.0, 0.0] * n, dtype=torch.float64, device="cuda").reshape(n, 3).t().contiguous().flatten(),
                                             None, edges, True)
        torch.cuda.synchronize()
        assert got.tolist() == [0] * 12 and int(bad.item()) == 0
    # invalid points are reported in d_bad (the call does not wait for the verdict)
    x = torch.tensor([1.0, 0.0, 0.5, 0.0, 1.0, 0.5, 0.0, 0.0, 0.5], dtype=torch.float64, device="cuda")  # third point: |u|^2 = 0.75
    _, bad = acf.acf_pair_count_static(x, None, edges, True)
    torch.cuda.synchronize()
    assert int(bad.item()) == 1
    # the largest size it takes, against the closed form of the total: every pair of a full-range histogram is counted
    n = acf.ACF_STATIC_MAX_POINTS
    ra, dec = uniform_patch(n, (0.0, 360.0), (-90.0, 90.0), 73)
    full = np.array([1.0, 0.5, 0.0, -0.5, -1.0])
    got, bad = acf.acf_pair_count_static(dev(acf.acf_radec_to_xyz(ra, dec)), None, full, True)
    torch.cuda.synchronize()
    assert int(bad.item()) == 0 and int(acf.counts_to_numpy(got).sum()) == n * (n - 1) // 2
