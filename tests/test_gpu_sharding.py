"""The row-sharded count of paper_1208_3658_b200.sharding on a GPU (the pair matrix cut into
sub-matrices; "division of the dataset into sub-sets ... clusters of independent GPUs").

One device stands in for the ranks one after the other -- the ranks of a sharded count never wait on one
another, their only exchange is the sum of the histograms at the end -- so every rank's slice goes through
acf_pair_count_rows exactly as sharded_pair_count issues it, and the summed histograms must equal the
one-call result bit for bit (weighted sums to 1e-12), at the full sizes of configurations 4 and 3.
"""
import numpy as np
import pytest

from paper_1208_3658_b200.sharding import pairs_before_row, row_ranges, sharded_pair_count, sharded_pair_count_prepared
from workloads import make_config

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


def to_np(acf, out, weighted):
    if weighted:
        return acf.counts_to_numpy(out[0]), out[1].cpu().numpy()
    return acf.counts_to_numpy(out[0] if isinstance(out, tuple) else out), None


@pytest.mark.parametrize("name,scale,world", [("full_sky", 1.0, 8), ("survey_scale", 1.0, 4), ("tiny", 0.0005, 8)])
def test_rank_slices_add_up_to_the_unsharded_count(acf, ctx, name, scale, world):
    import torch
    w = make_config(name, scale)
    weighted = w.w_d is not None
    xd = torch.from_numpy(acf.acf_radec_to_xyz(w.ra_d, w.dec_d)).cuda()
    xr = torch.from_numpy(acf.acf_radec_to_xyz(w.ra_r, w.dec_r)).cuda()
    wd = torch.from_numpy(w.w_d).cuda() if weighted else None
    wr = torch.from_numpy(w.w_r).cuda() if weighted else None
    for a, wa, b, wb, auto in ((xd, wd, None, None, True), (xd, wd, xr, wr, False)):
        n_a = a.numel() // 3
        n_b = n_a if auto else b.numel() // 3
        whole = acf.acf_pair_count_rows(ctx, a, wa, 0, n_a, b, wb, w.cos_edges, auto)
        torch.cuda.synchronize()
        whole_c, whole_w = to_np(acf, whole, weighted)
        sum_c = np.zeros_like(whole_c)
        sum_w = np.zeros(w.nbins)
        nominal = 0
        for rank in range(world):
            # no process group: the reduction inside is a no-op and the rank's own histogram comes back
            out = sharded_pair_count(ctx, a, wa, b, wb, w.cos_edges, auto, rank, world)
            torch.cuda.synchronize()
            c, s = to_np(acf, out, weighted)
            st = acf.acf_get_stats(ctx)
            lo, hi = row_ranges(n_a, n_b, auto, world)[rank]
            assert st["pairs_nominal"] == pairs_before_row(hi, n_a, n_b, auto) - pairs_before_row(lo, n_a, n_b, auto)
            nominal += st["pairs_nominal"]
            sum_c += c
            if weighted:
                sum_w += s
        assert nominal == (n_a * (n_a - 1) // 2 if auto else n_a * n_b)
        assert sum_c.tolist() == whole_c.tolist(), (name, auto)
        if weighted:
            np.testing.assert_allclose(sum_w, whole_w, rtol=1e-12, atol=0)
        # the same job on prepared catalogues: interleaved tile slices, nothing prepared twice
        ca = acf.acf_prepare(ctx, a, wa)
        cb = None if auto else acf.acf_prepare(ctx, b, wb)
        sum_c[:] = 0
        sum_w[:] = 0
        evaluated = []
        for rank in range(world):
            out = sharded_pair_count_prepared(ctx, ca, cb, w.cos_edges, rank, world)
            torch.cuda.synchronize()
            c, s = to_np(acf, out, weighted)
            evaluated.append(acf.acf_get_stats(ctx)["pairs_evaluated"])
            sum_c += c
            if weighted:
                sum_w += s
        acf.acf_release(ctx, ca)
        acf.acf_release(ctx, cb)
        assert sum_c.tolist() == whole_c.tolist(), (name, auto, "prepared")
        if weighted:
            np.testing.assert_allclose(sum_w, whole_w, rtol=1e-12, atol=0)
        if scale == 1.0:
            assert max(evaluated) <= 1.15 * (sum(evaluated) / world), evaluated   # the slices are balanced
    if scale < 0.01:
        # more ranks than rows: empty slices are legal and count nothing
        assert any(lo == hi for lo, hi in row_ranges(w.n_d, w.n_d, True, 64))
        tot = sum(int(acf.counts_to_numpy(sharded_pair_count(ctx, xd, None, None, None, w.cos_edges, True, r, 64)[0]).sum())
                  for r in range(64))
        assert tot == int(acf.counts_to_numpy(acf.acf_pair_count(ctx, xd, None, w.cos_edges, True)).sum())
