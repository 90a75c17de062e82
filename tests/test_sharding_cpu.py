"""Host logic of the multi-GPU path on CPU: triangle-balanced row ranges and the gloo reduction,
world_size 2.  Each rank counts its row range with the CPU oracle (standing in for its GPU) and the
summed histograms must equal the unsharded count exactly (additivity)."""
import os
import socket

import numpy as np
import pytest

from paper_1208_3658_b200.sharding import pairs_before_row, row_ranges
from workloads import make_config


def test_row_ranges_cover_and_balance():
    for n_a, n_b, auto, world in [(10, 10, True, 3), (1000, 1000, True, 8), (1000, 777, False, 7), (5, 0, False, 2),
                                  (1, 1, True, 4), (0, 0, True, 2), (12345, 12345, True, 2)]:
        rr = row_ranges(n_a, n_b, auto, world)
        assert len(rr) == world and rr[0][0] == 0 and rr[-1][1] == n_a
        assert all(a[1] == b[0] for a, b in zip(rr[:-1], rr[1:])) and all(lo <= hi for lo, hi in rr)
        total = pairs_before_row(n_a, n_a, n_b, auto)
        assert total == (n_a * (n_a - 1) // 2 if auto else n_a * n_b)
        per = [pairs_before_row(hi, n_a, n_b, auto) - pairs_before_row(lo, n_a, n_b, auto) for lo, hi in rr]
        assert sum(per) == total
        if n_a >= 1000:
            assert max(per) - min(per) <= max(n_a, n_b) + 1   # within one row of pairs


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    from oracle import oracle as O
    from paper_1208_3658_b200.sharding import all_reduce_counts, row_ranges
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = make_config("full_sky", 0.002)
        xd, xr = O.radec_to_xyz(w.ra_d, w.dec_d), O.radec_to_xyz(w.ra_r, w.dec_r)
        res = {}
        for key, (a, b, auto, wa, wb) in {"dd": (xd, None, True, w.w_d, None), "dr": (xd, xr, False, w.w_d, w.w_r)}.items():
            n_a = a.size // 3
            n_b = n_a if auto else b.size // 3
            lo, hi = row_ranges(n_a, n_b, auto, world)[rank]
            c, s = O.pair_count(a, b, w.cos_edges, auto, w_a=wa, w_b=wb, rows=(lo, hi))
            ct = torch.from_numpy(c.astype(np.int64))
            st = torch.from_numpy(np.asarray(s, dtype=np.float64).copy())
            all_reduce_counts(ct, st)
            res[key] = (ct.numpy().astype(np.uint64), st.numpy())
            # the slice holds the pairs pairs_before_row says it does: bins over [0, 180] deg catch them all
            from paper_1208_3658_b200.sharding import pairs_before_row
            c_all = O.pair_count(a, b, np.array([1.0, 0.0, -1.0]), auto, rows=(lo, hi))
            assert int(c_all.sum()) == pairs_before_row(hi, n_a, n_b, auto) - pairs_before_row(lo, n_a, n_b, auto)
        if rank == 0:
            q.put(res)
    finally:
        dist.destroy_process_group()


def test_gloo_world2_sharded_counts_equal_unsharded(oracle):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = make_config("full_sky", 0.002)
    xd, xr = oracle.radec_to_xyz(w.ra_d, w.dec_d), oracle.radec_to_xyz(w.ra_r, w.dec_r)
    dd, wdd = oracle.pair_count(xd, None, w.cos_edges, True, w_a=w.w_d)
    dr, wdr = oracle.pair_count(xd, xr, w.cos_edges, False, w_a=w.w_d, w_b=w.w_r)
    assert res["dd"][0].tolist() == dd.tolist() and res["dr"][0].tolist() == dr.tolist()
    np.testing.assert_allclose(res["dd"][1], wdd, rtol=1e-12)
    np.testing.assert_allclose(res["dr"][1], wdr, rtol=1e-12)
