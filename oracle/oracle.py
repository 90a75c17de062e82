"""ctypes face of oracle/acf_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It builds the C oracle with gcc on first use (or when
the source is newer than the shared object) and marshals numpy arrays.  The definition
(O1-O8) lives in acf_oracle.c, with citations into PAPER.md (arXiv 1208.3658 sect. 2, Eq. 2,
Appendix A); the only arithmetic written here is the resampling at the end of the file: the delete-one
jackknife (`jackknife`, `jackknife_cov`: remove a region, recount with the C functions, numpy mean
and outer products) and the ensemble of random catalogues (`random_ensemble`: one count per
catalogue, numpy mean and sample covariance), pinned on hand examples in tests/test_oracle_pins.py.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "acf_oracle.c")
_LIB = os.path.join(_HERE, "libacf_oracle.so")
_CFLAGS = ["-O2", "-mfma", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC", "-std=c11"]
_lock = threading.Lock()
_lib = None

c_double_p = ctypes.POINTER(ctypes.c_double)
c_float_p = ctypes.POINTER(ctypes.c_float)
c_u64_p = ctypes.POINTER(ctypes.c_uint64)


def build(force: bool = False) -> str:
    """Compile acf_oracle.c -> libacf_oracle.so (beside the source). Returns the path."""
    stale = force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
    if stale:
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.run(["gcc", *_CFLAGS, _SRC, "-o", tmp, "-lm"], check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    with _lock:
        if _lib is None:
            lib = ctypes.CDLL(build())
            sz = ctypes.c_size_t
            lib.oracle_num_threads.restype = ctypes.c_int
            lib.oracle_set_num_threads.argtypes = [ctypes.c_int]
            lib.oracle_radec_to_xyz.argtypes = [c_double_p, c_double_p, sz, c_double_p]
            lib.oracle_pair_count_rows.argtypes = [
                c_double_p, c_float_p, sz, sz, sz, c_double_p, c_float_p, sz,
                c_double_p, ctypes.c_int, ctypes.c_int, c_u64_p, c_double_p]
            lib.oracle_pair_count.argtypes = [
                c_double_p, sz, c_double_p, sz, c_double_p, ctypes.c_int, ctypes.c_int, c_u64_p]
            lib.oracle_pair_count_weighted.argtypes = [
                c_double_p, c_float_p, sz, c_double_p, c_float_p, sz, c_double_p, ctypes.c_int,
                ctypes.c_int, c_u64_p, c_double_p]
            lib.oracle_pair_count_decwindow.argtypes = [
                c_double_p, c_double_p, sz, c_double_p, c_double_p, sz, c_double_p, ctypes.c_int,
                ctypes.c_int, c_u64_p]
            lib.oracle_pair_count_cellwindow.argtypes = [
                c_double_p, c_double_p, c_double_p, sz, sz, sz, c_double_p, c_double_p, c_double_p, sz,
                c_double_p, ctypes.c_int, ctypes.c_int, c_u64_p]
            lib.oracle_pair_count_theta.argtypes = [
                c_double_p, c_double_p, sz, c_double_p, c_double_p, sz, c_double_p, ctypes.c_int,
                ctypes.c_int, ctypes.c_double, c_u64_p, c_u64_p, c_u64_p, sz]
            lib.oracle_wtheta.argtypes = [c_u64_p, c_u64_p, c_u64_p, ctypes.c_uint64, ctypes.c_uint64,
                                          ctypes.c_int, c_double_p]
            lib.oracle_estimator.argtypes = [ctypes.c_int, c_u64_p, c_u64_p, c_u64_p, ctypes.c_uint64, ctypes.c_uint64,
                                             ctypes.c_int, c_double_p]
            lib.oracle_theta_edges.argtypes = [ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_int, c_double_p]
            lib.oracle_cos_edges.argtypes = [c_double_p, ctypes.c_int, c_double_p]
            lib.oracle_wtheta_weighted.argtypes = [c_double_p, c_double_p, c_double_p, c_float_p, sz,
                                                   c_float_p, sz, ctypes.c_int, c_double_p]
            _lib = lib
    return _lib


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(c_double_p)


def _f32(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a, a.ctypes.data_as(c_float_p)


def _u64(a):
    a = np.ascontiguousarray(a, dtype=np.uint64)
    return a, a.ctypes.data_as(c_u64_p)


def _check(rc, what):
    if rc != 0:
        raise ValueError("%s failed with code %d" % (what, rc))


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().oracle_set_num_threads(int(n))


def radec_to_xyz(ra_deg, dec_deg) -> np.ndarray:
    """O1. Returns xyz as one float64 array of length 3n laid out [x | y | z]."""
    ra, pra = _f64(ra_deg)
    dec, pdec = _f64(dec_deg)
    if ra.shape != dec.shape or ra.ndim != 1:
        raise ValueError("ra/dec must be 1-D and of equal length")
    out = np.empty(3 * ra.size, dtype=np.float64)
    _check(_load().oracle_radec_to_xyz(pra, pdec, ra.size, out.ctypes.data_as(c_double_p)), "radec_to_xyz")
    return out


def _n_of(xyz) -> int:
    if xyz.ndim != 1 or xyz.size % 3:
        raise ValueError("xyz must be a flat [x|y|z] array")
    return xyz.size // 3


def pair_count(xyz_a, xyz_b, cos_edges, is_auto: bool, w_a=None, w_b=None, rows=None):
    """O2-O6. xyz_b is ignored (taken as xyz_a) when is_auto. Returns counts, or
    (counts, wsums) when weights are given. rows=(i0, i1) restricts A's rows."""
    a, pa = _f64(xyz_a)
    n_a = _n_of(a)
    if is_auto:
        b, pb, n_b = a, pa, n_a
    else:
        b, pb = _f64(xyz_b)
        n_b = _n_of(b)
    e, pe = _f64(cos_edges)
    nbins = e.size - 1
    counts = np.zeros(max(nbins, 1), dtype=np.uint64)
    i0, i1 = (0, n_a) if rows is None else rows
    weighted = w_a is not None
    if weighted:
        wa, pwa = _f32(w_a)
        if is_auto:
            wb, pwb = wa, pwa
        else:
            wb, pwb = _f32(w_b)
        if wa.size != n_a or wb.size != n_b:
            raise ValueError("weight length mismatch")
        wsums = np.zeros(max(nbins, 1), dtype=np.float64)
        pws = wsums.ctypes.data_as(c_double_p)
    else:
        pwa = pwb = ctypes.cast(None, c_float_p)
        pws = ctypes.cast(None, c_double_p)
    rc = _load().oracle_pair_count_rows(pa, pwa, n_a, i0, i1, pb, pwb, n_b, pe, nbins, int(bool(is_auto)),
                                        counts.ctypes.data_as(c_u64_p), pws)
    _check(rc, "pair_count")
    return (counts, wsums) if weighted else counts


def pair_count_decwindow(xyz_a, dec_a_deg, xyz_b, dec_b_deg, cos_edges, is_auto: bool):
    a, pa = _f64(xyz_a)
    da, pda = _f64(dec_a_deg)
    if is_auto:
        b, pb, db, pdb = a, pa, da, pda
    else:
        b, pb = _f64(xyz_b)
        db, pdb = _f64(dec_b_deg)
    e, pe = _f64(cos_edges)
    nbins = e.size - 1
    counts = np.zeros(max(nbins, 1), dtype=np.uint64)
    rc = _load().oracle_pair_count_decwindow(pa, pda, _n_of(a), pb, pdb, _n_of(b), pe, nbins,
                                             int(bool(is_auto)), counts.ctypes.data_as(c_u64_p))
    _check(rc, "pair_count_decwindow")
    return counts


def pair_count_cellwindow(xyz_a, ra_a_deg, dec_a_deg, xyz_b, ra_b_deg, dec_b_deg, cos_edges, is_auto: bool, rows=None):
    """O2-O6 with the Dec + RA window of acf_oracle.c (a superset of the counted pairs): configs 3 and 5."""
    a, pa = _f64(xyz_a)
    ra, pra = _f64(ra_a_deg)
    da, pda = _f64(dec_a_deg)
    if is_auto:
        b, pb, rb, prb, db, pdb = a, pa, ra, pra, da, pda
    else:
        b, pb = _f64(xyz_b)
        rb, prb = _f64(ra_b_deg)
        db, pdb = _f64(dec_b_deg)
    if ra.size != _n_of(a) or da.size != _n_of(a) or rb.size != _n_of(b) or db.size != _n_of(b):
        raise ValueError("ra/dec length mismatch")
    e, pe = _f64(cos_edges)
    nbins = e.size - 1
    counts = np.zeros(max(nbins, 1), dtype=np.uint64)
    i0, i1 = (0, _n_of(a)) if rows is None else rows
    rc = _load().oracle_pair_count_cellwindow(pa, pra, pda, _n_of(a), i0, i1, pb, prb, pdb, _n_of(b), pe, nbins,
                                              int(bool(is_auto)), counts.ctypes.data_as(c_u64_p))
    _check(rc, "pair_count_cellwindow")
    return counts


def pair_count_theta(ra_a, dec_a, ra_b, dec_b, theta_edges_deg, is_auto: bool, rel_tol=1e-9, near_cap=1024):
    """O8 (Appendix A trig formula). Returns (counts, n_near, near_pairs[(i, j)...])."""
    ra1, p1 = _f64(ra_a)
    de1, q1 = _f64(dec_a)
    if is_auto:
        ra2, p2, de2, q2 = ra1, p1, de1, q1
    else:
        ra2, p2 = _f64(ra_b)
        de2, q2 = _f64(dec_b)
    te, pte = _f64(theta_edges_deg)
    nbins = te.size - 1
    counts = np.zeros(max(nbins, 1), dtype=np.uint64)
    n_near = ctypes.c_uint64(0)
    near = np.zeros(2 * near_cap, dtype=np.uint64)
    rc = _load().oracle_pair_count_theta(p1, q1, ra1.size, p2, q2, ra2.size, pte, nbins, int(bool(is_auto)),
                                         float(rel_tol), counts.ctypes.data_as(c_u64_p), ctypes.byref(n_near),
                                         near.ctypes.data_as(c_u64_p), near_cap)
    _check(rc, "pair_count_theta")
    k = min(int(n_near.value), near_cap)
    return counts, int(n_near.value), near[: 2 * k].reshape(-1, 2)


def wtheta(dd, dr, rr, n_d: int, n_r: int) -> np.ndarray:
    """O7, Eq. 2."""
    dd, pdd = _u64(dd)
    dr, pdr = _u64(dr)
    rr, prr = _u64(rr)
    w = np.empty(dd.size, dtype=np.float64)
    _check(_load().oracle_wtheta(pdd, pdr, prr, int(n_d), int(n_r), dd.size, w.ctypes.data_as(c_double_p)), "wtheta")
    return w


def estimator(kind: int, dd, dr, rr, n_d: int, n_r: int) -> np.ndarray:
    """0 Landy-Szalay (O7), 1 natural, 2 Davis-Peebles, 3 Hamilton."""
    dd, pdd = _u64(dd)
    dr, pdr = _u64(dr)
    rr, prr = _u64(rr)
    w = np.empty(dd.size, dtype=np.float64)
    _check(_load().oracle_estimator(int(kind), pdd, pdr, prr, int(n_d), int(n_r), dd.size, w.ctypes.data_as(c_double_p)), "estimator")
    return w


def theta_edges(mode: int, lo_deg: float, hi_deg: float, nbins: int) -> np.ndarray:
    """0 even, 1 natural log, 2 log10 (the two give the same edges)."""
    theta = np.empty(int(nbins) + 1, dtype=np.float64)
    _check(_load().oracle_theta_edges(int(mode), ctypes.c_double(lo_deg), ctypes.c_double(hi_deg), int(nbins),
                                      theta.ctypes.data_as(c_double_p)), "theta_edges")
    return theta


def cos_edges(theta_deg) -> np.ndarray:
    theta, pt = _f64(theta_deg)
    e = np.empty(theta.size, dtype=np.float64)
    _check(_load().oracle_cos_edges(pt, theta.size, e.ctypes.data_as(c_double_p)), "cos_edges")
    return e


def jackknife_cov(w_jk) -> np.ndarray:
    """Delete-one jackknife covariance of N resampled estimates (rows of w_jk):
    cov = (N - 1)/N sum_k (w_k - mean)(w_k - mean)^T, mean = (1/N) sum_k w_k."""
    w_jk = np.asarray(w_jk, dtype=np.float64)
    n = w_jk.shape[0]
    dev = w_jk - w_jk.mean(axis=0)
    return (n - 1) / n * (dev.T @ dev)


def jackknife(xyz_d, region_d, xyz_r, region_r, n_regions: int, cos_edges, kind: int = 0):
    """PAPER.md:201 (resampling errors), by the definition: for every region k the points of region k are
    removed from both catalogues, DD, DR, RR are counted afresh and the estimator is formed.
    region_*: the region index of every point.  -> (w_full, w_jk, cov)."""
    xd = np.asarray(xyz_d, dtype=np.float64).reshape(3, -1)
    xr = np.asarray(xyz_r, dtype=np.float64).reshape(3, -1)
    region_d, region_r = np.asarray(region_d), np.asarray(region_r)

    def est(a, b):
        a, b = np.ascontiguousarray(a).reshape(-1), np.ascontiguousarray(b).reshape(-1)
        dd = pair_count(a, None, cos_edges, True)
        dr = pair_count(a, b, cos_edges, False)
        rr = pair_count(b, None, cos_edges, True)
        return estimator(kind, dd, dr, rr, a.size // 3, b.size // 3)

    w_full = est(xd, xr)
    w_jk = np.stack([est(xd[:, region_d != k], xr[:, region_r != k]) for k in range(n_regions)])
    return w_full, w_jk, jackknife_cov(w_jk)


def ensemble_cov(w_k) -> np.ndarray:
    """Sample covariance of K estimates (rows of w_k): 1/(K - 1) sum_k (w_k - mean)(w_k - mean)^T."""
    w_k = np.asarray(w_k, dtype=np.float64)
    dev = w_k - w_k.mean(axis=0)
    return dev.T @ dev / (w_k.shape[0] - 1)


def random_ensemble(xyz_d, xyz_r_list, cos_edges, kind: int = 0):
    """PAPER.md:201 (Monte-Carlo errors), by the definition: the data counted once, every random catalogue of the
    ensemble counted on its own (DR_k, RR_k), the estimator formed with each.  -> (dd, dr[K], rr[K], w[K], mean, cov)."""
    xd = np.ascontiguousarray(xyz_d, dtype=np.float64)
    dd = pair_count(xd, None, cos_edges, True)
    dr, rr, w = [], [], []
    for xr in xyz_r_list:
        xr = np.ascontiguousarray(xr, dtype=np.float64)
        dr.append(pair_count(xd, xr, cos_edges, False))
        rr.append(pair_count(xr, None, cos_edges, True))
        w.append(estimator(kind, dd, dr[-1], rr[-1], xd.size // 3, xr.size // 3))
    w = np.stack(w)
    return dd, np.stack(dr), np.stack(rr), w, w.mean(axis=0), (ensemble_cov(w) if len(xyz_r_list) > 1 else None)


def wtheta_weighted(dd, dr, rr, w_d, w_r) -> np.ndarray:
    dd, pdd = _f64(dd)
    dr, pdr = _f64(dr)
    rr, prr = _f64(rr)
    wd, pwd = _f32(w_d)
    wr, pwr = _f32(w_r)
    w = np.empty(dd.size, dtype=np.float64)
    _check(_load().oracle_wtheta_weighted(pdd, pdr, prr, pwd, wd.size, pwr, wr.size, dd.size,
                                          w.ctypes.data_as(c_double_p)), "wtheta_weighted")
    return w
