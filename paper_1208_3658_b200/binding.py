"""Thin Python face of libacf.so (include/acf.h): argument marshalling only.

Every function has the name and the argument order of its C entry point; device buffers are
torch CUDA tensors (PyTorch is used for device memory and streams, nothing else), host buffers
are numpy arrays.  Every step of the method runs inside the library's kernels.  There is no
fallback: if libacf.so cannot be loaded this module raises.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

ACF_OK, ACF_EINVAL, ACF_ENOMEM, ACF_ECUDA = 0, -1, -2, -3
ACF_OPT_KERNEL, ACF_OPT_PRUNE, ACF_OPT_STATS, ACF_OPT_WINDOWS, ACF_OPT_BULK = 1, 2, 3, 4, 5
ACF_KERNEL_AUTO, ACF_KERNEL_FP64, ACF_KERNEL_TABLE, ACF_KERNEL_WINDOW = 0, 1, 2, 3
ACF_MAX_BINS = 1024
ACF_EST_LANDY_SZALAY, ACF_EST_NATURAL, ACF_EST_DAVIS_PEEBLES, ACF_EST_HAMILTON = 0, 1, 2, 3
ACF_BINS_EVEN, ACF_BINS_LOG, ACF_BINS_LOG10 = 0, 1, 2

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libacf.so")

EXPORTS = [
    "acf_create", "acf_destroy", "acf_last_error", "acf_set_option", "acf_set_stream", "acf_radec_to_xyz",
    "acf_pair_count", "acf_pair_count_weighted", "acf_pair_count_rows", "acf_wtheta", "acf_wtheta_weighted",
    "acf_estimator", "acf_theta_edges", "acf_cos_edges", "acf_jackknife", "acf_correlate_host", "acf_get_stats", "acf_version",
    "acf_prepare", "acf_prepare_rows", "acf_prepare_again", "acf_release", "acf_pair_count_prepared", "acf_random_ensemble",
    "acf_pair_count_static",
]


class AcfError(RuntimeError):
    def __init__(self, code, message):
        super().__init__("libacf error %d: %s" % (code, message))
        self.code = code


class acf_stats(ctypes.Structure):
    _fields_ = [
        ("pairs_nominal", ctypes.c_uint64), ("pairs_evaluated", ctypes.c_uint64), ("pairs_fp64", ctypes.c_uint64),
        ("pairs_window", ctypes.c_uint64),
        ("tile_pairs_total", ctypes.c_uint64), ("tile_pairs_pruned", ctypes.c_uint64),
        ("kernel_launches", ctypes.c_uint64), ("device_ms", ctypes.c_double), ("pair_kernel_ms", ctypes.c_double),
        ("pairs_chord", ctypes.c_uint64), ("pairs_bulk", ctypes.c_uint64),
    ]

    def as_dict(self):
        return {name: getattr(self, name) for name, _ in self._fields_}


_lib = None


def load_library(build_if_missing: bool = True):
    """dlopen libacf.so (building it with nvcc first if it is absent) and declare prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        if not build_if_missing:
            raise ImportError("libacf.so is missing at %s: run `python -m paper_1208_3658_b200.build`" % LIB_PATH)
        from .build import build_lib
        build_lib()
    lib = ctypes.CDLL(LIB_PATH)
    vp, sz, i32, i64, u64 = ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int, ctypes.c_int64, ctypes.c_uint64
    lib.acf_create.argtypes = [ctypes.POINTER(vp), i32, vp]
    lib.acf_destroy.argtypes = [vp]
    lib.acf_destroy.restype = None
    lib.acf_last_error.argtypes = [vp]
    lib.acf_last_error.restype = ctypes.c_char_p
    lib.acf_set_option.argtypes = [vp, i32, i64]
    lib.acf_set_stream.argtypes = [vp, vp]
    lib.acf_radec_to_xyz.argtypes = [vp, vp, sz, vp]
    lib.acf_pair_count.argtypes = [vp, vp, sz, vp, sz, vp, i32, i32, vp]
    lib.acf_pair_count_weighted.argtypes = [vp, vp, vp, sz, vp, vp, sz, vp, i32, i32, vp, vp]
    lib.acf_pair_count_rows.argtypes = [vp, vp, vp, sz, sz, sz, vp, vp, sz, vp, i32, i32, vp, vp]
    lib.acf_wtheta.argtypes = [vp, vp, vp, u64, u64, i32, vp]
    lib.acf_wtheta_weighted.argtypes = [vp, vp, vp, vp, sz, vp, sz, i32, vp]
    lib.acf_estimator.argtypes = [i32, vp, vp, vp, u64, u64, i32, vp]
    lib.acf_theta_edges.argtypes = [i32, ctypes.c_double, ctypes.c_double, i32, vp]
    lib.acf_cos_edges.argtypes = [vp, i32, vp]
    lib.acf_jackknife.argtypes = [vp, vp, sz, vp, vp, sz, vp, i32, vp, i32, i32, vp, vp, vp]
    lib.acf_correlate_host.argtypes = [vp, vp, vp, vp, sz, vp, vp, vp, sz, vp, i32, vp, vp, vp, vp, vp, vp, vp]
    lib.acf_prepare.argtypes = [vp, vp, vp, sz, ctypes.POINTER(vp)]
    lib.acf_prepare_rows.argtypes = [vp, vp, vp, sz, sz, sz, ctypes.POINTER(vp)]
    lib.acf_prepare_again.argtypes = [vp, vp, vp, vp, sz, sz, sz]
    lib.acf_release.argtypes = [vp, vp]
    lib.acf_release.restype = None
    lib.acf_pair_count_prepared.argtypes = [vp, vp, vp, vp, i32, i32, i32, vp, vp]
    lib.acf_random_ensemble.argtypes = [vp, vp, vp, vp, i32, vp, i32, i32, vp, vp, vp, vp, vp, vp]
    lib.acf_pair_count_static.argtypes = [i32, vp, sz, vp, sz, vp, i32, i32, vp, vp, vp, ctypes.c_char_p, sz]
    lib.acf_get_stats.argtypes = [vp, ctypes.POINTER(acf_stats)]
    lib.acf_version.restype = ctypes.c_char_p
    for name in EXPORTS:
        getattr(lib, name)  # AttributeError here = the library does not export what acf.h declares
    _lib = lib
    return lib


def _raise(ctx, rc):
    msg = load_library().acf_last_error(ctx)
    raise AcfError(rc, msg.decode() if msg else "")


def _host(a, dtype):
    a = np.ascontiguousarray(a, dtype=dtype)
    return a, a.ctypes.data


def _dev(t, dtype, what):
    import torch
    if t is None:
        return None, 0
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError("%s must be a CUDA torch tensor" % what)
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError("%s must be a contiguous %s tensor" % (what, dtype))
    return t, t.data_ptr()


def _n_points(t):
    if t.dim() != 1 or t.numel() % 3:
        raise ValueError("xyz must be a flat [x|y|z] tensor of length 3n")
    return t.numel() // 3


# ---------------------------------------------------------------- functions named as in acf.h

def acf_version() -> str:
    return load_library().acf_version().decode()


def acf_create(device: int = 0, cuda_stream: int | None = None):
    """-> opaque context handle.  cuda_stream: a raw cudaStream_t (int) or None for torch's current stream AT THIS
    MOMENT: the context stays bound to that stream (acf_set_stream changes it); tensors produced on another
    stream must be synchronised with it by the caller."""
    import torch
    lib = load_library()
    if not torch.cuda.is_available():
        raise AcfError(ACF_ECUDA, "no CUDA device: libacf has no CPU fallback")
    if cuda_stream is None:
        cuda_stream = torch.cuda.current_stream(device).cuda_stream
    ctx = ctypes.c_void_p()
    rc = lib.acf_create(ctypes.byref(ctx), int(device), ctypes.c_void_p(cuda_stream))
    if rc != ACF_OK:
        _raise(None, rc)
    return ctx


def acf_destroy(ctx) -> None:
    load_library().acf_destroy(ctx)


def acf_last_error(ctx) -> str:
    return load_library().acf_last_error(ctx).decode()


def acf_set_option(ctx, option: int, value: int) -> None:
    rc = load_library().acf_set_option(ctx, int(option), int(value))
    if rc != ACF_OK:
        _raise(ctx, rc)


def acf_set_stream(ctx, cuda_stream: int) -> None:
    rc = load_library().acf_set_stream(ctx, ctypes.c_void_p(cuda_stream))
    if rc != ACF_OK:
        _raise(ctx, rc)


def acf_radec_to_xyz(ra_deg, dec_deg) -> np.ndarray:
    """HOST.  -> float64 array of length 3n laid out [x | y | z]."""
    ra, pra = _host(ra_deg, np.float64)
    dec, pdec = _host(dec_deg, np.float64)
    if ra.ndim != 1 or ra.shape != dec.shape:
        raise ValueError("ra/dec must be 1-D and of equal length")
    out = np.empty(3 * ra.size, dtype=np.float64)
    rc = load_library().acf_radec_to_xyz(pra, pdec, ra.size, out.ctypes.data)
    if rc != ACF_OK:
        raise AcfError(rc, "acf_radec_to_xyz")
    return out


def acf_pair_count_rows(ctx, d_a, d_wa, i_begin, i_end, d_b, d_wb, cos_edges, is_auto, d_counts=None, d_wsums=None):
    """DEVICE tensors in, DEVICE tensors out (int64 view of the u64 counts; float64 sums or None).
    Asynchronous on the context's stream."""
    import torch
    a, pa = _dev(d_a, torch.float64, "d_a")
    n_a = _n_points(a)
    if is_auto:
        b, pb, n_b = a, pa, n_a
        d_wb = d_wa
    else:
        b, pb = _dev(d_b, torch.float64, "d_b")
        n_b = _n_points(b)
    e, pe = _host(cos_edges, np.float64)
    nbins = e.size - 1
    weighted = d_wa is not None
    wa, pwa = _dev(d_wa, torch.float32, "d_wa")
    wb, pwb = _dev(d_wb, torch.float32, "d_wb")
    if weighted and (wa.numel() != n_a or wb.numel() != n_b):
        raise ValueError("weight length mismatch")
    if d_counts is None:
        d_counts = torch.empty(max(nbins, 1), dtype=torch.int64, device=a.device)
    if weighted and d_wsums is None:
        d_wsums = torch.empty(max(nbins, 1), dtype=torch.float64, device=a.device)
    _, pc = _dev(d_counts, torch.int64, "d_counts")
    _, pw = _dev(d_wsums, torch.float64, "d_wsums") if weighted else (None, 0)
    rc = load_library().acf_pair_count_rows(ctx, pa, pwa, n_a, int(i_begin), int(i_end), pb, pwb, n_b, pe, nbins,
                                            int(bool(is_auto)), pc, pw)
    if rc != ACF_OK:
        _raise(ctx, rc)
    return (d_counts, d_wsums) if weighted else d_counts


class Catalog:
    """A prepared catalogue (acf_prepare).  Keeps the tensors the handle refers to alive."""

    def __init__(self, ctx, handle, d_xyz, d_w, n):
        self.ctx, self.handle, self.d_xyz, self.d_w, self.n = ctx, handle, d_xyz, d_w, n


def acf_prepare(ctx, d_xyz, d_w=None, rows=None) -> Catalog:
    """DEVICE tensors in; validates, sorts and builds the caps once.  rows=(i_begin, i_end): acf_prepare_rows."""
    import torch
    a, pa = _dev(d_xyz, torch.float64, "d_xyz")
    n = _n_points(a)
    w, pw = _dev(d_w, torch.float32, "d_w")
    if w is not None and w.numel() != n:
        raise ValueError("weight length mismatch")
    h = ctypes.c_void_p()
    if rows is None:
        rc = load_library().acf_prepare(ctx, pa, pw, n, ctypes.byref(h))
        cnt = n
    else:
        rc = load_library().acf_prepare_rows(ctx, pa, pw, n, int(rows[0]), int(rows[1]), ctypes.byref(h))
        cnt = int(rows[1]) - int(rows[0])
    if rc != ACF_OK:
        _raise(ctx, rc)
    return Catalog(ctx, h, a, w, cnt)


def acf_prepare_rows(ctx, d_xyz, d_w, i_begin, i_end) -> Catalog:
    return acf_prepare(ctx, d_xyz, d_w, rows=(i_begin, i_end))


def acf_prepare_again(ctx, cat: Catalog, d_xyz, d_w=None, rows=None) -> Catalog:
    """Re-prepares the handle on new data, reusing its device memory."""
    import torch
    a, pa = _dev(d_xyz, torch.float64, "d_xyz")
    n = _n_points(a)
    w, pw = _dev(d_w, torch.float32, "d_w")
    lo, hi = (0, n) if rows is None else (int(rows[0]), int(rows[1]))
    rc = load_library().acf_prepare_again(ctx, cat.handle, pa, pw, n, lo, hi)
    cat.d_xyz, cat.d_w, cat.n = a, w, hi - lo
    if rc != ACF_OK:
        _raise(ctx, rc)
    return cat


def acf_release(ctx, cat: Catalog) -> None:
    if cat is not None and cat.handle is not None:
        load_library().acf_release(ctx, cat.handle)
        cat.handle = None


def acf_pair_count_prepared(ctx, a: Catalog, b: Catalog | None, cos_edges, part: int = 0, n_parts: int = 1, weighted=None,
                            d_counts=None, d_wsums=None):
    """Counts on prepared catalogues; b None: auto-count of a.  Asynchronous.  weighted defaults to "a has weights".
    -> d_counts, or (d_counts, d_wsums)."""
    import torch
    e, pe = _host(cos_edges, np.float64)
    nbins = e.size - 1
    if weighted is None:
        weighted = a.d_w is not None and (b is None or b.d_w is not None)
    dev = a.d_xyz.device
    if d_counts is None:
        d_counts = torch.empty(max(nbins, 1), dtype=torch.int64, device=dev)
    if weighted and d_wsums is None:
        d_wsums = torch.empty(max(nbins, 1), dtype=torch.float64, device=dev)
    _, pc = _dev(d_counts, torch.int64, "d_counts")
    _, pw = _dev(d_wsums, torch.float64, "d_wsums") if weighted else (None, 0)
    rc = load_library().acf_pair_count_prepared(ctx, a.handle, None if b is None else b.handle, pe, nbins, int(part), int(n_parts), pc, pw)
    if rc != ACF_OK:
        _raise(ctx, rc)
    return (d_counts, d_wsums) if weighted else d_counts


def acf_pair_count(ctx, d_a, d_b, cos_edges, is_auto, d_counts=None):
    import torch
    a, pa = _dev(d_a, torch.float64, "d_a")
    n_a = _n_points(a)
    if is_auto:
        pb, n_b = pa, n_a
    else:
        b, pb = _dev(d_b, torch.float64, "d_b")
        n_b = _n_points(b)
    e, pe = _host(cos_edges, np.float64)
    nbins = e.size - 1
    if d_counts is None:
        d_counts = torch.empty(max(nbins, 1), dtype=torch.int64, device=a.device)
    _, pc = _dev(d_counts, torch.int64, "d_counts")
    rc = load_library().acf_pair_count(ctx, pa, n_a, pb, n_b, pe, nbins, int(bool(is_auto)), pc)
    if rc != ACF_OK:
        _raise(ctx, rc)
    return d_counts


ACF_STATIC_MAX_POINTS = 131072


def acf_pair_count_static(d_a, d_b, cos_edges, is_auto, d_counts=None, d_bad=None, cuda_stream=None):
    """The count of acf_pair_count by the entry point that allocates nothing (no context; at most
    ACF_STATIC_MAX_POINTS points per catalogue).  Pass d_counts (int64[nbins]) and d_bad (int32[1]) to keep this
    wrapper from allocating too.  cuda_stream: a raw cudaStream_t (int) or None for torch's current stream.
    -> (d_counts, d_bad); asynchronous."""
    import torch
    a, pa = _dev(d_a, torch.float64, "d_a")
    n_a = _n_points(a)
    if is_auto:
        pb, n_b = pa, n_a
    else:
        b, pb = _dev(d_b, torch.float64, "d_b")
        n_b = _n_points(b)
    e, pe = _host(cos_edges, np.float64)
    nbins = e.size - 1
    if d_counts is None:
        d_counts = torch.empty(max(nbins, 1), dtype=torch.int64, device=a.device)
    if d_bad is None:
        d_bad = torch.empty(1, dtype=torch.int32, device=a.device)
    _, pc = _dev(d_counts, torch.int64, "d_counts")
    _, pbad = _dev(d_bad, torch.int32, "d_bad")
    if cuda_stream is None:
        cuda_stream = torch.cuda.current_stream(a.device).cuda_stream
    err = ctypes.create_string_buffer(512)
    rc = load_library().acf_pair_count_static(a.device.index, pa, n_a, pb, n_b, pe, nbins, int(bool(is_auto)), pc, pbad,
                                              cuda_stream, err, len(err))
    if rc != ACF_OK:
        raise AcfError(rc, err.value.decode())
    return d_counts, d_bad


def acf_pair_count_weighted(ctx, d_a, d_wa, d_b, d_wb, cos_edges, is_auto, d_counts=None, d_wsums=None):
    import torch
    a, _ = _dev(d_a, torch.float64, "d_a")
    if d_wa is None:
        raise ValueError("d_wa is required")
    return acf_pair_count_rows(ctx, a, d_wa, 0, _n_points(a), d_b, d_wb, cos_edges, is_auto, d_counts, d_wsums)


def acf_wtheta(dd, dr, rr, n_d: int, n_r: int) -> np.ndarray:
    dd, pdd = _host(dd, np.uint64)
    dr, pdr = _host(dr, np.uint64)
    rr, prr = _host(rr, np.uint64)
    w = np.empty(dd.size, dtype=np.float64)
    rc = load_library().acf_wtheta(pdd, pdr, prr, int(n_d), int(n_r), dd.size, w.ctypes.data)
    if rc != ACF_OK:
        raise AcfError(rc, "acf_wtheta")
    return w


def acf_estimator(kind: int, dd, dr, rr, n_d: int, n_r: int) -> np.ndarray:
    dd, pdd = _host(dd, np.uint64)
    dr, pdr = _host(dr, np.uint64)
    rr, prr = _host(rr, np.uint64)
    w = np.empty(dd.size, dtype=np.float64)
    rc = load_library().acf_estimator(int(kind), pdd, pdr, prr, int(n_d), int(n_r), dd.size, w.ctypes.data)
    if rc != ACF_OK:
        raise AcfError(rc, "acf_estimator")
    return w


def acf_theta_edges(mode: int, lo_deg: float, hi_deg: float, nbins: int) -> np.ndarray:
    theta = np.empty(max(0, int(nbins)) + 1, dtype=np.float64)
    rc = load_library().acf_theta_edges(int(mode), float(lo_deg), float(hi_deg), int(nbins), theta.ctypes.data)
    if rc != ACF_OK:
        raise AcfError(rc, "acf_theta_edges")
    return theta


def acf_cos_edges(theta_deg) -> np.ndarray:
    theta, pt = _host(theta_deg, np.float64)
    out = np.empty(theta.size, dtype=np.float64)
    rc = load_library().acf_cos_edges(pt, theta.size, out.ctypes.data)
    if rc != ACF_OK:
        raise AcfError(rc, "acf_cos_edges")
    return out


def acf_jackknife(ctx, d_xyz_d, off_d, d_xyz_r, off_r, cos_edges, estimator: int = ACF_EST_LANDY_SZALAY) -> dict:
    """Delete-one jackknife over regions; the catalogues (device tensors) are ordered by region and
    off_d / off_r give each region's row range.  -> {"w": ..., "w_jk": (regions, nbins), "cov": (nbins, nbins)}."""
    import torch
    d_xyz_d, _ = _dev(d_xyz_d, torch.float64, "d_xyz_d")
    d_xyz_r, _ = _dev(d_xyz_r, torch.float64, "d_xyz_r")
    off_d = np.ascontiguousarray(off_d, dtype=np.uint64)
    off_r = np.ascontiguousarray(off_r, dtype=np.uint64)
    edges, pe = _host(cos_edges, np.float64)
    nbins, n_regions = edges.size - 1, off_d.size - 1
    if off_r.size != off_d.size:
        raise ValueError("off_d and off_r must name the same regions")
    w = np.empty(nbins, dtype=np.float64)
    w_jk = np.empty((n_regions, nbins), dtype=np.float64)
    cov = np.empty((nbins, nbins), dtype=np.float64)
    rc = load_library().acf_jackknife(ctx, d_xyz_d.data_ptr(), _n_points(d_xyz_d), off_d.ctypes.data, d_xyz_r.data_ptr(),
                                      _n_points(d_xyz_r), off_r.ctypes.data, n_regions, pe, nbins, int(estimator),
                                      w.ctypes.data, w_jk.ctypes.data, cov.ctypes.data)
    if rc != ACF_OK:
        raise AcfError(rc, acf_last_error(ctx))
    return {"w": w, "w_jk": w_jk, "cov": cov}


def acf_random_ensemble(ctx, data: Catalog, d_xyz_r_list, cos_edges, estimator: int = ACF_EST_LANDY_SZALAY) -> dict:
    """Monte-Carlo errors from an ensemble of random catalogues (device tensors).
    -> {"dd", "dr" (K, nbins), "rr" (K, nbins), "w" (K, nbins), "mean", "cov"}."""
    import torch
    K = len(d_xyz_r_list)
    tensors = [_dev(t, torch.float64, "d_xyz_r[%d]" % k)[0] for k, t in enumerate(d_xyz_r_list)]
    ptrs = (ctypes.c_void_p * K)(*[t.data_ptr() for t in tensors])
    sizes = (ctypes.c_size_t * K)(*[_n_points(t) for t in tensors])
    e, pe = _host(cos_edges, np.float64)
    nbins = e.size - 1
    out = {"dd": np.zeros(nbins, np.uint64), "dr": np.zeros((K, nbins), np.uint64), "rr": np.zeros((K, nbins), np.uint64),
           "w": np.zeros((K, nbins)), "mean": np.zeros(nbins), "cov": np.zeros((nbins, nbins)) if K > 1 else None}
    rc = load_library().acf_random_ensemble(ctx, data.handle, ctypes.cast(ptrs, ctypes.c_void_p), ctypes.cast(sizes, ctypes.c_void_p), K, pe, nbins,
                                            int(estimator), out["dd"].ctypes.data, out["dr"].ctypes.data, out["rr"].ctypes.data,
                                            out["w"].ctypes.data, out["mean"].ctypes.data, out["cov"].ctypes.data if K > 1 else None)
    if rc != ACF_OK:
        _raise(ctx, rc)
    return out


def acf_wtheta_weighted(wdd, wdr, wrr, w_d, w_r) -> np.ndarray:
    wdd, p1 = _host(wdd, np.float64)
    wdr, p2 = _host(wdr, np.float64)
    wrr, p3 = _host(wrr, np.float64)
    w_d, p4 = _host(w_d, np.float32)
    w_r, p5 = _host(w_r, np.float32)
    w = np.empty(wdd.size, dtype=np.float64)
    rc = load_library().acf_wtheta_weighted(p1, p2, p3, p4, w_d.size, p5, w_r.size, wdd.size, w.ctypes.data)
    if rc != ACF_OK:
        raise AcfError(rc, "acf_wtheta_weighted")
    return w


def acf_correlate_host(ctx, ra_d, dec_d, w_d, ra_r, dec_r, w_r, cos_edges):
    """HOST arrays in, HOST arrays out; synchronous.  -> dict(dd, dr, rr, [wdd, wdr, wrr], w)."""
    ra_d, p1 = _host(ra_d, np.float64)
    dec_d, p2 = _host(dec_d, np.float64)
    ra_r, p3 = _host(ra_r, np.float64)
    dec_r, p4 = _host(dec_r, np.float64)
    e, pe = _host(cos_edges, np.float64)
    nbins = e.size - 1
    weighted = w_d is not None
    pw1 = pw2 = 0
    if weighted:
        w_d, pw1 = _host(w_d, np.float32)
        w_r, pw2 = _host(w_r, np.float32)
    out = {k: np.zeros(max(nbins, 1), dtype=np.uint64) for k in ("dd", "dr", "rr")}
    if weighted:
        out.update({k: np.zeros(max(nbins, 1), dtype=np.float64) for k in ("wdd", "wdr", "wrr")})
    out["w"] = np.zeros(max(nbins, 1), dtype=np.float64)
    g = lambda k: out[k].ctypes.data if k in out else 0
    rc = load_library().acf_correlate_host(ctx, p1, p2, pw1, ra_d.size, p3, p4, pw2, ra_r.size, pe, nbins,
                                           g("dd"), g("dr"), g("rr"), g("wdd"), g("wdr"), g("wrr"), g("w"))
    if rc != ACF_OK:
        _raise(ctx, rc)
    return out


def acf_get_stats(ctx) -> dict:
    st = acf_stats()
    rc = load_library().acf_get_stats(ctx, ctypes.byref(st))
    if rc != ACF_OK:
        _raise(ctx, rc)
    return st.as_dict()


def counts_to_numpy(d_counts) -> np.ndarray:
    """Device int64 view of u64 counts -> host uint64 array (synchronises)."""
    return d_counts.cpu().numpy().view(np.uint64)
