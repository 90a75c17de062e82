"""CPU-side checks of libacf.so (-m "not gpu"): it builds, loads, exports every symbol that
include/acf.h declares, its pure-host entry points agree with the oracle, and with no GPU it
fails loudly instead of falling back."""
import ctypes
import math
import os
import re

import numpy as np
import pytest

from conftest import ROOT, read_golden
from workloads import full_sky


@pytest.fixture(scope="module")
def acf():
    import paper_1208_3658_b200 as P
    P.load_library()
    return P


def test_exports_match_header(acf):
    header = open(os.path.join(ROOT, "include", "acf.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(acf_[a-z0-9_]+)\s*\(", header))
    assert {"acf_create", "acf_pair_count", "acf_wtheta"} <= declared   # the names north_star fixes
    lib = ctypes.CDLL(os.path.join(ROOT, "paper_1208_3658_b200", "libacf.so"))
    for name in sorted(declared):
        assert hasattr(lib, name), "libacf.so does not export %s" % name
    from paper_1208_3658_b200.binding import EXPORTS
    assert set(EXPORTS) == declared


def test_no_gpu_means_error_not_fallback(acf):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(acf.AcfError) as ei:
        acf.acf_create(0)
    assert ei.value.code == -3
    # straight through the C ABI as well
    lib = acf.load_library()
    ctx = ctypes.c_void_p()
    assert lib.acf_create(ctypes.byref(ctx), 0, None) == -3
    assert not ctx.value
    assert b"no CUDA device" in lib.acf_last_error(None)


def test_binding_constants_match_header(acf):
    """Every enumerator and #define of include/acf.h that the binding repeats has the header's value."""
    header = open(os.path.join(ROOT, "include", "acf.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    values = {m.group(1): int(m.group(2)) for m in re.finditer(r"\b(ACF_[A-Z0-9_]+)\s*=\s*(-?\d+)", header)}
    values.update({m.group(1): int(m.group(2)) for m in re.finditer(r"#define\s+(ACF_[A-Z0-9_]+)\s+\(?(-?\d+)\)?", header)})
    assert {"ACF_OPT_KERNEL", "ACF_KERNEL_WINDOW", "ACF_EST_HAMILTON", "ACF_BINS_LOG10", "ACF_OPT_BULK", "ACF_MAX_BINS"} <= set(values)
    import paper_1208_3658_b200.binding as B
    checked = 0
    for name, val in values.items():
        if hasattr(B, name):
            assert getattr(B, name) == val, name
            checked += 1
    assert checked >= 20
    # the statistics structure: same fields, same order as the header
    fields = re.search(r"typedef struct acf_stats \{(.*?)\} acf_stats;", header, flags=re.S).group(1)
    names = re.findall(r"(?:uint64_t|double)\s+(\w+);", fields)
    assert names == [f for f, _ in B.acf_stats._fields_]


def test_radec_to_xyz_matches_oracle_bitwise(acf, oracle):
    ra, dec = full_sky(50000, 77)
    assert acf.acf_radec_to_xyz(ra, dec).tobytes() == oracle.radec_to_xyz(ra, dec).tobytes()
    rows = read_golden("radec_unit_vectors.txt")
    xyz = acf.acf_radec_to_xyz([float(r[0]) for r in rows], [float(r[1]) for r in rows]).reshape(3, -1).T
    want = np.array([[float(v) for v in r[2:5]] for r in rows])
    assert np.max(np.abs(xyz - want)) < 3e-16


def test_wtheta_golden_and_oracle(acf, oracle):
    for r in read_golden("wtheta_examples.txt"):
        n_d, n_r, dd, dr, rr = (int(v) for v in r[:5])
        w = acf.acf_wtheta([dd], [dr], [rr], n_d, n_r)[0]
        assert math.isnan(w) if r[5] == "nan" else abs(w - float(r[5])) < 1e-15
    rng = np.random.default_rng(3)
    dd, dr, rr = (rng.integers(0, 10 ** 9, size=40).astype(np.uint64) for _ in range(3))
    rr[5] = 0
    a = acf.acf_wtheta(dd, dr, rr, 123456, 234567)
    b = oracle.wtheta(dd, dr, rr, 123456, 234567)
    np.testing.assert_allclose(a, b, rtol=0, atol=1e-10, equal_nan=True)
    wd = rng.lognormal(0, 0.3, 1000).astype(np.float32)
    wr = rng.lognormal(0, 0.3, 1500).astype(np.float32)
    x, y, z = (rng.uniform(1, 1e5, size=40) for _ in range(3))
    np.testing.assert_allclose(acf.acf_wtheta_weighted(x, y, z, wd, wr), oracle.wtheta_weighted(x, y, z, wd, wr),
                               rtol=0, atol=1e-10)


def test_wtheta_weighted_golden_non_unit_weights(acf):
    # the same hand-computed fixture that pins the oracle's weighted estimator (sum w^2 != sum w != n)
    n = 0
    for r in read_golden("wtheta_weighted_examples.txt"):
        n_d = int(r[0])
        w_d = np.array([float(v) for v in r[1:1 + n_d]], dtype=np.float32)
        n_r = int(r[1 + n_d])
        w_r = np.array([float(v) for v in r[2 + n_d:2 + n_d + n_r]], dtype=np.float32)
        wdd, wdr, wrr = (float(v) for v in r[2 + n_d + n_r:5 + n_d + n_r])
        want = r[5 + n_d + n_r]
        got = acf.acf_wtheta_weighted([wdd], [wdr], [wrr], w_d, w_r)[0]
        assert math.isnan(got) if want == "nan" else abs(got - float(want)) < 1e-15, (r, got)
        n += 1
    assert n >= 6


def test_estimators_and_bin_presets_against_golden_and_oracle(acf, oracle):
    # PAPER.md:65 (other estimators) and PAPER.md:103 (bin presets): pure host entry points
    for r in read_golden("estimator_examples.txt"):
        n_d, n_r, dd, dr, rr = (int(v) for v in r[:5])
        for kind in range(4):
            w = acf.acf_estimator(kind, [dd], [dr], [rr], n_d, n_r)[0]
            want = float("nan") if r[5 + kind] == "nan" else float(r[5 + kind])
            assert (math.isnan(w) and math.isnan(want)) or abs(w - want) < 1e-15, (r, kind, w)
    rng = np.random.default_rng(4)
    dd, dr, rr = (rng.integers(0, 10 ** 9, size=50).astype(np.uint64) for _ in range(3))
    rr[5] = 0
    dr[7] = 0
    for kind in range(4):
        np.testing.assert_allclose(acf.acf_estimator(kind, dd, dr, rr, 123456, 234567), oracle.estimator(kind, dd, dr, rr, 123456, 234567),
                                   rtol=0, atol=1e-10, equal_nan=True)
    assert acf.acf_estimator(0, dd, dr, rr, 123456, 234567).tobytes() == acf.acf_wtheta(dd, dr, rr, 123456, 234567).tobytes()
    for mode, lo, hi, nb in ((acf.ACF_BINS_EVEN, 0.0, 120.0, 254), (acf.ACF_BINS_LOG, 1 / 60, 180.0, 40), (acf.ACF_BINS_LOG10, 0.1 / 60, 3.0, 30)):
        theta = acf.acf_theta_edges(mode, lo, hi, nb)
        assert theta.tobytes() == oracle.theta_edges(mode, lo, hi, nb).tobytes()    # same libm, same operations
        assert acf.acf_cos_edges(theta).tobytes() == oracle.cos_edges(theta).tobytes()
        e = acf.acf_cos_edges(theta)
        assert np.all(np.diff(e) < 0) and (hi < 180.0 or e[-1] == -1.0) and (lo > 0.0 or e[0] == 1.0)
    for r in read_golden("bin_presets.txt"):
        if r[0] != "cos":
            mode = {"even": acf.ACF_BINS_EVEN, "log": acf.ACF_BINS_LOG, "log10": acf.ACF_BINS_LOG10}[r[0]]
            np.testing.assert_allclose(acf.acf_theta_edges(mode, float(r[1]), float(r[2]), int(r[3])), [float(v) for v in r[4:]], rtol=4e-16)
    lib = acf.load_library()
    buf = (ctypes.c_double * 8)()
    assert lib.acf_theta_edges(acf.ACF_BINS_LOG, 0.0, 10.0, 4, buf) == -1      # log bins from 0
    assert lib.acf_theta_edges(acf.ACF_BINS_EVEN, 5.0, 5.0, 4, buf) == -1      # empty range
    assert lib.acf_theta_edges(7, 1.0, 5.0, 4, buf) == -1                      # unknown preset
    assert lib.acf_estimator(9, buf, buf, buf, 1, 1, 1, buf) == -1


def test_host_argument_errors(acf):
    lib = acf.load_library()
    assert lib.acf_wtheta(None, None, None, 1, 1, 3, None) == -1
    assert lib.acf_radec_to_xyz(None, None, 5, None) == -1
    assert lib.acf_radec_to_xyz(None, None, 0, None) == 0
    assert lib.acf_set_option(None, 1, 0) == -1
    assert lib.acf_get_stats(None, None) == -1
    lib.acf_destroy(None)   # no-op
