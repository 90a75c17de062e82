"""paper_1208_3658_b200 -- B200-native angular pair counts (DD, DR, RR) and w(theta).

The hot path of arXiv 1208.3658 sect. 2 as hand-written sm_100a CUDA kernels behind a C ABI
(include/acf.h -> libacf.so); this package is the thin ctypes binding over it.
"""
from .binding import (ACF_KERNEL_AUTO, ACF_KERNEL_FP64, ACF_KERNEL_TABLE, ACF_KERNEL_WINDOW, ACF_OPT_KERNEL, ACF_OPT_PRUNE, ACF_OPT_STATS, ACF_OPT_WINDOWS, ACF_OPT_BULK, AcfError,
                      acf_correlate_host, acf_create, acf_destroy, acf_get_stats, acf_last_error, acf_pair_count,
                      acf_pair_count_rows, acf_pair_count_weighted, acf_radec_to_xyz, acf_set_option,
                      acf_set_stream, acf_version, acf_wtheta, acf_estimator, acf_theta_edges, acf_cos_edges, acf_jackknife,
                      ACF_EST_LANDY_SZALAY, ACF_EST_NATURAL, ACF_EST_DAVIS_PEEBLES, ACF_EST_HAMILTON, ACF_BINS_EVEN, ACF_BINS_LOG, ACF_BINS_LOG10, acf_wtheta_weighted, counts_to_numpy, load_library,
                      acf_prepare, acf_prepare_rows, acf_prepare_again, acf_release, acf_pair_count_prepared, acf_random_ensemble, Catalog,
                      acf_pair_count_static, ACF_STATIC_MAX_POINTS)

__all__ = [
    "ACF_KERNEL_AUTO", "ACF_KERNEL_FP64", "ACF_KERNEL_TABLE", "ACF_KERNEL_WINDOW", "ACF_OPT_KERNEL", "ACF_OPT_PRUNE", "ACF_OPT_STATS", "ACF_OPT_WINDOWS", "ACF_OPT_BULK", "AcfError",
    "acf_correlate_host", "acf_create", "acf_destroy", "acf_get_stats", "acf_last_error", "acf_pair_count",
    "acf_pair_count_rows", "acf_pair_count_weighted", "acf_radec_to_xyz", "acf_set_option", "acf_set_stream",
    "acf_version", "acf_wtheta", "acf_estimator", "acf_theta_edges", "acf_cos_edges", "acf_jackknife", "ACF_EST_LANDY_SZALAY", "ACF_EST_NATURAL",
    "ACF_EST_DAVIS_PEEBLES", "ACF_EST_HAMILTON", "ACF_BINS_EVEN", "ACF_BINS_LOG", "ACF_BINS_LOG10", "acf_wtheta_weighted", "counts_to_numpy", "load_library",
    "acf_prepare", "acf_prepare_rows", "acf_prepare_again", "acf_release", "acf_pair_count_prepared", "acf_random_ensemble", "Catalog",
    "acf_pair_count_static", "ACF_STATIC_MAX_POINTS",
]
