// acf_host.cpp -- the pure-host entry points of libacf (no CUDA): canonical unit vectors and
// the w(theta) estimator.  Compiled by g++ with -ffp-contract=off and no fast-math, so that
// acf_radec_to_xyz is exactly "one rounded multiply per product around glibc sin/cos"
// (include/acf.h; Appendix A, Eq. 2).
#include <cmath>
#include <cstddef>
#include <cstdint>
#include <limits>
#include <thread>
#include <vector>

#include "acf.h"

namespace {
// pi/180 rounded to double; degrees -> radians is a single multiply by this constant.
constexpr double kDegToRad = 0.017453292519943295;
}  // namespace

extern "C" int acf_radec_to_xyz(const double *ra_deg, const double *dec_deg, size_t n, double *xyz_host)
{
    if (n == 0) return ACF_OK;
    if (!ra_deg || !dec_deg || !xyz_host) return ACF_EINVAL;
    double *x = xyz_host, *y = xyz_host + n, *z = xyz_host + 2 * n;
    auto range = [=](size_t lo, size_t hi) {
        for (size_t i = lo; i < hi; ++i) {
            const double alpha = ra_deg[i] * kDegToRad;
            const double delta = dec_deg[i] * kDegToRad;
            const double cos_delta = std::cos(delta);
            x[i] = cos_delta * std::cos(alpha);
            y[i] = cos_delta * std::sin(alpha);
            z[i] = std::sin(delta);
        }
    };
    // every point is independent, so splitting the index range over threads changes no bit of the result
    unsigned n_thr = std::thread::hardware_concurrency();
    if (n_thr > 16) n_thr = 16;
    if (n < (size_t(1) << 16) || n_thr < 2) {
        range(0, n);
        return ACF_OK;
    }
    std::vector<std::thread> pool;
    try {
        for (unsigned t = 1; t < n_thr; ++t) pool.emplace_back(range, n * t / n_thr, n * (t + 1) / n_thr);
    } catch (...) {
        // no more threads to be had: the caller's thread does what is left
        const size_t done = pool.size() + 1;
        range(n * done / n_thr, n);
    }
    range(0, n / n_thr);
    for (auto &th : pool) th.join();
    return ACF_OK;
}

// Eq. 2 with pair-normalised terms (reading R2).
static inline double landy_szalay(double dd, double dr, double rr, double ndd, double ndr, double nrr)
{
    if (!(rr > 0.0) || !(ndd > 0.0) || !(ndr > 0.0) || !(nrr > 0.0))
        return std::numeric_limits<double>::quiet_NaN();
    const double fdd = dd / ndd, fdr = dr / ndr, frr = rr / nrr;
    return (fdd - 2.0 * fdr + frr) / frr;
}

extern "C" int acf_wtheta(const uint64_t *dd, const uint64_t *dr, const uint64_t *rr, uint64_t n_d,
                          uint64_t n_r, int nbins, double *w_host)
{
    if (!dd || !dr || !rr || !w_host || nbins < 1) return ACF_EINVAL;
    const double nd = (double)n_d, nr = (double)n_r;
    const double ndd = nd * (nd - 1.0) / 2.0, ndr = nd * nr, nrr = nr * (nr - 1.0) / 2.0;
    for (int k = 0; k < nbins; ++k)
        w_host[k] = landy_szalay((double)dd[k], (double)dr[k], (double)rr[k], ndd, ndr, nrr);
    return ACF_OK;
}

extern "C" int acf_wtheta_weighted(const double *wdd, const double *wdr, const double *wrr, const float *w_d,
                                   size_t n_d, const float *w_r, size_t n_r, int nbins, double *w_host)
{
    if (!wdd || !wdr || !wrr || !w_host || nbins < 1) return ACF_EINVAL;
    if ((n_d && !w_d) || (n_r && !w_r)) return ACF_EINVAL;
    long double sd = 0, sd2 = 0, sr = 0, sr2 = 0;
    for (size_t i = 0; i < n_d; ++i) {
        sd += w_d[i];
        sd2 += (long double)w_d[i] * w_d[i];
    }
    for (size_t i = 0; i < n_r; ++i) {
        sr += w_r[i];
        sr2 += (long double)w_r[i] * w_r[i];
    }
    const double ndd = (double)((sd * sd - sd2) / 2), ndr = (double)(sd * sr),
                 nrr = (double)((sr * sr - sr2) / 2);
    for (int k = 0; k < nbins; ++k) w_host[k] = landy_szalay(wdd[k], wdr[k], wrr[k], ndd, ndr, nrr);
    return ACF_OK;
}

// other estimators on the same pair-normalised counts.
extern "C" int acf_estimator(int kind, const uint64_t *dd, const uint64_t *dr, const uint64_t *rr, uint64_t n_d,
                             uint64_t n_r, int nbins, double *w_host)
{
    if (!dd || !dr || !rr || !w_host || nbins < 1) return ACF_EINVAL;
    if (kind < ACF_EST_LANDY_SZALAY || kind > ACF_EST_HAMILTON) return ACF_EINVAL;
    const double nan = std::numeric_limits<double>::quiet_NaN();
    const double nd = (double)n_d, nr = (double)n_r;
    const double ndd = nd * (nd - 1.0) / 2.0, ndr = nd * nr, nrr = nr * (nr - 1.0) / 2.0;
    for (int k = 0; k < nbins; ++k) {
        if (kind == ACF_EST_LANDY_SZALAY) {
            w_host[k] = landy_szalay((double)dd[k], (double)dr[k], (double)rr[k], ndd, ndr, nrr);
            continue;
        }
        if (!(ndd > 0.0) || !(ndr > 0.0) || !(nrr > 0.0)) {
            w_host[k] = nan;
            continue;
        }
        const double fdd = (double)dd[k] / ndd, fdr = (double)dr[k] / ndr, frr = (double)rr[k] / nrr;
        if (kind == ACF_EST_NATURAL) w_host[k] = frr > 0.0 ? fdd / frr - 1.0 : nan;
        else if (kind == ACF_EST_DAVIS_PEEBLES) w_host[k] = fdr > 0.0 ? fdd / fdr - 1.0 : nan;
        else w_host[k] = fdr > 0.0 ? fdd * frr / (fdr * fdr) - 1.0 : nan;
    }
    return ACF_OK;
}

// the bin presets.
extern "C" int acf_theta_edges(int mode, double lo_deg, double hi_deg, int nbins, double *theta_deg_host)
{
    if (!theta_deg_host || nbins < 1 || nbins > ACF_MAX_BINS) return ACF_EINVAL;
    if (!(lo_deg >= 0.0) || !(hi_deg > lo_deg) || !(hi_deg <= 180.0)) return ACF_EINVAL;
    if (mode == ACF_BINS_EVEN) {
        for (int k = 0; k <= nbins; ++k) theta_deg_host[k] = lo_deg + (hi_deg - lo_deg) * ((double)k / (double)nbins);
    } else if (mode == ACF_BINS_LOG || mode == ACF_BINS_LOG10) {
        if (!(lo_deg > 0.0)) return ACF_EINVAL;
        const double ratio = hi_deg / lo_deg;
        for (int k = 0; k <= nbins; ++k) theta_deg_host[k] = lo_deg * std::pow(ratio, (double)k / (double)nbins);
    } else {
        return ACF_EINVAL;
    }
    theta_deg_host[0] = lo_deg;
    theta_deg_host[nbins] = hi_deg;
    for (int k = 0; k < nbins; ++k)
        if (!(theta_deg_host[k + 1] > theta_deg_host[k])) return ACF_EINVAL;  // bins too fine for doubles
    return ACF_OK;
}

extern "C" int acf_cos_edges(const double *theta_deg, int n_edges, double *cos_edges_host)
{
    if (!theta_deg || !cos_edges_host || n_edges < 2) return ACF_EINVAL;
    for (int k = 0; k < n_edges; ++k) {
        const double t = theta_deg[k];
        if (!(t >= 0.0) || !(t <= 180.0) || (k > 0 && !(t > theta_deg[k - 1]))) return ACF_EINVAL;
        cos_edges_host[k] = t == 0.0 ? 1.0 : (t == 180.0 ? -1.0 : std::cos(t * kDegToRad));
    }
    for (int k = 1; k < n_edges; ++k)
        if (!(cos_edges_host[k] < cos_edges_host[k - 1])) return ACF_EINVAL;  // edges closer than a double resolves
    return ACF_OK;
}
