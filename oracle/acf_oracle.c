/*
 * acf_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, double-precision CPU oracle for the angular pair-count histogram
 * (DD, DR, RR) and the w(theta) estimator of arXiv 1208.3658 (Bard, Bellis,
 * Allen, Yepremyan, Kratochvil, "Cosmological calculations on the GPU"), sect. 2.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call this file.  It shares no code, header,
 * table or constant with paper_1208_3658_b200/csrc (the CUDA path) and the CUDA
 * path never calls it.
 *
 * What it computes (the method is an exact count -- PAPER.md:72 "the exact
 * calculation ... for all angular scales" -- so the oracle is the definition
 * written out, one pair at a time):
 *
 *   O1  canonical unit vector of (RA, Dec) in degrees            PAPER.md:207-219 (App. A; C = cos theta, :215)
 *   O2  pair cosine c = fma(xi,xj, fma(yi,yj, zi*zj)), clamped   PAPER.md:215 (C term = u_i . u_j)
 *   O3  pairs outside the binned range are dropped
 *   O4  bin k : e[k+1] < c <= e[k]  (theta_k <= theta < theta_k+1, last bin closed)
 *   O5  counts[k] += 1 ; weighted: wsum[k] += (double)wi*(double)wj
 *   O6  auto: unordered pairs i<j, n(n-1)/2 of them; cross: all n_a*n_b
 *   O7  Landy-Szalay  w = (DD - 2DR + RR)/RR on pair-normalised counts    PAPER.md:65-68 (Eq. 2)
 *   O8  theta-domain cross-check with the App. A trigonometric formula
 *
 * Readings of the paper where it is silent (inclusive edges, clamping, Eq. 2
 * normalisation, atan2, weights) are the ones listed in DESIGN.md "Readings".
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): regular polyhedra and equator
 * rings with hand-counted separations, edge inclusivity at c == e_k +- 1 ulp,
 * sum(counts) = n(n-1)/2 or n_a*n_b, swap symmetry, cross(a,a) = 2 auto(a) + n,
 * row-block additivity, bin merging, O8 vs O1-O4, closed-form expected counts on
 * the uniform sphere, w(theta) ~ 0 on unclustered data, Neyman-Scott closed form,
 * dyadic-weight exact sums.  No function here is "parity unpinned".
 *
 * Build: gcc -O2 -mfma -ffp-contract=off -fopenmp -shared -fPIC (see oracle.py).
 * -ffp-contract=off + explicit fma() pin the arithmetic of O2: the compiler may
 * neither fuse nor un-fuse anything.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_EINVAL (-1)
#define ORACLE_ENOMEM (-2)

/* pi/180 as the nearest double; one multiply converts degrees to radians (O1). */
static const double DEG2RAD = 0.017453292519943295;
static const double RAD2DEG = 57.29577951308232;

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* O1 -- PAPER.md:207-219.  xyz is SoA: x[0..n) | y[0..n) | z[0..n).
 * x = cos(dec) cos(ra), y = cos(dec) sin(ra), z = sin(dec); the dot product of two
 * such vectors is the paper's C = sin d1 sin d2 + cos d1 cos d2 cos(a2 - a1). */
int oracle_radec_to_xyz(const double *ra_deg, const double *dec_deg, size_t n, double *xyz)
{
    if ((!ra_deg || !dec_deg || !xyz) && n) return ORACLE_EINVAL;
    double *x = xyz, *y = xyz + n, *z = xyz + 2 * n;
    for (size_t i = 0; i < n; ++i) {
        double a = ra_deg[i] * DEG2RAD;
        double d = dec_deg[i] * DEG2RAD;
        double cd = cos(d);
        x[i] = cd * cos(a);
        y[i] = cd * sin(a);
        z[i] = sin(d);
    }
    return ORACLE_OK;
}

/* edges: nbins+1 doubles, strictly descending, inside [-1, 1]. */
static int edges_ok(const double *e, int nbins)
{
    if (!e || nbins < 1) return 0;
    for (int m = 0; m <= nbins; ++m) {
        if (!(e[m] >= -1.0 && e[m] <= 1.0)) return 0;
        if (m && !(e[m] < e[m - 1])) return 0;
    }
    return 1;
}

/* O2: the pair cosine.  IEEE round-to-nearest, two fused multiply-adds around one
 * rounded product, then the clamp to [-1, 1] (reading R10). */
static inline double pair_cos(double xi, double yi, double zi, double xj, double yj, double zj)
{
    double c = fma(xi, xj, fma(yi, yj, zi * zj));
    if (c > 1.0) c = 1.0;
    if (c < -1.0) c = -1.0;
    return c;
}

/* O3 + O4: returns the bin of c, or -1 if the pair is dropped.
 * k = #{ m in [1, nbins-1] : c <= e[m] }. */
static inline int bin_of(double c, const double *e, int nbins)
{
    if (c > e[0] || c < e[nbins]) return -1;
    int k = 0;
    for (int m = 1; m < nbins; ++m) k += (c <= e[m]);
    return k;
}

/*
 * Rows [i0, i1) of catalogue A against catalogue B.
 *   is_auto = 0 : every j in [0, n_b)            (O6 cross, "n n_r calculations")
 *   is_auto = 1 : every j in (i, n_b), B == A    (O6 auto,  PAPER.md:70 "n(n-1)/2 calculations")
 * w_a / w_b may be NULL (then wsums must be NULL too).  counts and wsums are
 * overwritten.  Weighted sums: per row in long double, rows combined in long
 * double (reading R15), so the oracle sits on the accurate side of the tolerance.
 */
int oracle_pair_count_rows(const double *xyz_a, const float *w_a, size_t n_a, size_t i0, size_t i1,
                           const double *xyz_b, const float *w_b, size_t n_b,
                           const double *cos_edges, int nbins, int is_auto,
                           uint64_t *counts, double *wsums)
{
    if (!counts || !edges_ok(cos_edges, nbins)) return ORACLE_EINVAL;
    if ((n_a && !xyz_a) || (n_b && !xyz_b)) return ORACLE_EINVAL;
    if (i0 > i1 || i1 > n_a) return ORACLE_EINVAL;
    if (is_auto && (xyz_a != xyz_b || n_a != n_b)) return ORACLE_EINVAL;
    int weighted = (wsums != NULL);
    if (weighted && (!w_a || !w_b)) return ORACLE_EINVAL;

    const double *xa = xyz_a, *ya = xyz_a + n_a, *za = xyz_a + 2 * n_a;
    const double *xb = xyz_b, *yb = xyz_b + n_b, *zb = xyz_b + 2 * n_b;

    memset(counts, 0, sizeof(uint64_t) * (size_t)nbins);
    long double *wtot = (long double *)calloc((size_t)nbins, sizeof(long double));
    if (!wtot) return ORACLE_ENOMEM;
    int failed = 0;

#pragma omp parallel
    {
        uint64_t *cnt = (uint64_t *)calloc((size_t)nbins, sizeof(uint64_t));
        long double *wth = (long double *)calloc((size_t)nbins, sizeof(long double));
        long double *wrow = (long double *)calloc((size_t)nbins, sizeof(long double));
        if (!cnt || !wth || !wrow) {
#pragma omp atomic write
            failed = 1;
        } else {
#pragma omp for schedule(dynamic, 16)
            for (long long ii = (long long)i0; ii < (long long)i1; ++ii) {
                size_t i = (size_t)ii;
                double xi = xa[i], yi = ya[i], zi = za[i];
                double wi = weighted ? (double)w_a[i] : 0.0;
                size_t j0 = is_auto ? i + 1 : 0;
                if (weighted) memset(wrow, 0, sizeof(long double) * (size_t)nbins);
                for (size_t j = j0; j < n_b; ++j) {
                    double c = pair_cos(xi, yi, zi, xb[j], yb[j], zb[j]);
                    int k = bin_of(c, cos_edges, nbins);
                    if (k < 0) continue;
                    cnt[k] += 1;
                    if (weighted) wrow[k] += (long double)(wi * (double)w_b[j]); /* exact product: 24+24 bits */
                }
                if (weighted)
                    for (int k = 0; k < nbins; ++k) wth[k] += wrow[k];
            }
#pragma omp critical
            {
                for (int k = 0; k < nbins; ++k) {
                    counts[k] += cnt[k];
                    wtot[k] += wth[k];
                }
            }
        }
        free(cnt);
        free(wth);
        free(wrow);
    }
    if (weighted)
        for (int k = 0; k < nbins; ++k) wsums[k] = (double)wtot[k];
    free(wtot);
    return failed ? ORACLE_ENOMEM : ORACLE_OK;
}

/* DD / RR (is_auto = 1) or DR (is_auto = 0): PAPER.md:65-70. */
int oracle_pair_count(const double *xyz_a, size_t n_a, const double *xyz_b, size_t n_b,
                      const double *cos_edges, int nbins, int is_auto, uint64_t *counts)
{
    return oracle_pair_count_rows(xyz_a, NULL, n_a, 0, n_a, xyz_b, NULL, n_b, cos_edges, nbins, is_auto,
                                  counts, NULL);
}

/* Same with pair weight w_i * w_j (reading R11; not in the paper, BASELINE config 4). */
int oracle_pair_count_weighted(const double *xyz_a, const float *w_a, size_t n_a, const double *xyz_b,
                               const float *w_b, size_t n_b, const double *cos_edges, int nbins,
                               int is_auto, uint64_t *counts, double *wsums)
{
    if (!wsums) return ORACLE_EINVAL;
    return oracle_pair_count_rows(xyz_a, w_a, n_a, 0, n_a, xyz_b, w_b, n_b, cos_edges, nbins, is_auto,
                                  counts, wsums);
}

/*
 * Dec-window variant for small theta_max: identical O1-O6 pair by pair, but row i
 * only visits the j with |dec_j - dec_i| <= theta_max + margin.  theta >= |delta
 * dec| on the sphere, so every skipped pair has c < e[nbins] and would have been
 * dropped by O3 anyway: the visited set is a superset of the counted set.  Used
 * only where the plain loop is out of reach (BASELINE configs 3 and 5); tests
 * check it equals oracle_pair_count exactly wherever both can run.
 */
typedef struct {
    double dec;
    size_t idx;
} dec_key;

static int dec_key_cmp(const void *pa, const void *pb)
{
    const dec_key *a = (const dec_key *)pa, *b = (const dec_key *)pb;
    if (a->dec < b->dec) return -1;
    if (a->dec > b->dec) return 1;
    return (a->idx > b->idx) - (a->idx < b->idx);
}

int oracle_pair_count_decwindow(const double *xyz_a, const double *dec_a_deg, size_t n_a,
                                const double *xyz_b, const double *dec_b_deg, size_t n_b,
                                const double *cos_edges, int nbins, int is_auto, uint64_t *counts)
{
    if (!counts || !edges_ok(cos_edges, nbins)) return ORACLE_EINVAL;
    if ((n_a && (!xyz_a || !dec_a_deg)) || (n_b && (!xyz_b || !dec_b_deg))) return ORACLE_EINVAL;
    if (is_auto && (xyz_a != xyz_b || n_a != n_b)) return ORACLE_EINVAL;

    /* half-width of the window in degrees: theta_max plus a margin that dwarfs
     * every rounding in O1/O2 (1e-6 deg moves c by >= 3e-12 at theta_max >= 0.01 deg). */
    double width = acos(cos_edges[nbins]) * RAD2DEG + 1e-6;

    memset(counts, 0, sizeof(uint64_t) * (size_t)nbins);
    dec_key *keys = (dec_key *)malloc(sizeof(dec_key) * (n_b ? n_b : 1));
    if (!keys) return ORACLE_ENOMEM;
    for (size_t j = 0; j < n_b; ++j) {
        keys[j].dec = dec_b_deg[j];
        keys[j].idx = j;
    }
    qsort(keys, n_b, sizeof(dec_key), dec_key_cmp);

    const double *xa = xyz_a, *ya = xyz_a + n_a, *za = xyz_a + 2 * n_a;
    const double *xb = xyz_b, *yb = xyz_b + n_b, *zb = xyz_b + 2 * n_b;
    int failed = 0;

#pragma omp parallel
    {
        uint64_t *cnt = (uint64_t *)calloc((size_t)nbins, sizeof(uint64_t));
        if (!cnt) {
#pragma omp atomic write
            failed = 1;
        } else {
#pragma omp for schedule(dynamic, 64)
            for (long long ii = 0; ii < (long long)n_a; ++ii) {
                size_t i = (size_t)ii;
                double lo = dec_a_deg[i] - width, hi = dec_a_deg[i] + width;
                /* first key with dec >= lo */
                size_t l = 0, r = n_b;
                while (l < r) {
                    size_t m = l + (r - l) / 2;
                    if (keys[m].dec < lo) l = m + 1; else r = m;
                }
                double xi = xa[i], yi = ya[i], zi = za[i];
                for (size_t s = l; s < n_b && keys[s].dec <= hi; ++s) {
                    size_t j = keys[s].idx;
                    if (is_auto && j <= i) continue; /* O6: unordered pairs i<j once */
                    double c = pair_cos(xi, yi, zi, xb[j], yb[j], zb[j]);
                    int k = bin_of(c, cos_edges, nbins);
                    if (k >= 0) cnt[k] += 1;
                }
            }
#pragma omp critical
            for (int k = 0; k < nbins; ++k) counts[k] += cnt[k];
        }
        free(cnt);
    }
    free(keys);
    return failed ? ORACLE_ENOMEM : ORACLE_OK;
}

/*
 * Dec + RA window variant, for a small theta_max on a wide footprint (BASELINE configs 3 and 5: the Dec
 * window alone still visits 14-22 % of the pair matrix, 1.8e13 pairs on config 5).  Identical O1-O6 pair
 * by pair; row i visits only the j whose Dec lies in the band of row i or a neighbouring band (bands of
 * height W_dec = theta_max + margin) and whose RA lies within W_ra(i) of ra_i (modulo 360).  Both
 * windows are supersets of the counted set:
 *   theta >= |d2 - d1|                                             (as in oracle_pair_count_decwindow)
 *   hav(theta) = hav(d2 - d1) + cos d1 cos d2 hav(a2 - a1),  hav(x) = sin^2(x/2)   (haversine formula,
 *     equivalent to the C term of PAPER.md:215)   =>   sin^2((a2 - a1)/2) <= hav(theta) / (cos d1 cos d2);
 *   a visited j has |d2| <= |d1| + 2 W_dec (own or neighbouring band), so cos d2 >= cos(min(90 deg,
 *   |d1| + 2 W_dec)) =: cmin, and a pair with theta <= theta_max has
 *     |a2 - a1| <= 2 asin( sqrt( hav(theta_max) / (cos d1 * cmin) ) ) =: W_ra(i)
 *   (no RA bound at all, W_ra = 180 deg, when that ratio reaches 1: rows near a pole).
 * Every skipped pair therefore has theta > theta_max, i.e. c < e[nbins], and O3 would have dropped it.
 * Tests check it equals oracle_pair_count exactly wherever both can run (patches, RA wrap-around,
 * points at the poles, theta_max up to 180 deg).  Unweighted.  Rows [i0, i1) of A.
 */
typedef struct {
    int band;
    double ra; /* in [0, 360) */
    size_t idx;
} cell_key;

static int cell_key_cmp(const void *pa, const void *pb)
{
    const cell_key *a = (const cell_key *)pa, *b = (const cell_key *)pb;
    if (a->band != b->band) return a->band < b->band ? -1 : 1;
    if (a->ra < b->ra) return -1;
    if (a->ra > b->ra) return 1;
    return (a->idx > b->idx) - (a->idx < b->idx);
}

static double wrap360(double ra)
{
    double r = fmod(ra, 360.0);
    if (r < 0.0) r += 360.0;
    if (r >= 360.0) r = 0.0;
    return r;
}

/* first key of [l, r) with ra >= v */
static size_t cell_lower(const cell_key *k, size_t l, size_t r, double v)
{
    while (l < r) {
        size_t m = l + (r - l) / 2;
        if (k[m].ra < v) l = m + 1; else r = m;
    }
    return l;
}

int oracle_pair_count_cellwindow(const double *xyz_a, const double *ra_a_deg, const double *dec_a_deg, size_t n_a,
                                 size_t i0, size_t i1, const double *xyz_b, const double *ra_b_deg,
                                 const double *dec_b_deg, size_t n_b, const double *cos_edges, int nbins,
                                 int is_auto, uint64_t *counts)
{
    if (!counts || !edges_ok(cos_edges, nbins)) return ORACLE_EINVAL;
    if ((n_a && (!xyz_a || !ra_a_deg || !dec_a_deg)) || (n_b && (!xyz_b || !ra_b_deg || !dec_b_deg))) return ORACLE_EINVAL;
    if (i0 > i1 || i1 > n_a) return ORACLE_EINVAL;
    if (is_auto && (xyz_a != xyz_b || n_a != n_b)) return ORACLE_EINVAL;

    const double theta_max = acos(cos_edges[nbins]);            /* radians */
    const double w_dec = theta_max * RAD2DEG + 1e-6;            /* degrees; the margin dwarfs every rounding here */
    const double hav_max = sin(0.5 * theta_max) * sin(0.5 * theta_max) * (1.0 + 1e-9);
    const int n_bands = (int)floor(180.0 / w_dec) + 1;
    memset(counts, 0, sizeof(uint64_t) * (size_t)nbins);

    cell_key *keys = (cell_key *)malloc(sizeof(cell_key) * (n_b ? n_b : 1));
    size_t *start = (size_t *)calloc((size_t)n_bands + 1, sizeof(size_t));
    if (!keys || !start) {
        free(keys);
        free(start);
        return ORACLE_ENOMEM;
    }
    for (size_t j = 0; j < n_b; ++j) {
        int band = (int)floor((dec_b_deg[j] + 90.0) / w_dec);
        if (band < 0) band = 0;
        if (band >= n_bands) band = n_bands - 1;
        keys[j].band = band;
        keys[j].ra = wrap360(ra_b_deg[j]);
        keys[j].idx = j;
        start[band + 1] += 1;
    }
    for (int b = 0; b < n_bands; ++b) start[b + 1] += start[b];
    qsort(keys, n_b, sizeof(cell_key), cell_key_cmp);

    const double *xa = xyz_a, *ya = xyz_a + n_a, *za = xyz_a + 2 * n_a;
    const double *xb = xyz_b, *yb = xyz_b + n_b, *zb = xyz_b + 2 * n_b;
    int failed = 0;

#pragma omp parallel
    {
        uint64_t *cnt = (uint64_t *)calloc((size_t)nbins, sizeof(uint64_t));
        if (!cnt) {
#pragma omp atomic write
            failed = 1;
        } else {
#pragma omp for schedule(dynamic, 64)
            for (long long ii = (long long)i0; ii < (long long)i1; ++ii) {
                size_t i = (size_t)ii;
                double di = dec_a_deg[i], ai = wrap360(ra_a_deg[i]);
                int band = (int)floor((di + 90.0) / w_dec);
                if (band < 0) band = 0;
                if (band >= n_bands) band = n_bands - 1;
                /* RA half-width of row i, degrees */
                double far = fabs(di) + 2.0 * w_dec;
                double cmin = far >= 90.0 ? 0.0 : cos(far * DEG2RAD);
                double den = cos(di * DEG2RAD) * cmin;
                double w_ra = 180.0;
                if (den > 0.0 && hav_max < den) w_ra = 2.0 * asin(sqrt(hav_max / den)) * RAD2DEG + 1e-6;
                double xi = xa[i], yi = ya[i], zi = za[i];
                for (int b = band - 1; b <= band + 1; ++b) {
                    if (b < 0 || b >= n_bands) continue;
                    size_t l = start[b], r = start[b + 1];
                    /* up to two RA runs of the band: [lo, hi], wrapped at 0 / 360 */
                    size_t run_l[2], run_r[2];
                    int n_runs = 1;
                    if (w_ra >= 180.0) {
                        run_l[0] = l;
                        run_r[0] = r;
                    } else {
                        double lo = ai - w_ra, hi = ai + w_ra;
                        if (lo < 0.0) {
                            run_l[0] = l;
                            run_r[0] = cell_lower(keys, l, r, nextafter(hi, 1e300));
                            run_l[1] = cell_lower(keys, l, r, lo + 360.0);
                            run_r[1] = r;
                            n_runs = 2;
                        } else if (hi >= 360.0) {
                            run_l[0] = l;
                            run_r[0] = cell_lower(keys, l, r, nextafter(hi - 360.0, 1e300));
                            run_l[1] = cell_lower(keys, l, r, lo);
                            run_r[1] = r;
                            n_runs = 2;
                        } else {
                            run_l[0] = cell_lower(keys, l, r, lo);
                            run_r[0] = cell_lower(keys, l, r, nextafter(hi, 1e300));
                        }
                        /* two runs that meet or overlap (w_ra close to 180): visit nothing twice */
                        if (n_runs == 2 && run_l[1] < run_r[0]) run_l[1] = run_r[0];
                    }
                    for (int t = 0; t < n_runs; ++t)
                        for (size_t s = run_l[t]; s < run_r[t]; ++s) {
                            size_t j = keys[s].idx;
                            if (is_auto && j <= i) continue; /* O6: unordered pairs i<j once */
                            double c = pair_cos(xi, yi, zi, xb[j], yb[j], zb[j]);
                            int k = bin_of(c, cos_edges, nbins);
                            if (k >= 0) cnt[k] += 1;
                        }
                }
            }
#pragma omp critical
            for (int k = 0; k < nbins; ++k) counts[k] += cnt[k];
        }
        free(cnt);
    }
    free(keys);
    free(start);
    return failed ? ORACLE_ENOMEM : ORACLE_OK;
}

/*
 * O8 -- the paper's own separation formula, PAPER.md:207-219 (Appendix A), with
 * atan2 in place of arctan(./C) so that theta lands in [0, 180] deg (reading R6):
 *   da = a2 - a1
 *   A  = cos^2 d2 sin^2 da
 *   B  = cos d1 sin d2 - sin d1 cos d2 cos da
 *   C  = sin d1 sin d2 + cos d1 cos d2 cos da
 *   theta = (180/pi) atan2( sqrt(A + B^2), C )
 * Binned in the theta domain: theta_edges_deg ascending, theta_k <= theta <
 * theta_k+1, last bin closed above (the same inclusivity as O4).  Pairs whose
 * theta is within rel_tol (relative) of any edge are counted in *n_near and, up
 * to near_cap of them, listed as (i, j) in near_ij -- listed, not hidden.
 * Small inputs only: single thread, one pair at a time.
 */
int oracle_pair_count_theta(const double *ra_a, const double *dec_a, size_t n_a, const double *ra_b,
                            const double *dec_b, size_t n_b, const double *theta_edges_deg, int nbins,
                            int is_auto, double rel_tol, uint64_t *counts, uint64_t *n_near,
                            uint64_t *near_ij, size_t near_cap)
{
    if (!counts || !theta_edges_deg || nbins < 1 || !n_near) return ORACLE_EINVAL;
    for (int m = 1; m <= nbins; ++m)
        if (!(theta_edges_deg[m] > theta_edges_deg[m - 1])) return ORACLE_EINVAL;
    if (is_auto && (ra_a != ra_b || dec_a != dec_b || n_a != n_b)) return ORACLE_EINVAL;
    memset(counts, 0, sizeof(uint64_t) * (size_t)nbins);
    *n_near = 0;
    for (size_t i = 0; i < n_a; ++i) {
        double a1 = ra_a[i] * DEG2RAD, d1 = dec_a[i] * DEG2RAD;
        size_t j0 = is_auto ? i + 1 : 0;
        for (size_t j = j0; j < n_b; ++j) {
            double a2 = ra_b[j] * DEG2RAD, d2 = dec_b[j] * DEG2RAD;
            double da = a2 - a1;
            double A = cos(d2) * cos(d2) * sin(da) * sin(da);
            double B = cos(d1) * sin(d2) - sin(d1) * cos(d2) * cos(da);
            double C = sin(d1) * sin(d2) + cos(d1) * cos(d2) * cos(da);
            double theta = RAD2DEG * atan2(sqrt(A + B * B), C);
            for (int m = 0; m <= nbins; ++m) {
                double e = theta_edges_deg[m];
                if (fabs(theta - e) <= rel_tol * e) {
                    if (near_ij && *n_near < near_cap) {
                        near_ij[2 * (*n_near)] = i;
                        near_ij[2 * (*n_near) + 1] = j;
                    }
                    *n_near += 1;
                    break;
                }
            }
            if (theta < theta_edges_deg[0] || theta > theta_edges_deg[nbins]) continue;
            int k = 0;
            for (int m = 1; m < nbins; ++m) k += (theta >= theta_edges_deg[m]);
            counts[k] += 1;
        }
    }
    return ORACLE_OK;
}

/*
 * O7 -- PAPER.md:65-68, Eq. 2:  w = (DD - 2 DR + RR) / RR, each term divided by
 * its number of pairs (reading R2: with raw counts DR has about twice the pairs of
 * DD, and Eq. 2 would read -2 on unclustered data).
 *   dd = DD_k / (n_d (n_d - 1) / 2),  dr = DR_k / (n_d n_r),  rr = RR_k / (n_r (n_r - 1) / 2)
 * RR_k = 0  =>  NaN (reading R13).
 */
int oracle_wtheta(const uint64_t *dd, const uint64_t *dr, const uint64_t *rr, uint64_t n_d,
                  uint64_t n_r, int nbins, double *w)
{
    if (!dd || !dr || !rr || !w || nbins < 1) return ORACLE_EINVAL;
    double ndd = (double)n_d * ((double)n_d - 1.0) / 2.0;
    double ndr = (double)n_d * (double)n_r;
    double nrr = (double)n_r * ((double)n_r - 1.0) / 2.0;
    for (int k = 0; k < nbins; ++k) {
        if (rr[k] == 0 || nrr <= 0.0 || ndd <= 0.0 || ndr <= 0.0) {
            w[k] = NAN;
            continue;
        }
        double fdd = (double)dd[k] / ndd;
        double fdr = (double)dr[k] / ndr;
        double frr = (double)rr[k] / nrr;
        w[k] = (fdd - 2.0 * fdr + frr) / frr;
    }
    return ORACLE_OK;
}

/* Weighted O7: the same estimator on weighted sums, with the weighted pair
 * totals as normalisers: auto ((sum w)^2 - sum w^2)/2, cross (sum w_d)(sum w_r). */
int oracle_wtheta_weighted(const double *dd, const double *dr, const double *rr, const float *w_d,
                           size_t n_d, const float *w_r, size_t n_r, int nbins, double *w)
{
    if (!dd || !dr || !rr || !w || nbins < 1 || (n_d && !w_d) || (n_r && !w_r)) return ORACLE_EINVAL;
    long double sd = 0, sd2 = 0, sr = 0, sr2 = 0;
    for (size_t i = 0; i < n_d; ++i) {
        sd += (long double)w_d[i];
        sd2 += (long double)w_d[i] * (long double)w_d[i];
    }
    for (size_t i = 0; i < n_r; ++i) {
        sr += (long double)w_r[i];
        sr2 += (long double)w_r[i] * (long double)w_r[i];
    }
    double ndd = (double)((sd * sd - sd2) / 2);
    double ndr = (double)(sd * sr);
    double nrr = (double)((sr * sr - sr2) / 2);
    for (int k = 0; k < nbins; ++k) {
        if (!(rr[k] > 0.0) || !(nrr > 0.0) || !(ndd > 0.0) || !(ndr > 0.0)) {
            w[k] = NAN;
            continue;
        }
        double fdd = dd[k] / ndd, fdr = dr[k] / ndr, frr = rr[k] / nrr;
        w[k] = (fdd - 2.0 * fdr + frr) / frr;
    }
    return ORACLE_OK;
}

/*
 * "allows the user to easily experiment with other estimators".  The usual ones on the
 * pair-normalised counts dd, dr, rr of O7 (kind 0 is O7 itself):
 *   1 natural (Peebles-Hauser)  dd / rr - 1
 *   2 Davis-Peebles             dd / dr - 1
 *   3 Hamilton                  dd rr / dr^2 - 1
 * NaN where the denominator is zero.
 */
int oracle_estimator(int kind, const uint64_t *dd, const uint64_t *dr, const uint64_t *rr, uint64_t n_d,
                     uint64_t n_r, int nbins, double *w)
{
    if (kind == 0) return oracle_wtheta(dd, dr, rr, n_d, n_r, nbins, w);
    if (!dd || !dr || !rr || !w || nbins < 1 || kind < 0 || kind > 3) return ORACLE_EINVAL;
    double ndd = (double)n_d * ((double)n_d - 1.0) / 2.0;
    double ndr = (double)n_d * (double)n_r;
    double nrr = (double)n_r * ((double)n_r - 1.0) / 2.0;
    for (int k = 0; k < nbins; ++k) {
        w[k] = NAN;
        if (nrr <= 0.0 || ndd <= 0.0 || ndr <= 0.0) continue;
        double fdd = (double)dd[k] / ndd;
        double fdr = (double)dr[k] / ndr;
        double frr = (double)rr[k] / nrr;
        if (kind == 1 && rr[k] != 0) w[k] = fdd / frr - 1.0;
        if (kind == 2 && dr[k] != 0) w[k] = fdd / fdr - 1.0;
        if (kind == 3 && dr[k] != 0) w[k] = fdd * frr / (fdr * fdr) - 1.0;
    }
    return ORACLE_OK;
}

/*
 * bins between a low and a high limit, "evenly spaced, natural log or log base 10".
 * mode 0: theta_k = lo + (hi - lo) k / n;  mode 1, 2: theta_k = lo (hi / lo)^(k / n) (the two logarithms
 * give the same edges: reading R5).  The end edges are lo and hi exactly.
 */
int oracle_theta_edges(int mode, double lo, double hi, int nbins, double *theta)
{
    if (!theta || nbins < 1 || !(lo >= 0.0) || !(hi > lo) || !(hi <= 180.0)) return ORACLE_EINVAL;
    if (mode != 0 && !(lo > 0.0)) return ORACLE_EINVAL;
    if (mode < 0 || mode > 2) return ORACLE_EINVAL;
    for (int k = 0; k <= nbins; ++k) {
        double f = (double)k / (double)nbins;
        theta[k] = mode == 0 ? lo + (hi - lo) * f : lo * pow(hi / lo, f);
    }
    theta[0] = lo;
    theta[nbins] = hi;
    return ORACLE_OK;
}

/* Cosine edges of angle edges in degrees (reading R5): cos(theta pi/180), 1 and -1 exactly at 0 and 180. */
int oracle_cos_edges(const double *theta, int n, double *e)
{
    if (!theta || !e || n < 2) return ORACLE_EINVAL;
    for (int k = 0; k < n; ++k)
        e[k] = theta[k] == 0.0 ? 1.0 : (theta[k] == 180.0 ? -1.0 : cos(theta[k] * 0.017453292519943295));
    return ORACLE_OK;
}
