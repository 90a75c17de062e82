/*
 * acf.h -- C ABI of libacf: angular pair-count histograms (DD, DR, RR) and the
 * w(theta) estimator of arXiv 1208.3658 (Bard et al., "Cosmological calculations on
 * the GPU", sect. 2), computed by hand-written sm_100a CUDA kernels on one B200.
 *
 * Citations are lines of the paper text with the section they fall in.
 *
 * WHAT IS COMPUTED (the definition every kernel must reproduce bit for bit):
 *   canonical vector  u = (cos d cos a, cos d sin a, sin d) of (RA a, Dec d)      PAPER.md:207-219 (App. A)
 *   pair cosine       c = fma(x_i, x_j, fma(y_i, y_j, z_i * z_j)) in IEEE double,
 *                     clamped to [-1, 1]; c is the C term of App. A = cos(theta)
 *   range             a pair with c > e[0] or c < e[nbins] is dropped
 *   bin               k such that e[k+1] < c <= e[k]; the last bin also takes
 *                     c == e[nbins]  (theta_k <= theta < theta_k+1 in angle)
 *   counts[k] += 1 ; weighted: wsums[k] += (double)w_i * (double)w_j
 *   pair set          is_auto: unordered pairs i < j, n(n-1)/2 of them;
 *                     cross: all n_a * n_b ordered pairs
 *   estimator         w = (DD - 2 DR + RR) / RR on pair-normalised counts          PAPER.md:65-68 (Eq. 2)
 * Counts are exact u64 integers under this double-precision definition whatever
 * the internal arithmetic (fp32 is used only where a pair is provably more than a
 * rounding bound away from every bin edge; every other pair is re-evaluated in
 * fp64).  Weighted sums are fp64 sums of exact products; their summation order is
 * unspecified (agreement with a long-double reference is ~1e-14 relative).
 *
 * CONVENTIONS
 *   - "HOST" / "DEVICE" says where a pointer must live.  The caller owns every
 *     buffer it passes; the library owns only the context and the scratch memory
 *     inside it (grown lazily, freed by acf_destroy).  No PyTorch types cross the ABI.
 *   - xyz arrays are structure-of-arrays doubles of length 3n: x[0..n) | y[0..n) | z[0..n).
 *   - cos_edges: HOST, nbins+1 doubles, strictly descending, all within [-1, 1]
 *     (cosines of ascending angle edges).  1 <= nbins <= ACF_MAX_BINS.
 *   - Device work is enqueued on the context's stream and is asynchronous unless
 *     stated; results in device buffers are valid after that stream is synchronised.
 *     (acf_pair_count* prepare their catalogues on the fly and wait on the host for the validation verdict; the
 *     counts on prepared handles never wait.)
 *   - A catalogue holds at most 2^31 - 1 points; the tile-level work list keeps one bit per tile of 1024 points
 *     of the second catalogue in 48 KB of shared memory, i.e. up to 4.0e8 points there (ACF_EINVAL beyond).
 *   - Every function returns ACF_OK (0) or a negative ACF_E* code, never throws,
 *     aborts or prints; acf_last_error() gives the message of the last failure on
 *     that context.  A context is not thread-safe: one caller at a time.
 *   - There is no CPU fallback: with no usable CUDA device acf_create fails.
 */
#ifndef ACF_H
#define ACF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ACF_OK 0
#define ACF_EINVAL (-1) /* bad argument: null pointer, bad edges, non-unit vectors, ... */
#define ACF_ENOMEM (-2) /* host or device allocation failed */
#define ACF_ECUDA (-3)  /* a CUDA runtime call or a kernel failed */

#define ACF_MAX_BINS 1024

typedef struct acf_ctx acf_ctx;         /* opaque; library-owned */
typedef struct acf_catalog acf_catalog; /* opaque; a catalogue prepared on the device (acf_prepare) */

/* Options for acf_set_option. */
enum {
    /* Which pair kernel runs.  ACF_KERNEL_AUTO (default) = the fast fp32-certify path: the window
     * kernel for every call (the table kernel only where the window kernel's shared memory does not
     * fit or its weights do not pack, see below); ACF_KERNEL_FP64 = the reference kernel that evaluates the definition
     * in double for every pair (slow; the arbiter the fast path defers to, kept callable for
     * debugging); ACF_KERNEL_TABLE = fast path, cell-table kernel (single-edge windows in registers,
     * everything else through a bin table and per-lane shared-memory histograms);
     * ACF_KERNEL_WINDOW = fast path, window kernel (every group of pairs classified in registers
     * against the few edges its bounding caps allow; unweighted groups that more than three edges can
     * separate, pair by pair through a cell table of the squared chord length; weights whose range
     * exceeds 2^13 are handed to the table kernel's per-pair path, whatever the choice).  All four give the same counts.  With very many
     * bins a kernel's shared-memory histograms may not fit: AUTO then takes the other fast kernel, an
     * explicit choice returns ACF_EINVAL. */
    ACF_OPT_KERNEL = 1,
    /* 1 (default): tile pairs -- and, inside the tile pairs that remain, pairs of groups of 128 points --
     * that provably hold no in-range pair are skipped ("ignoring calculations that would
     * fall outside the bin range"); 0: every pair is evaluated. */
    ACF_OPT_PRUNE = 2,
    /* 1: collect acf_stats device counters (pairs evaluated, fp64 re-checks); default 1. */
    ACF_OPT_STATS = 3,
    /* 1 (default): where the bounding caps of a warp's i-points and of a group of j-points show that
     * at most one bin edge can separate their pairs, every pair is tested against that one edge and
     * tallied in registers; 0: every pair goes through the bin table and the shared-memory histogram.
     * The counts are the same either way. */
    ACF_OPT_WINDOWS = 4,
    /* 0 (default): every in-range pair is evaluated on its own, as the paper's method does;
     * 1: where the bounding caps of two groups of 128 points prove that all their pairs fall into one
     * and the same bin, the window kernel adds the group's pair count and weight product to that bin
     * without visiting the pairs (the counterpart, inside the range, of skipping what lies outside it;
     * still exact: the proof is the same fp64 bound that picks the edges of a window).  Such pairs are
     * reported in acf_stats.pairs_bulk and not in pairs_evaluated. */
    ACF_OPT_BULK = 5
};
enum { ACF_KERNEL_AUTO = 0, ACF_KERNEL_FP64 = 1, ACF_KERNEL_TABLE = 2, ACF_KERNEL_WINDOW = 3 };

/* Counters of the most recent acf_pair_count* call on a context. */
typedef struct acf_stats {
    uint64_t pairs_nominal;      /* n(n-1)/2 or n_a*n_b (of the requested row range) */
    uint64_t pairs_evaluated;    /* pair cosines actually computed on the device */
    uint64_t pairs_fp64;         /* pairs re-evaluated in double (inside a guard band of an edge) */
    uint64_t pairs_window;       /* of pairs_evaluated: classified against a single edge (ACF_OPT_WINDOWS) */
    uint64_t tile_pairs_total;   /* tile pairs the call is made of */
    uint64_t tile_pairs_pruned;  /* tile pairs skipped as provably out of range */
    uint64_t kernel_launches;    /* CUDA kernels launched by the call */
    double device_ms;            /* device time of the call, CUDA events on the ctx stream */
    double pair_kernel_ms;       /* of which: first to last pair-kernel launch (the dominant kernel) */
    uint64_t pairs_chord;        /* pairs whose row the fp32 chord length decided: those of windows at small separations,
                                    which are classified on it, and those the fp32 cosine had left open (not in pairs_fp64) */
    uint64_t pairs_bulk;         /* pairs counted group by group without being evaluated (ACF_OPT_BULK) */
} acf_stats;

/* Create a context on CUDA device `device`.  cuda_stream: a cudaStream_t (as void*) all
 * work is enqueued on, or NULL for the legacy default stream.  *out is set on success.
 * ACF_ECUDA if the device is missing or is not compute capability 10.x. */
int acf_create(acf_ctx **out, int device, void *cuda_stream);

/* Synchronise the stream, free the context and all its scratch.  NULL is a no-op. */
void acf_destroy(acf_ctx *ctx);

/* Message of the last failure on ctx (ctx-owned, valid until the next call); "" if none.
 * With ctx == NULL: the message of the last failed acf_create in this thread. */
const char *acf_last_error(const acf_ctx *ctx);

/* Set ACF_OPT_* (see above).  ACF_EINVAL for an unknown option or value. */
int acf_set_option(acf_ctx *ctx, int option, int64_t value);

/* Change the stream later calls enqueue on (the previous one is synchronised first). */
int acf_set_stream(acf_ctx *ctx, void *cuda_stream);

/*
 * Canonical unit vectors (App. A).  Pure host function, glibc sin/cos in
 * double:  r = deg * (pi/180 as a double);  x = cos(d)*cos(a), y = cos(d)*sin(a), z = sin(d).
 * ra_deg, dec_deg: HOST, n doubles (degrees).  xyz_host: HOST, 3n doubles, SoA, overwritten.
 * This defines the vectors every count is made from; parity runs use it, not a device sincos.
 */
int acf_radec_to_xyz(const double *ra_deg, const double *dec_deg, size_t n, double *xyz_host);

/*
 * Pair-count histogram: DD or RR with is_auto = 1, DR with 0.
 *   d_a, d_b : DEVICE, canonical xyz SoA of n_a / n_b points.  Components must be finite and
 *              |x^2+y^2+z^2 - 1| <= 1e-6, else ACF_EINVAL (checked on the device; this
 *              error is reported by this same call, which then synchronises).
 *   is_auto  : 1 counts unordered pairs i<j of one catalogue (d_b must equal d_a and n_b n_a);
 *              0 counts all n_a*n_b pairs.
 *   d_counts : DEVICE, nbins uint64, overwritten.
 * n = 0 (or n = 1 in auto mode) gives all-zero counts and ACF_OK.
 * The call prepares both catalogues (sort, caps) every time and waits on the host for the validation verdict while the
 * pair kernel is already running; counts that share catalogues are better made on handles (acf_prepare).
 */
int acf_pair_count(acf_ctx *ctx, const double *d_a, size_t n_a, const double *d_b, size_t n_b,
                   const double *cos_edges, int nbins, int is_auto, uint64_t *d_counts);

/*
 * The same count without any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it).  Needs no context.  Its kernel is a variant of the fp64
 * reference kernel (every pair evaluated in double as defined above: the counts are those of acf_pair_count, bit
 * for bit) whose scratch memory -- the device copy of the edges, a status word, one partial histogram per CTA --
 * is a fixed array in the library's device image: 4.2 MB that every GPU which loads the library holds until the
 * process exits.  Hence the limit: at most ACF_STATIC_MAX_POINTS points per catalogue, ACF_EINVAL beyond
 * (unweighted counts only).  The call enqueues a memset, a copy of the edges and two kernels on cuda_stream and
 * returns; it calls no cudaMalloc, cudaFree or allocating library routine.  The first call on a device asks the
 * runtime for the array's address (and thereby loads the device image there): make it outside a capture.
 *   device      : the GPU that d_a, d_b, d_counts, d_bad and cuda_stream belong to (the caller's current
 *                 device is restored on return).
 *   d_a, d_b, n_a, n_b, cos_edges, nbins, is_auto : as for acf_pair_count.
 *   d_counts    : DEVICE, nbins uint64, overwritten (it need not be zeroed).
 *   d_bad       : DEVICE, one uint32, or NULL: overwritten with the number of invalid points found (non-finite,
 *                 or |x^2+y^2+z^2 - 1| > 1e-6).  The call does not wait for this verdict: where it is not
 *                 zero, d_counts is not to be used.
 *   cuda_stream : the cudaStream_t to enqueue on (NULL: the default stream).
 *   err, err_len: HOST buffer that receives the message of a failure ("" on success), or NULL.
 * All calls share the one array, which keeps the last call's contents: what must start at zero is cleared by
 * every call, but calls that OVERLAP on one GPU (two streams, two host threads) race and give wrong counts.
 * Calls on one stream are ordered and safe.
 */
#define ACF_STATIC_MAX_POINTS 131072
int acf_pair_count_static(int device, const double *d_a, size_t n_a, const double *d_b, size_t n_b,
                          const double *cos_edges, int nbins, int is_auto, uint64_t *d_counts, uint32_t *d_bad,
                          void *cuda_stream, char *err, size_t err_len);

/*
 * Same, with pair weight w_i * w_j (not in the paper; BASELINE.json config 4).
 *   d_wa, d_wb : DEVICE, n_a / n_b floats, finite and >= 0.  In auto mode d_wb must equal d_wa.
 *   d_wsums    : DEVICE, nbins doubles, overwritten with sum over counted pairs of
 *                (double)w_i * (double)w_j.  d_counts as above (unweighted), both are produced.
 */
int acf_pair_count_weighted(acf_ctx *ctx, const double *d_a, const float *d_wa, size_t n_a,
                            const double *d_b, const float *d_wb, size_t n_b, const double *cos_edges,
                            int nbins, int is_auto, uint64_t *d_counts, double *d_wsums);

/*
 * Row range of the pair matrix: rows i in [i_begin, i_end) of catalogue A against B (the
 * paper's sub-matrix decomposition; basis of chunking and of sharding rows
 * over GPUs).  In auto mode row i pairs with j > i only, so the counts of
 * disjoint row ranges covering [0, n_a) add up to the full acf_pair_count result.
 * d_wa/d_wb/d_wsums may all be NULL (unweighted).
 */
int acf_pair_count_rows(acf_ctx *ctx, const double *d_a, const float *d_wa, size_t n_a, size_t i_begin,
                        size_t i_end, const double *d_b, const float *d_wb, size_t n_b,
                        const double *cos_edges, int nbins, int is_auto, uint64_t *d_counts,
                        double *d_wsums);

/*
 * Prepared catalogues (sect. 2.1: the coordinates are copied to the device once and many
 * sub-matrix kernels are launched on them).  acf_prepare validates a catalogue (as acf_pair_count does), sorts it
 * along a space-filling curve and builds its fp32 copies and bounding caps ONCE; any number of counts can then be
 * made on the handle -- DD, DR and RR of an estimate prepare each catalogue once instead of twice, a jackknife
 * prepares every region once -- and those counts are truly asynchronous: the validation verdict was fetched by
 * acf_prepare, so acf_pair_count_prepared never waits on the host.
 *   d_xyz, d_w : DEVICE, as for acf_pair_count_weighted (d_w NULL: unit weights).  The handle REFERS to these
 *                buffers (the exact re-evaluation of near-edge pairs reads the caller's doubles): they must stay
 *                allocated and unchanged until acf_release.
 *   [i_begin, i_end) : the rows that make up the catalogue (acf_prepare: all n of them)
 * acf_prepare* synchronise the stream once (the verdict); ACF_EINVAL for non-unit / non-finite points or bad weights.
 * acf_release frees the handle's device memory after the stream has drained; NULL is a no-op.  acf_destroy frees
 * the handles that are still alive.
 */
int acf_prepare(acf_ctx *ctx, const double *d_xyz, const float *d_w, size_t n, acf_catalog **out);
int acf_prepare_rows(acf_ctx *ctx, const double *d_xyz, const float *d_w, size_t n, size_t i_begin, size_t i_end,
                     acf_catalog **out);
/* Prepares `cat` again on new data (or the same buffers with new contents), reusing its device memory: a pipeline
 * that counts one catalogue after another of about the same size (the many random catalogues of a Monte-Carlo error
 * estimate) allocates once.  Same arguments, waits and errors as acf_prepare_rows; after an error the
 * handle holds an empty catalogue. */
int acf_prepare_again(acf_ctx *ctx, acf_catalog *cat, const double *d_xyz, const float *d_w, size_t n, size_t i_begin,
                      size_t i_end);
void acf_release(acf_ctx *ctx, acf_catalog *cat);

/*
 * Pair-count histogram of prepared catalogues: b == NULL (or b == a) counts the unordered pairs of a (DD, RR),
 * otherwise all pairs of a x b (DR).  Weighted sums are produced iff d_wsums != NULL (both catalogues must then
 * have been prepared with weights).  Asynchronous on the context's stream; d_counts / d_wsums are overwritten.
 *   part, n_parts : the call counts slice `part` of `n_parts` disjoint slices of the pair matrix (rows of a in the
 *                   order of the prepared catalogue, dealt out tile by tile: balanced whatever is pruned).  The
 *                   histograms of the n_parts slices add up to the whole count: this is the unit of work of a job
 *                   sharded over GPUs, every rank holding both catalogues.  0, 1: the whole count.
 */
int acf_pair_count_prepared(acf_ctx *ctx, const acf_catalog *a, const acf_catalog *b, const double *cos_edges, int nbins,
                            int part, int n_parts, uint64_t *d_counts, double *d_wsums);

/*
 * Landy-Szalay estimator, Eq. 2, pure host, O(nbins):
 *   w[k] = (dd - 2 dr + rr) / rr  with  dd = DD[k] / (n_d(n_d-1)/2),  dr = DR[k] / (n_d n_r),
 *   rr = RR[k] / (n_r(n_r-1)/2);  NaN where RR[k] == 0.
 * dd, dr, rr: HOST, nbins uint64.  w_host: HOST, nbins doubles, overwritten.
 */
int acf_wtheta(const uint64_t *dd, const uint64_t *dr, const uint64_t *rr, uint64_t n_d, uint64_t n_r,
               int nbins, double *w_host);

/* Weighted form: the same expression on weighted sums with normalisers
 * ((sum w)^2 - sum w^2)/2 (auto) and (sum w_d)(sum w_r) (cross).  All pointers HOST. */
int acf_wtheta_weighted(const double *wdd, const double *wdr, const double *wrr, const float *w_d,
                        size_t n_d, const float *w_r, size_t n_r, int nbins, double *w_host);

/*
 * Other estimators on the same three histograms ("allows the user to easily experiment
 * with other estimators"), pure host, O(nbins).  With dd, dr, rr the pair-normalised counts of acf_wtheta:
 *   ACF_EST_LANDY_SZALAY  (dd - 2 dr + rr) / rr     (Eq. 2; the same values as acf_wtheta)
 *   ACF_EST_NATURAL       dd / rr - 1               (Peebles & Hauser)
 *   ACF_EST_DAVIS_PEEBLES dd / dr - 1
 *   ACF_EST_HAMILTON      dd rr / dr^2 - 1
 * NaN where the estimator's denominator is zero.  ACF_EINVAL for an unknown kind.
 */
enum { ACF_EST_LANDY_SZALAY = 0, ACF_EST_NATURAL = 1, ACF_EST_DAVIS_PEEBLES = 2, ACF_EST_HAMILTON = 3 };
int acf_estimator(int kind, const uint64_t *dd, const uint64_t *dr, const uint64_t *rr, uint64_t n_d,
                  uint64_t n_r, int nbins, double *w_host);

/*
 * The paper's bin presets (a low and a high limit and "evenly spaced, natural log or
 * log base 10" bins), pure host.  theta_deg_host: HOST, nbins + 1 doubles, overwritten, ascending:
 *   ACF_BINS_EVEN   theta_k = lo + (hi - lo) k / nbins
 *   ACF_BINS_LOG    theta_k = lo (hi / lo)^(k / nbins)   (lo > 0; natural log and log10 spacing are the
 *   ACF_BINS_LOG10                                        same edges, both names are accepted)
 * with theta_0 = lo and theta_nbins = hi exactly; 0 <= lo < hi <= 180.
 * acf_cos_edges turns angle edges (degrees, ascending within [0, 180]) into the descending cosine edges
 * the pair counts take: cos(theta pi/180) by libm, exactly 1 and -1 at 0 and 180 degrees.
 */
enum { ACF_BINS_EVEN = 0, ACF_BINS_LOG = 1, ACF_BINS_LOG10 = 2 };
int acf_theta_edges(int mode, double lo_deg, double hi_deg, int nbins, double *theta_deg_host);
int acf_cos_edges(const double *theta_deg, int n_edges, double *cos_edges_host);

/*
 * Delete-one jackknife of an estimator over n_regions regions of the sky (PAPER.md:201 names "a full
 * MC-based calculation of the errors" as what the speed-up makes affordable; resampling the catalogues
 * by region is its usual form).  For every region k the histograms are recounted without the points of
 * region k -- as DD - (pairs with a point in k), each such set counted by acf_pair_count_rows calls on the
 * device -- and the estimator of the remaining points is formed; cov is the jackknife covariance
 *   cov[a][b] = (N - 1)/N  sum_k (w_k[a] - mean[a]) (w_k[b] - mean[b]),   mean = (1/N) sum_k w_k.
 *   d_xyz_d, d_xyz_r : DEVICE canonical vectors (SoA, 3 n doubles), points ORDERED BY REGION: region k is
 *                      rows [off[k], off[k+1]) (a region may be empty)
 *   off_d, off_r     : HOST, n_regions + 1 offsets, off[0] = 0, off[n_regions] = n, non-decreasing
 *   estimator        : ACF_EST_*
 *   w_full           : HOST, nbins doubles: the estimator of the full catalogues
 *   w_jk             : HOST, n_regions x nbins doubles, row k = the estimator without region k
 *   cov              : HOST, nbins x nbins doubles, or NULL
 * Unweighted.  Synchronous.  2 <= n_regions.  ACF_EINVAL for bad offsets or arguments.
 */
int acf_jackknife(acf_ctx *ctx, const double *d_xyz_d, size_t n_d, const size_t *off_d, const double *d_xyz_r,
                  size_t n_r, const size_t *off_r, int n_regions, const double *cos_edges, int nbins,
                  int estimator, double *w_full, double *w_jk, double *cov);

/*
 * Monte-Carlo errors from an ensemble of random catalogues (the speed-up makes "a full MC-based
 * calculation of the errors" affordable): the data are counted once (DD), every random catalogue k of the ensemble
 * gives DR_k and RR_k, and the estimator is formed n_random times.  The catalogues stream through two internal
 * handles (prepared on the device one after the other, nothing allocated per catalogue) and all 2 n_random + 1
 * counts are enqueued without a host wait in between; the validation verdicts are collected at the end.
 *   data       : the prepared data catalogue (acf_prepare)
 *   d_xyz_r    : HOST array of n_random DEVICE pointers, catalogue k: canonical xyz SoA of n_r[k] points
 *   n_r        : HOST, n_random sizes
 *   dd         : HOST, nbins uint64;  dr, rr : HOST, n_random x nbins uint64 (row k = catalogue k)
 *   w          : HOST, n_random x nbins doubles: the estimator with random catalogue k
 *   mean, cov  : HOST, nbins / nbins x nbins doubles or NULL: mean over k and the sample covariance
 *                cov[a][b] = 1/(K - 1) sum_k (w_k[a] - mean[a]) (w_k[b] - mean[b])  (K = n_random >= 2 for cov)
 * Unweighted.  Synchronous.  ACF_EINVAL if any catalogue fails validation (nothing is returned then).
 */
int acf_random_ensemble(acf_ctx *ctx, const acf_catalog *data, const double *const *d_xyz_r, const size_t *n_r, int n_random,
                        const double *cos_edges, int nbins, int estimator, uint64_t *dd, uint64_t *dr, uint64_t *rr,
                        double *w, double *mean, double *cov);

/*
 * The whole job from HOST buffers: canonicalise both catalogues (acf_radec_to_xyz), copy them
 * to the device, count DD, DR, RR, copy the histograms back and apply Eq. 2.  Synchronous.
 *   ra_*, dec_* : HOST doubles (degrees);  w_d, w_r : HOST floats or both NULL (unweighted)
 *   dd, dr, rr  : HOST, nbins uint64 each, overwritten
 *   wdd, wdr, wrr : HOST, nbins doubles each (weighted sums) or all NULL when unweighted
 *   w_host      : HOST, nbins doubles: the estimator (of the weighted sums when weighted)
 */
int acf_correlate_host(acf_ctx *ctx, const double *ra_d, const double *dec_d, const float *w_d, size_t n_d,
                       const double *ra_r, const double *dec_r, const float *w_r, size_t n_r,
                       const double *cos_edges, int nbins, uint64_t *dd, uint64_t *dr, uint64_t *rr,
                       double *wdd, double *wdr, double *wrr, double *w_host);

/* Counters of the last acf_pair_count* call (synchronises the stream). */
int acf_get_stats(acf_ctx *ctx, acf_stats *out);

/* Library version string, e.g. "acf-b200 0.1 (sm_100a)". */
const char *acf_version(void);

#ifdef __cplusplus
}
#endif
#endif /* ACF_H */
