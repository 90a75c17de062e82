// acf_api.cu -- the C ABI of libacf (include/acf.h): argument checking, context and scratch
// management, and the enqueueing of the device pipeline.  All arithmetic of the method runs in
// the kernels (acf_kernels_*.cu) except the two pure-host functions in acf_host.cpp.
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "acf_internal.h"

namespace {

thread_local char g_create_error[256] = "";

int create_fail(int code, const char *msg, cudaError_t e = cudaSuccess)
{
    if (e != cudaSuccess)
        snprintf(g_create_error, sizeof(g_create_error), "%s: %s", msg, cudaGetErrorString(e));
    else
        snprintf(g_create_error, sizeof(g_create_error), "%s", msg);
    return code;
}

// host-side check of the edge array (include/acf.h CONVENTIONS)
const char *check_edges(const double *e, int nbins)
{
    if (!e) return "cos_edges is NULL";
    if (nbins < 1 || nbins > ACF_MAX_BINS) return "nbins must be in [1, ACF_MAX_BINS]";
    for (int m = 0; m <= nbins; ++m) {
        if (!(e[m] >= -1.0 && e[m] <= 1.0)) return "cos_edges must lie within [-1, 1]";
        if (m && !(e[m] < e[m - 1])) return "cos_edges must be strictly descending";
    }
    return nullptr;
}

}  // namespace

extern "C" const char *acf_version(void) { return "acf-b200 0.1 (sm_100a)"; }

extern "C" int acf_create(acf_ctx **out, int device, void *cuda_stream)
{
    if (!out) return create_fail(ACF_EINVAL, "out is NULL");
    *out = nullptr;
    int count = 0;
    cudaError_t e = cudaGetDeviceCount(&count);
    if (e != cudaSuccess || count == 0) return create_fail(ACF_ECUDA, "no CUDA device (libacf has no CPU fallback)", e);
    if (device < 0 || device >= count) return create_fail(ACF_EINVAL, "device index out of range");
    cudaDeviceProp prop;
    if ((e = cudaGetDeviceProperties(&prop, device)) != cudaSuccess) return create_fail(ACF_ECUDA, "cudaGetDeviceProperties", e);
    if (prop.major != 10) return create_fail(ACF_ECUDA, "libacf is built for sm_100a only (compute capability 10.x required)");
    if ((e = cudaSetDevice(device)) != cudaSuccess) return create_fail(ACF_ECUDA, "cudaSetDevice", e);

    acf_ctx *ctx = new (std::nothrow) acf_ctx();
    if (!ctx) return create_fail(ACF_ENOMEM, "out of host memory");
    ctx->device = device;
    ctx->stream = static_cast<cudaStream_t>(cuda_stream);
    ctx->num_sms = prop.multiProcessorCount;
    ctx->max_smem_optin = (int)prop.sharedMemPerBlockOptin;
    bool ok = cudaEventCreate(&ctx->ev_start) == cudaSuccess && cudaEventCreate(&ctx->ev_stop) == cudaSuccess &&
              cudaEventCreateWithFlags(&ctx->ev_flag, cudaEventDisableTiming) == cudaSuccess &&
              cudaEventCreate(&ctx->ev_k0) == cudaSuccess && cudaEventCreate(&ctx->ev_k1) == cudaSuccess &&
              cudaMalloc(&ctx->d_counters, sizeof(unsigned long long) * acf::kNumCounters) == cudaSuccess &&
              cudaHostAlloc(&ctx->h_counters, sizeof(unsigned long long) * acf::kNumCounters, cudaHostAllocDefault) == cudaSuccess;
    if (!ok) {
        e = cudaGetLastError();
        acf_destroy(ctx);
        return create_fail(ACF_ECUDA, "context allocation failed", e);
    }
    memset(ctx->h_counters, 0, sizeof(unsigned long long) * acf::kNumCounters);
    g_create_error[0] = 0;
    *out = ctx;
    return ACF_OK;
}

extern "C" void acf_destroy(acf_ctx *ctx)
{
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    ctx->s_edges.release();
    for (int i = 0; i < 2; ++i) {
        ctx->s_pts[i].release();
        ctx->s_perm[i].release();
        ctx->s_keys[i].release();
        ctx->s_caps[i].release();
        ctx->s_gcaps[i].release();
        ctx->s_scaps[i].release();
        ctx->s_pts2[i].release();
        ctx->s_vj[i].release();
        ctx->s_pack[i].release();
    }
    ctx->s_work.release();
    ctx->s_misc.release();
    for (auto &s : ctx->s_host_stage) s.release();
    if (ctx->h_stage) cudaFreeHost(ctx->h_stage);
    if (ctx->d_counters) cudaFree(ctx->d_counters);
    if (ctx->h_counters) cudaFreeHost(ctx->h_counters);
    if (ctx->ev_start) cudaEventDestroy(ctx->ev_start);
    if (ctx->ev_stop) cudaEventDestroy(ctx->ev_stop);
    if (ctx->ev_flag) cudaEventDestroy(ctx->ev_flag);
    if (ctx->ev_k0) cudaEventDestroy(ctx->ev_k0);
    if (ctx->ev_k1) cudaEventDestroy(ctx->ev_k1);
    delete ctx;
}

extern "C" const char *acf_last_error(const acf_ctx *ctx) { return ctx ? ctx->err : g_create_error; }

extern "C" int acf_set_option(acf_ctx *ctx, int option, int64_t value)
{
    if (!ctx) return ACF_EINVAL;
    switch (option) {
    case ACF_OPT_KERNEL:
        if (value < ACF_KERNEL_AUTO || value > ACF_KERNEL_WINDOW) return acf::fail(ctx, ACF_EINVAL, "unknown kernel %lld", (long long)value);
        ctx->opt_kernel = (int)value;
        return ACF_OK;
    case ACF_OPT_PRUNE:
        ctx->opt_prune = value != 0;
        return ACF_OK;
    case ACF_OPT_STATS:
        ctx->opt_stats = value != 0;
        return ACF_OK;
    case ACF_OPT_WINDOWS:
        ctx->opt_windows = value != 0;
        return ACF_OK;
    case ACF_OPT_BULK:
        ctx->opt_bulk = value != 0;
        return ACF_OK;
    default:
        return acf::fail(ctx, ACF_EINVAL, "unknown option %d", option);
    }
}

extern "C" int acf_set_stream(acf_ctx *ctx, void *cuda_stream)
{
    if (!ctx) return ACF_EINVAL;
    ACF_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    ACF_CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->stream = static_cast<cudaStream_t>(cuda_stream);
    return ACF_OK;
}

extern "C" int acf_pair_count_rows(acf_ctx *ctx, const double *d_a, const float *d_wa, size_t n_a, size_t i_begin,
                                   size_t i_end, const double *d_b, const float *d_wb, size_t n_b,
                                   const double *cos_edges, int nbins, int is_auto, uint64_t *d_counts,
                                   double *d_wsums)
{
    if (!ctx) return ACF_EINVAL;
    ctx->err[0] = 0;
    if (const char *why = check_edges(cos_edges, nbins)) return acf::fail(ctx, ACF_EINVAL, "%s", why);
    if (!d_counts) return acf::fail(ctx, ACF_EINVAL, "d_counts is NULL");
    if ((n_a && !d_a) || (n_b && !d_b)) return acf::fail(ctx, ACF_EINVAL, "catalogue pointer is NULL");
    if (i_begin > i_end || i_end > n_a) return acf::fail(ctx, ACF_EINVAL, "row range [%zu, %zu) outside [0, %zu]", i_begin, i_end, n_a);
    is_auto = is_auto != 0;
    if (is_auto && (d_a != d_b || n_a != n_b)) return acf::fail(ctx, ACF_EINVAL, "is_auto needs d_b == d_a and n_b == n_a");
    const bool weighted = d_wsums != nullptr;
    if (weighted && ((n_a && !d_wa) || (n_b && !d_wb))) return acf::fail(ctx, ACF_EINVAL, "weighted call needs d_wa and d_wb");
    if (weighted && is_auto && d_wa != d_wb) return acf::fail(ctx, ACF_EINVAL, "is_auto needs d_wb == d_wa");
    if (!weighted) d_wa = d_wb = nullptr;
    if (n_a >= (size_t(1) << 31) || n_b >= (size_t(1) << 31)) return acf::fail(ctx, ACF_EINVAL, "catalogues are limited to 2^31-1 points");

    ACF_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    ctx->last = acf_stats{};
    ctx->pair_timed = false;
    {
        // pairs the call is defined over
        // auto: T(n - i_begin) - T(n - i_end) with T(m) = m(m-1)/2 pairs among the last m points
        auto tri = [](size_t m) { return (unsigned __int128)m * (m ? m - 1 : 0) / 2; };
        const unsigned __int128 nominal = is_auto ? tri(n_a - i_begin) - tri(n_a - i_end)
                                                  : (unsigned __int128)(i_end - i_begin) * n_b;
        ctx->last.pairs_nominal = (uint64_t)nominal;
    }
    ACF_CUDA_TRY(ctx, cudaEventRecord(ctx->ev_start, st));
    ACF_CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_counters, 0, sizeof(unsigned long long) * acf::kNumCounters, st));
    ACF_CUDA_TRY(ctx, cudaMemsetAsync(d_counts, 0, sizeof(uint64_t) * (size_t)nbins, st));
    if (weighted) ACF_CUDA_TRY(ctx, cudaMemsetAsync(d_wsums, 0, sizeof(double) * (size_t)nbins, st));
    ctx->stats_pending = true;

    const bool empty = i_begin == i_end || n_b == 0 || (is_auto && n_a < 2);
    if (!empty) {
        ACF_CUDA_TRY(ctx, acf::launch_validate(ctx, d_a, d_wa, n_a));
        if (!is_auto) ACF_CUDA_TRY(ctx, acf::launch_validate(ctx, d_b, d_wb, n_b));
        ACF_CUDA_TRY(ctx, cudaMemcpyAsync(&ctx->h_counters[acf::kCtrBadInput], &ctx->d_counters[acf::kCtrBadInput],
                                          sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
        ACF_CUDA_TRY(ctx, cudaEventRecord(ctx->ev_flag, st));

        if (ctx->opt_kernel != ACF_KERNEL_FP64) {
            int rc = acf::run_pair_count_fast(ctx, d_a, d_wa, n_a, i_begin, i_end, d_b, d_wb, n_b, cos_edges, nbins,
                                              is_auto, reinterpret_cast<unsigned long long *>(d_counts), d_wsums);
            if (rc != ACF_OK) return rc;
        } else {
            ACF_CUDA_TRY(ctx, ctx->s_edges.reserve(sizeof(double) * (size_t)(nbins + 1)));
            ACF_CUDA_TRY(ctx, cudaMemcpyAsync(ctx->s_edges.ptr, cos_edges, sizeof(double) * (size_t)(nbins + 1), cudaMemcpyHostToDevice, st));
            ACF_CUDA_TRY(ctx, acf::launch_pair_count_fp64(ctx, d_a, d_wa, n_a, i_begin, i_end, d_b, d_wb, n_b,
                                                          ctx->s_edges.as<double>(), nbins, is_auto,
                                                          reinterpret_cast<unsigned long long *>(d_counts), d_wsums));
        }
    }
    ACF_CUDA_TRY(ctx, cudaEventRecord(ctx->ev_stop, st));

    if (!empty) {
        // wait for the validation verdict only (the pair kernel keeps running asynchronously)
        ACF_CUDA_TRY(ctx, cudaEventSynchronize(ctx->ev_flag));
        if (ctx->h_counters[acf::kCtrBadInput] != 0) {
            cudaStreamSynchronize(st);
            cudaMemsetAsync(d_counts, 0, sizeof(uint64_t) * (size_t)nbins, st);
            if (weighted) cudaMemsetAsync(d_wsums, 0, sizeof(double) * (size_t)nbins, st);
            cudaStreamSynchronize(st);
            return acf::fail(ctx, ACF_EINVAL, "%llu input points are not finite unit vectors (|r^2 - 1| <= 1e-6) or carry a negative / non-finite weight",
                             ctx->h_counters[acf::kCtrBadInput]);
        }
    }
    return ACF_OK;
}

extern "C" int acf_pair_count(acf_ctx *ctx, const double *d_a, size_t n_a, const double *d_b, size_t n_b,
                              const double *cos_edges, int nbins, int is_auto, uint64_t *d_counts)
{
    return acf_pair_count_rows(ctx, d_a, nullptr, n_a, 0, n_a, d_b, nullptr, n_b, cos_edges, nbins, is_auto, d_counts, nullptr);
}

extern "C" int acf_pair_count_weighted(acf_ctx *ctx, const double *d_a, const float *d_wa, size_t n_a,
                                       const double *d_b, const float *d_wb, size_t n_b, const double *cos_edges,
                                       int nbins, int is_auto, uint64_t *d_counts, double *d_wsums)
{
    if (!ctx) return ACF_EINVAL;
    if (!d_wsums) return acf::fail(ctx, ACF_EINVAL, "d_wsums is NULL");
    return acf_pair_count_rows(ctx, d_a, d_wa, n_a, 0, n_a, d_b, d_wb, n_b, cos_edges, nbins, is_auto, d_counts, d_wsums);
}

extern "C" int acf_get_stats(acf_ctx *ctx, acf_stats *out)
{
    if (!ctx || !out) return ACF_EINVAL;
    ACF_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    if (ctx->stats_pending) {
        ACF_CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_counters, ctx->d_counters, sizeof(unsigned long long) * acf::kNumCounters,
                                          cudaMemcpyDeviceToHost, ctx->stream));
        ACF_CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, ctx->ev_start, ctx->ev_stop) == cudaSuccess) ctx->last.device_ms = ms;
        if (ctx->pair_timed && cudaEventElapsedTime(&ms, ctx->ev_k0, ctx->ev_k1) == cudaSuccess) ctx->last.pair_kernel_ms = ms;
        ctx->last.pairs_evaluated = ctx->h_counters[acf::kCtrPairsEvaluated];
        ctx->last.pairs_fp64 = ctx->h_counters[acf::kCtrPairsFp64];
        ctx->last.pairs_window = ctx->h_counters[acf::kCtrPairsWindow];
        ctx->last.pairs_chord = ctx->h_counters[acf::kCtrPairsChord];
        ctx->last.pairs_bulk = ctx->h_counters[acf::kCtrPairsBulk];
        ctx->last.tile_pairs_total = ctx->h_counters[acf::kCtrTilePairsTotal];
        ctx->last.tile_pairs_pruned = ctx->h_counters[acf::kCtrTilePairsPruned];
        ctx->stats_pending = false;
    }
    *out = ctx->last;
    return ACF_OK;
}

// Delete-one jackknife (include/acf.h).  Pairs with a point in region k, for a catalogue ordered by region:
// rows k of the auto-count (pairs inside k and from k to the regions after it) plus the rows before k
// against region k.  The cross-count loses D_k x R, D x R_k and gets D_k x R_k back.
extern "C" int acf_jackknife(acf_ctx *ctx, const double *d_xyz_d, size_t n_d, const size_t *off_d, const double *d_xyz_r,
                             size_t n_r, const size_t *off_r, int n_regions, const double *cos_edges, int nbins,
                             int estimator, double *w_full, double *w_jk, double *cov)
{
    if (!ctx) return ACF_EINVAL;
    ctx->err[0] = 0;
    if (const char *why = check_edges(cos_edges, nbins)) return acf::fail(ctx, ACF_EINVAL, "%s", why);
    if (!d_xyz_d || !d_xyz_r || !off_d || !off_r || !w_full || !w_jk) return acf::fail(ctx, ACF_EINVAL, "NULL argument");
    if (n_regions < 2) return acf::fail(ctx, ACF_EINVAL, "n_regions must be at least 2");
    if (estimator < ACF_EST_LANDY_SZALAY || estimator > ACF_EST_HAMILTON) return acf::fail(ctx, ACF_EINVAL, "unknown estimator");
    size_t max_d = 0, max_r = 0;
    for (int k = 0; k < n_regions; ++k) {
        if (off_d[k + 1] < off_d[k] || off_r[k + 1] < off_r[k]) return acf::fail(ctx, ACF_EINVAL, "region offsets must not decrease");
        if (off_d[k + 1] - off_d[k] > max_d) max_d = off_d[k + 1] - off_d[k];
        if (off_r[k + 1] - off_r[k] > max_r) max_r = off_r[k + 1] - off_r[k];
    }
    if (off_d[0] != 0 || off_r[0] != 0 || off_d[n_regions] != n_d || off_r[n_regions] != n_r)
        return acf::fail(ctx, ACF_EINVAL, "region offsets must run from 0 to n");
    ACF_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    const size_t nb = (size_t)nbins;
    // scratch: the points of region k of either catalogue as catalogues of their own, and 8 histograms
    ACF_CUDA_TRY(ctx, ctx->s_host_stage[0].reserve(sizeof(double) * 3 * (max_d ? max_d : 1)));
    ACF_CUDA_TRY(ctx, ctx->s_host_stage[1].reserve(sizeof(double) * 3 * (max_r ? max_r : 1)));
    ACF_CUDA_TRY(ctx, ctx->s_host_stage[4].reserve(sizeof(uint64_t) * 8 * nb));
    double *d_dk = ctx->s_host_stage[0].as<double>(), *d_rk = ctx->s_host_stage[1].as<double>();
    uint64_t *d_cnt = ctx->s_host_stage[4].as<uint64_t>();
    std::vector<uint64_t> h((size_t)8 * nb), tot((size_t)3 * nb), dd(nb), dr(nb), rr(nb);

    int rc;
    auto count = [&](const double *a, size_t na, size_t i0, size_t i1, const double *b, size_t nbp, int is_auto, int slot) -> int {
        return acf_pair_count_rows(ctx, a, nullptr, na, i0, i1, b, nullptr, nbp, cos_edges, nbins, is_auto, d_cnt + (size_t)slot * nb, nullptr);
    };
    auto fetch = [&](int slots) -> int {
        ACF_CUDA_TRY(ctx, cudaMemcpyAsync(h.data(), d_cnt, sizeof(uint64_t) * (size_t)slots * nb, cudaMemcpyDeviceToHost, st));
        ACF_CUDA_TRY(ctx, cudaStreamSynchronize(st));
        return ACF_OK;
    };
    auto subset = [&](const double *src, size_t n, size_t lo, size_t cnt, double *dst) -> int {
        for (int c = 0; c < 3 && cnt; ++c)
            ACF_CUDA_TRY(ctx, cudaMemcpyAsync(dst + (size_t)c * cnt, src + (size_t)c * n + lo, sizeof(double) * cnt, cudaMemcpyDeviceToDevice, st));
        return ACF_OK;
    };
    if ((rc = count(d_xyz_d, n_d, 0, n_d, d_xyz_d, n_d, 1, 0)) != ACF_OK) return rc;
    if ((rc = count(d_xyz_d, n_d, 0, n_d, d_xyz_r, n_r, 0, 1)) != ACF_OK) return rc;
    if ((rc = count(d_xyz_r, n_r, 0, n_r, d_xyz_r, n_r, 1, 2)) != ACF_OK) return rc;
    if ((rc = fetch(3)) != ACF_OK) return rc;
    tot.assign(h.begin(), h.begin() + 3 * (long)nb);
    if ((rc = acf_estimator(estimator, tot.data(), tot.data() + nb, tot.data() + 2 * nb, n_d, n_r, nbins, w_full)) != ACF_OK) return rc;

    for (int k = 0; k < n_regions; ++k) {
        const size_t d0 = off_d[k], d1 = off_d[k + 1], r0 = off_r[k], r1 = off_r[k + 1];
        const size_t ndk = d1 - d0, nrk = r1 - r0;
        if ((rc = subset(d_xyz_d, n_d, d0, ndk, d_dk)) != ACF_OK) return rc;
        if ((rc = subset(d_xyz_r, n_r, r0, nrk, d_rk)) != ACF_OK) return rc;
        // slots: 0 DD rows k, 1 DD rows before k x D_k, 2 RR rows k, 3 RR rows before k x R_k,
        //        4 D_k x R, 5 D x R_k, 6 D_k x R_k
        if ((rc = count(d_xyz_d, n_d, d0, d1, d_xyz_d, n_d, 1, 0)) != ACF_OK) return rc;
        if ((rc = count(d_xyz_d, n_d, 0, d0, d_dk, ndk, 0, 1)) != ACF_OK) return rc;
        if ((rc = count(d_xyz_r, n_r, r0, r1, d_xyz_r, n_r, 1, 2)) != ACF_OK) return rc;
        if ((rc = count(d_xyz_r, n_r, 0, r0, d_rk, nrk, 0, 3)) != ACF_OK) return rc;
        if ((rc = count(d_xyz_d, n_d, d0, d1, d_xyz_r, n_r, 0, 4)) != ACF_OK) return rc;
        if ((rc = count(d_xyz_d, n_d, 0, n_d, d_rk, nrk, 0, 5)) != ACF_OK) return rc;
        if ((rc = count(d_dk, ndk, 0, ndk, d_rk, nrk, 0, 6)) != ACF_OK) return rc;
        if ((rc = fetch(7)) != ACF_OK) return rc;
        for (size_t b = 0; b < nb; ++b) {
            dd[b] = tot[b] - h[b] - h[nb + b];
            rr[b] = tot[2 * nb + b] - h[2 * nb + b] - h[3 * nb + b];
            dr[b] = tot[nb + b] - h[4 * nb + b] - h[5 * nb + b] + h[6 * nb + b];
        }
        if ((rc = acf_estimator(estimator, dd.data(), dr.data(), rr.data(), n_d - ndk, n_r - nrk, nbins, w_jk + (size_t)k * nb)) != ACF_OK)
            return rc;
    }
    if (cov) {
        std::vector<double> mean(nb, 0.0);
        for (int k = 0; k < n_regions; ++k)
            for (size_t b = 0; b < nb; ++b) mean[b] += w_jk[(size_t)k * nb + b];
        for (size_t b = 0; b < nb; ++b) mean[b] /= (double)n_regions;
        const double f = (double)(n_regions - 1) / (double)n_regions;
        for (size_t a = 0; a < nb; ++a)
            for (size_t b = 0; b < nb; ++b) {
                double sum = 0.0;
                for (int k = 0; k < n_regions; ++k) sum += (w_jk[(size_t)k * nb + a] - mean[a]) * (w_jk[(size_t)k * nb + b] - mean[b]);
                cov[a * nb + b] = f * sum;
            }
    }
    return ACF_OK;
}

extern "C" int acf_correlate_host(acf_ctx *ctx, const double *ra_d, const double *dec_d, const float *w_d, size_t n_d,
                                  const double *ra_r, const double *dec_r, const float *w_r, size_t n_r,
                                  const double *cos_edges, int nbins, uint64_t *dd, uint64_t *dr, uint64_t *rr,
                                  double *wdd, double *wdr, double *wrr, double *w_host)
{
    if (!ctx) return ACF_EINVAL;
    ctx->err[0] = 0;
    if (const char *why = check_edges(cos_edges, nbins)) return acf::fail(ctx, ACF_EINVAL, "%s", why);
    if ((n_d && (!ra_d || !dec_d)) || (n_r && (!ra_r || !dec_r))) return acf::fail(ctx, ACF_EINVAL, "catalogue pointer is NULL");
    if (!dd || !dr || !rr || !w_host) return acf::fail(ctx, ACF_EINVAL, "output pointer is NULL");
    const bool weighted = w_d || w_r;
    if (weighted && ((n_d && !w_d) || (n_r && !w_r) || !wdd || !wdr || !wrr))
        return acf::fail(ctx, ACF_EINVAL, "weighted call needs w_d, w_r, wdd, wdr and wrr");
    ACF_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;

    // pinned staging: xyz of both catalogues, then the outputs
    const size_t xyz_bytes = sizeof(double) * 3 * (n_d + n_r);
    const size_t out_bytes = (sizeof(uint64_t) + sizeof(double)) * 3 * (size_t)nbins;
    if (ctx->h_stage_bytes < xyz_bytes + out_bytes) {
        if (ctx->h_stage) cudaFreeHost(ctx->h_stage);
        ctx->h_stage = nullptr;
        ctx->h_stage_bytes = 0;
        ACF_CUDA_TRY(ctx, cudaHostAlloc(&ctx->h_stage, xyz_bytes + out_bytes, cudaHostAllocDefault));
        ctx->h_stage_bytes = xyz_bytes + out_bytes;
    }
    double *h_xyz_d = static_cast<double *>(ctx->h_stage), *h_xyz_r = h_xyz_d + 3 * n_d;
    uint64_t *h_cnt = reinterpret_cast<uint64_t *>(h_xyz_r + 3 * n_r);
    double *h_ws = reinterpret_cast<double *>(h_cnt + 3 * (size_t)nbins);
    // the randoms are canonicalised on the host while the device counts DD (PAPER.md:128 names the
    // overlap of transfers and kernels as the step its own code did not take)
    acf_radec_to_xyz(ra_d, dec_d, n_d, h_xyz_d);

    ACF_CUDA_TRY(ctx, ctx->s_host_stage[0].reserve(sizeof(double) * 3 * (n_d ? n_d : 1)));
    ACF_CUDA_TRY(ctx, ctx->s_host_stage[1].reserve(sizeof(double) * 3 * (n_r ? n_r : 1)));
    ACF_CUDA_TRY(ctx, ctx->s_host_stage[2].reserve(sizeof(float) * (n_d ? n_d : 1)));
    ACF_CUDA_TRY(ctx, ctx->s_host_stage[3].reserve(sizeof(float) * (n_r ? n_r : 1)));
    ACF_CUDA_TRY(ctx, ctx->s_host_stage[4].reserve(sizeof(uint64_t) * 3 * (size_t)nbins));
    ACF_CUDA_TRY(ctx, ctx->s_host_stage[5].reserve(sizeof(double) * 3 * (size_t)nbins));
    double *d_xd = ctx->s_host_stage[0].as<double>(), *d_xr = ctx->s_host_stage[1].as<double>();
    float *d_wd = weighted ? ctx->s_host_stage[2].as<float>() : nullptr, *d_wr = weighted ? ctx->s_host_stage[3].as<float>() : nullptr;
    uint64_t *d_cnt = ctx->s_host_stage[4].as<uint64_t>();
    double *d_ws = weighted ? ctx->s_host_stage[5].as<double>() : nullptr;
    if (n_d) ACF_CUDA_TRY(ctx, cudaMemcpyAsync(d_xd, h_xyz_d, sizeof(double) * 3 * n_d, cudaMemcpyHostToDevice, st));
    if (weighted && n_d) ACF_CUDA_TRY(ctx, cudaMemcpyAsync(d_wd, w_d, sizeof(float) * n_d, cudaMemcpyHostToDevice, st));

    int rc;
    rc = acf_pair_count_rows(ctx, d_xd, d_wd, n_d, 0, n_d, d_xd, d_wd, n_d, cos_edges, nbins, 1, d_cnt, d_ws);
    if (rc != ACF_OK) return rc;
    acf_radec_to_xyz(ra_r, dec_r, n_r, h_xyz_r);
    if (n_r) ACF_CUDA_TRY(ctx, cudaMemcpyAsync(d_xr, h_xyz_r, sizeof(double) * 3 * n_r, cudaMemcpyHostToDevice, st));
    if (weighted && n_r) ACF_CUDA_TRY(ctx, cudaMemcpyAsync(d_wr, w_r, sizeof(float) * n_r, cudaMemcpyHostToDevice, st));
    rc = acf_pair_count_rows(ctx, d_xd, d_wd, n_d, 0, n_d, d_xr, d_wr, n_r, cos_edges, nbins, 0, d_cnt + nbins, d_ws ? d_ws + nbins : nullptr);
    if (rc != ACF_OK) return rc;
    rc = acf_pair_count_rows(ctx, d_xr, d_wr, n_r, 0, n_r, d_xr, d_wr, n_r, cos_edges, nbins, 1, d_cnt + 2 * nbins, d_ws ? d_ws + 2 * nbins : nullptr);
    if (rc != ACF_OK) return rc;

    ACF_CUDA_TRY(ctx, cudaMemcpyAsync(h_cnt, d_cnt, sizeof(uint64_t) * 3 * (size_t)nbins, cudaMemcpyDeviceToHost, st));
    if (weighted) ACF_CUDA_TRY(ctx, cudaMemcpyAsync(h_ws, d_ws, sizeof(double) * 3 * (size_t)nbins, cudaMemcpyDeviceToHost, st));
    ACF_CUDA_TRY(ctx, cudaStreamSynchronize(st));
    memcpy(dd, h_cnt, sizeof(uint64_t) * (size_t)nbins);
    memcpy(dr, h_cnt + nbins, sizeof(uint64_t) * (size_t)nbins);
    memcpy(rr, h_cnt + 2 * nbins, sizeof(uint64_t) * (size_t)nbins);
    if (weighted) {
        memcpy(wdd, h_ws, sizeof(double) * (size_t)nbins);
        memcpy(wdr, h_ws + nbins, sizeof(double) * (size_t)nbins);
        memcpy(wrr, h_ws + 2 * nbins, sizeof(double) * (size_t)nbins);
        return acf_wtheta_weighted(wdd, wdr, wrr, w_d, n_d, w_r, n_r, nbins, w_host);
    }
    return acf_wtheta(dd, dr, rr, n_d, n_r, nbins, w_host);
}
