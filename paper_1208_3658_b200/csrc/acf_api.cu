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
              cudaEventCreateWithFlags(&ctx->ev_tables, cudaEventDisableTiming) == cudaSuccess &&
              cudaEventCreateWithFlags(&ctx->ev_copy, cudaEventDisableTiming) == cudaSuccess &&
              cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking) == cudaSuccess &&
              cudaMalloc(&ctx->d_counters, sizeof(unsigned long long) * acf::kNumCounters) == cudaSuccess &&
              cudaHostAlloc(&ctx->h_counters, sizeof(unsigned long long) * (acf::kNumCounters + 2), cudaHostAllocDefault) == cudaSuccess;
    if (!ok) {
        e = cudaGetLastError();
        acf_destroy(ctx);
        return create_fail(ACF_ECUDA, "context allocation failed", e);
    }
    memset(ctx->h_counters, 0, sizeof(unsigned long long) * (acf::kNumCounters + 2));
    ctx->h_verdict = reinterpret_cast<int *>(ctx->h_counters + acf::kNumCounters);
    g_create_error[0] = 0;
    *out = ctx;
    return ACF_OK;
}

extern "C" void acf_destroy(acf_ctx *ctx)
{
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    if (ctx->copy_stream) cudaStreamSynchronize(ctx->copy_stream);
    while (ctx->catalogs) acf_release(ctx, ctx->catalogs);
    ctx->s_edges.release();
    for (int i = 0; i < 2; ++i) ctx->cat[i].release();
    ctx->s_keys.release();
    ctx->s_work.release();
    ctx->s_misc.release();
    for (auto &s : ctx->s_host_stage) s.release();
    if (ctx->h_stage) cudaFreeHost(ctx->h_stage);
    if (ctx->h_tables) cudaFreeHost(ctx->h_tables);
    if (ctx->ev_tables) cudaEventDestroy(ctx->ev_tables);
    if (ctx->ev_copy) cudaEventDestroy(ctx->ev_copy);
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
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
    if (!empty && ctx->opt_kernel == ACF_KERNEL_FP64) {
        // the reference kernel: validation into the slot's PackInfo, then the definition for every pair
        acf::Prepared a, b;
        for (int k = 0; k < 2; ++k) {
            ACF_CUDA_TRY(ctx, ctx->cat[k].slab.reserve(64));
            ACF_CUDA_TRY(ctx, cudaMemsetAsync(ctx->cat[k].slab.ptr, 0, 64, st));
        }
        a.pack = ctx->cat[0].slab.as<acf::PackInfo>();
        b.pack = ctx->cat[1].slab.as<acf::PackInfo>();
        ACF_CUDA_TRY(ctx, acf::launch_validate(ctx, d_a, n_a, 0, n_a, d_wa, a.pack));
        if (!is_auto) ACF_CUDA_TRY(ctx, acf::launch_validate(ctx, d_b, n_b, 0, n_b, d_wb, b.pack));
        ACF_CUDA_TRY(ctx, cudaMemcpyAsync(&ctx->h_verdict[0], &a.pack->bad, sizeof(int), cudaMemcpyDeviceToHost, st));
        ACF_CUDA_TRY(ctx, cudaMemcpyAsync(&ctx->h_verdict[1], &b.pack->bad, sizeof(int), cudaMemcpyDeviceToHost, st));
        ACF_CUDA_TRY(ctx, cudaEventRecord(ctx->ev_flag, st));
        ACF_CUDA_TRY(ctx, cudaEventSynchronize(ctx->ev_flag));  // (this kernel indexes nothing by the data, but a refused call must count nothing)
        if (ctx->h_verdict[0] == 0 && ctx->h_verdict[1] == 0) {
            ACF_CUDA_TRY(ctx, ctx->s_edges.reserve(sizeof(double) * (size_t)(nbins + 1)));
            ACF_CUDA_TRY(ctx, cudaMemcpyAsync(ctx->s_edges.ptr, cos_edges, sizeof(double) * (size_t)(nbins + 1), cudaMemcpyHostToDevice, st));
            ACF_CUDA_TRY(ctx, acf::launch_pair_count_fp64(ctx, d_a, d_wa, n_a, i_begin, i_end, d_b, d_wb, n_b,
                                                          ctx->s_edges.as<double>(), nbins, is_auto,
                                                          reinterpret_cast<unsigned long long *>(d_counts), d_wsums));
            ACF_CUDA_TRY(ctx, cudaStreamSynchronize(st));  // (cos_edges was copied from the caller's pageable array)
        }
    } else if (!empty) {
        // prepare what the call pairs -- rows [i_begin, i_end) of a as a catalogue of their own; for an auto-count
        // the rows after them as the second one -- and count; the verdicts of the validations travel behind
        acf::Prepared a, b;
        unsigned long long *cnt = reinterpret_cast<unsigned long long *>(d_counts);
        int rc = acf::prepare_catalogue(ctx, ctx->cat[0], d_a, n_a, i_begin, i_end - i_begin, d_wa, &a);
        if (rc != ACF_OK) return rc;
        ACF_CUDA_TRY(ctx, cudaMemcpyAsync(&ctx->h_verdict[0], &a.pack->bad, sizeof(int), cudaMemcpyDeviceToHost, st));
        ctx->h_verdict[1] = 0;
        if (is_auto) {
            if (i_end < n_a) {
                rc = acf::prepare_catalogue(ctx, ctx->cat[1], d_a, n_a, i_end, n_a - i_end, d_wa, &b);
                if (rc != ACF_OK) return rc;
                ACF_CUDA_TRY(ctx, cudaMemcpyAsync(&ctx->h_verdict[1], &b.pack->bad, sizeof(int), cudaMemcpyDeviceToHost, st));
            }
            ACF_CUDA_TRY(ctx, cudaEventRecord(ctx->ev_flag, st));
            rc = acf::count_prepared_part(ctx, a, a, 1, cos_edges, nbins, 0, 1, cnt, d_wsums);
            if (rc == ACF_OK && i_end < n_a) rc = acf::count_prepared_part(ctx, a, b, 0, cos_edges, nbins, 0, 1, cnt, d_wsums);
        } else {
            rc = acf::prepare_catalogue(ctx, ctx->cat[1], d_b, n_b, 0, n_b, d_wb, &b);
            if (rc != ACF_OK) return rc;
            ACF_CUDA_TRY(ctx, cudaMemcpyAsync(&ctx->h_verdict[1], &b.pack->bad, sizeof(int), cudaMemcpyDeviceToHost, st));
            ACF_CUDA_TRY(ctx, cudaEventRecord(ctx->ev_flag, st));
            rc = acf::count_prepared_part(ctx, a, b, 0, cos_edges, nbins, 0, 1, cnt, d_wsums);
        }
        if (rc != ACF_OK) return rc;
    }
    ACF_CUDA_TRY(ctx, cudaEventRecord(ctx->ev_stop, st));

    if (!empty) {
        // wait for the validation verdict only (the pair kernel keeps running asynchronously; it has seen the same
        // verdict on the device and counts nothing if it is bad)
        ACF_CUDA_TRY(ctx, cudaEventSynchronize(ctx->ev_flag));
        const long long bad = (long long)ctx->h_verdict[0] + ctx->h_verdict[1];
        if (bad != 0) {
            cudaStreamSynchronize(st);
            cudaMemsetAsync(d_counts, 0, sizeof(uint64_t) * (size_t)nbins, st);
            if (weighted) cudaMemsetAsync(d_wsums, 0, sizeof(double) * (size_t)nbins, st);
            cudaStreamSynchronize(st);
            return acf::fail(ctx, ACF_EINVAL, "%lld input points are not finite unit vectors (|r^2 - 1| <= 1e-6) or carry a negative / non-finite weight", bad);
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

// ---- prepared catalogues -------------------------------------------------------------------------------------------
extern "C" int acf_prepare_rows(acf_ctx *ctx, const double *d_xyz, const float *d_w, size_t n, size_t i_begin, size_t i_end,
                                acf_catalog **out)
{
    if (!ctx) return ACF_EINVAL;
    ctx->err[0] = 0;
    if (!out) return acf::fail(ctx, ACF_EINVAL, "out is NULL");
    *out = nullptr;
    if (n && !d_xyz) return acf::fail(ctx, ACF_EINVAL, "catalogue pointer is NULL");
    if (i_begin > i_end || i_end > n) return acf::fail(ctx, ACF_EINVAL, "row range [%zu, %zu) outside [0, %zu]", i_begin, i_end, n);
    if (n >= (size_t(1) << 31)) return acf::fail(ctx, ACF_EINVAL, "catalogues are limited to 2^31-1 points");
    ACF_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    acf_catalog *cat = new (std::nothrow) acf_catalog();
    if (!cat) return acf::fail(ctx, ACF_ENOMEM, "out of host memory");
    cat->ctx = ctx;
    cat->weighted = d_w != nullptr;
    ctx->last = acf_stats{};  // (acf_get_stats after a preparation: its kernel launches)
    ctx->stats_pending = false;
    int rc = acf::prepare_catalogue(ctx, cat->buf, d_xyz, n, i_begin, i_end - i_begin, d_w, &cat->p);
    if (rc == ACF_OK) {
        cudaError_t e = cudaMemcpyAsync(&ctx->h_verdict[0], &cat->p.pack->bad, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
        if (e != cudaSuccess) rc = acf::fail(ctx, ACF_ECUDA, "acf_prepare: %s", cudaGetErrorString(e));
        else if (ctx->h_verdict[0] != 0)
            rc = acf::fail(ctx, ACF_EINVAL, "%d input points are not finite unit vectors (|r^2 - 1| <= 1e-6) or carry a negative / non-finite weight",
                           ctx->h_verdict[0]);
    }
    if (rc != ACF_OK) {
        cudaStreamSynchronize(ctx->stream);
        cat->buf.release();
        delete cat;
        return rc;
    }
    cat->next = ctx->catalogs;
    if (ctx->catalogs) ctx->catalogs->prev = cat;
    ctx->catalogs = cat;
    ctx->n_catalogs++;
    *out = cat;
    return ACF_OK;
}

extern "C" int acf_prepare_again(acf_ctx *ctx, acf_catalog *cat, const double *d_xyz, const float *d_w, size_t n, size_t i_begin,
                                 size_t i_end)
{
    if (!ctx) return ACF_EINVAL;
    ctx->err[0] = 0;
    if (!cat || cat->ctx != ctx) return acf::fail(ctx, ACF_EINVAL, "catalogue handle is NULL or of another context");
    if (n && !d_xyz) return acf::fail(ctx, ACF_EINVAL, "catalogue pointer is NULL");
    if (i_begin > i_end || i_end > n) return acf::fail(ctx, ACF_EINVAL, "row range [%zu, %zu) outside [0, %zu]", i_begin, i_end, n);
    if (n >= (size_t(1) << 31)) return acf::fail(ctx, ACF_EINVAL, "catalogues are limited to 2^31-1 points");
    ACF_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cat->weighted = d_w != nullptr;
    ctx->last = acf_stats{};  // (acf_get_stats after a preparation: its kernel launches)
    ctx->stats_pending = false;
    int rc = acf::prepare_catalogue(ctx, cat->buf, d_xyz, n, i_begin, i_end - i_begin, d_w, &cat->p);
    if (rc == ACF_OK) {
        cudaError_t e = cudaMemcpyAsync(&ctx->h_verdict[0], &cat->p.pack->bad, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
        if (e != cudaSuccess) rc = acf::fail(ctx, ACF_ECUDA, "acf_prepare: %s", cudaGetErrorString(e));
        else if (ctx->h_verdict[0] != 0)
            rc = acf::fail(ctx, ACF_EINVAL, "%d input points are not finite unit vectors (|r^2 - 1| <= 1e-6) or carry a negative / non-finite weight",
                           ctx->h_verdict[0]);
    }
    if (rc != ACF_OK) {
        cat->p.n = 0;
        cat->p.n_tiles = 0;
    }
    return rc;
}

extern "C" int acf_prepare(acf_ctx *ctx, const double *d_xyz, const float *d_w, size_t n, acf_catalog **out)
{
    return acf_prepare_rows(ctx, d_xyz, d_w, n, 0, n, out);
}

extern "C" void acf_release(acf_ctx *ctx, acf_catalog *cat)
{
    if (!ctx || !cat || cat->ctx != ctx) return;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);  // counts on the handle may still be running
    if (cat->prev) cat->prev->next = cat->next;
    else ctx->catalogs = cat->next;
    if (cat->next) cat->next->prev = cat->prev;
    ctx->n_catalogs--;
    cat->buf.release();
    delete cat;
}

extern "C" int acf_pair_count_prepared(acf_ctx *ctx, const acf_catalog *a, const acf_catalog *b, const double *cos_edges, int nbins,
                                       int part, int n_parts, uint64_t *d_counts, double *d_wsums)
{
    if (!ctx) return ACF_EINVAL;
    ctx->err[0] = 0;
    if (const char *why = check_edges(cos_edges, nbins)) return acf::fail(ctx, ACF_EINVAL, "%s", why);
    if (!a || a->ctx != ctx || (b && b->ctx != ctx)) return acf::fail(ctx, ACF_EINVAL, "catalogue handle is NULL or of another context");
    if (!d_counts) return acf::fail(ctx, ACF_EINVAL, "d_counts is NULL");
    if (n_parts < 1 || part < 0 || part >= n_parts) return acf::fail(ctx, ACF_EINVAL, "part %d of %d", part, n_parts);
    const bool is_auto = b == nullptr || b == a;
    if (is_auto) b = a;
    const bool weighted = d_wsums != nullptr;
    if (weighted && (!a->weighted || !b->weighted)) return acf::fail(ctx, ACF_EINVAL, "weighted count of a catalogue prepared without weights");
    if (ctx->opt_kernel == ACF_KERNEL_FP64) return acf::fail(ctx, ACF_EINVAL, "the fp64 reference kernel counts unprepared catalogues only");
    ACF_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    ctx->last = acf_stats{};
    ctx->pair_timed = false;
    ctx->last.pairs_nominal = is_auto ? (uint64_t)a->p.n * (a->p.n ? a->p.n - 1 : 0) / 2 : (uint64_t)a->p.n * (uint64_t)b->p.n;  // (of all parts)
    ACF_CUDA_TRY(ctx, cudaEventRecord(ctx->ev_start, st));
    ACF_CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_counters, 0, sizeof(unsigned long long) * acf::kNumCounters, st));
    ACF_CUDA_TRY(ctx, cudaMemsetAsync(d_counts, 0, sizeof(uint64_t) * (size_t)nbins, st));
    if (weighted) ACF_CUDA_TRY(ctx, cudaMemsetAsync(d_wsums, 0, sizeof(double) * (size_t)nbins, st));
    ctx->stats_pending = true;
    // a catalogue prepared with weights counts unweighted as well: the kernels then read only its coordinates
    acf::Prepared pa = a->p, pb = b->p;
    int rc = acf::count_prepared_part(ctx, pa, pb, is_auto ? 1 : 0, cos_edges, nbins, part, n_parts,
                                      reinterpret_cast<unsigned long long *>(d_counts), d_wsums);
    if (rc != ACF_OK) return rc;
    ACF_CUDA_TRY(ctx, cudaEventRecord(ctx->ev_stop, st));
    return ACF_OK;
}

// Delete-one jackknife (include/acf.h).  Every region of either catalogue is prepared once; the histograms of all pairs
// of regions -- DD and RR: K (K + 1) / 2 counts each, DR: K^2 -- are counted on the handles into one device array and
// fetched once.  Together they are exactly the pairs of one DD, one DR and one RR count; the full histograms are their
// sums, and the histograms without region k are the full ones minus row and column k.
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
    for (int k = 0; k < n_regions; ++k)
        if (off_d[k + 1] < off_d[k] || off_r[k + 1] < off_r[k]) return acf::fail(ctx, ACF_EINVAL, "region offsets must not decrease");
    if (off_d[0] != 0 || off_r[0] != 0 || off_d[n_regions] != n_d || off_r[n_regions] != n_r)
        return acf::fail(ctx, ACF_EINVAL, "region offsets must run from 0 to n");
    if (ctx->opt_kernel == ACF_KERNEL_FP64) return acf::fail(ctx, ACF_EINVAL, "the jackknife runs on prepared catalogues: not with the fp64 reference kernel");
    ACF_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    const size_t nb = (size_t)nbins, K = (size_t)n_regions;
    std::vector<acf_catalog *> cd(K, nullptr), cr(K, nullptr);
    auto cleanup = [&]() {
        for (size_t k = 0; k < K; ++k) {
            acf_release(ctx, cd[k]);
            acf_release(ctx, cr[k]);
        }
    };
    int rc = ACF_OK;
    for (size_t k = 0; k < K && rc == ACF_OK; ++k) {
        rc = acf_prepare_rows(ctx, d_xyz_d, nullptr, n_d, off_d[k], off_d[k + 1], &cd[k]);
        if (rc == ACF_OK) rc = acf_prepare_rows(ctx, d_xyz_r, nullptr, n_r, off_r[k], off_r[k + 1], &cr[k]);
    }
    // histograms: DD[k][l] (k <= l), DR[k][l], RR[k][l] (k <= l): 3 K^2 slots of nbins
    const size_t slots = 3 * K * K;
    if (rc == ACF_OK && ctx->s_host_stage[4].reserve(sizeof(uint64_t) * slots * nb) != cudaSuccess) rc = acf::fail(ctx, ACF_ENOMEM, "out of device memory");
    uint64_t *d_cnt = ctx->s_host_stage[4].as<uint64_t>();
    if (rc == ACF_OK && cudaMemsetAsync(d_cnt, 0, sizeof(uint64_t) * slots * nb, st) != cudaSuccess) rc = acf::fail(ctx, ACF_ECUDA, "memset failed");
    unsigned long long launches = 0;
    for (size_t k = 0; k < K && rc == ACF_OK; ++k)
        for (size_t l = 0; l < K && rc == ACF_OK; ++l) {
            if (l >= k) {
                rc = acf_pair_count_prepared(ctx, cd[k], l == k ? nullptr : cd[l], cos_edges, nbins, 0, 1, d_cnt + (k * K + l) * nb, nullptr);
                launches += ctx->last.kernel_launches;
                if (rc == ACF_OK) rc = acf_pair_count_prepared(ctx, cr[k], l == k ? nullptr : cr[l], cos_edges, nbins, 0, 1, d_cnt + ((2 * K + k) * K + l) * nb, nullptr);
                launches += ctx->last.kernel_launches;
            }
            if (rc == ACF_OK) rc = acf_pair_count_prepared(ctx, cd[k], cr[l], cos_edges, nbins, 0, 1, d_cnt + ((K + k) * K + l) * nb, nullptr);
            launches += ctx->last.kernel_launches;
        }
    std::vector<uint64_t> h(slots * nb);
    if (rc == ACF_OK) {
        cudaError_t e = cudaMemcpyAsync(h.data(), d_cnt, sizeof(uint64_t) * slots * nb, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) rc = acf::fail(ctx, ACF_ECUDA, "acf_jackknife: %s", cudaGetErrorString(e));
    }
    cleanup();
    if (rc != ACF_OK) return rc;
    ctx->last.kernel_launches = launches;

    // totals, and per region the pairs that touch it
    std::vector<uint64_t> tot(3 * nb, 0), touch(3 * K * nb, 0), dd(nb), dr(nb), rr(nb);
    for (size_t k = 0; k < K; ++k)
        for (size_t l = 0; l < K; ++l)
            for (size_t b = 0; b < nb; ++b) {
                const uint64_t vdd = l >= k ? h[(k * K + l) * nb + b] : 0, vrr = l >= k ? h[((2 * K + k) * K + l) * nb + b] : 0;
                const uint64_t vdr = h[((K + k) * K + l) * nb + b];
                tot[b] += vdd;
                tot[nb + b] += vdr;
                tot[2 * nb + b] += vrr;
                // a pair of regions (k, l) touches k and l; DR[k][l] touches data region k and random region l
                touch[k * nb + b] += vdd;
                if (l != k) touch[l * nb + b] += vdd;
                touch[(2 * K + k) * nb + b] += vrr;
                if (l != k) touch[(2 * K + l) * nb + b] += vrr;
                touch[(K + k) * nb + b] += vdr;
                if (l != k) touch[(K + l) * nb + b] += vdr;
            }
    if ((rc = acf_estimator(estimator, tot.data(), tot.data() + nb, tot.data() + 2 * nb, n_d, n_r, nbins, w_full)) != ACF_OK) return rc;
    for (size_t k = 0; k < K; ++k) {
        const size_t ndk = off_d[k + 1] - off_d[k], nrk = off_r[k + 1] - off_r[k];
        for (size_t b = 0; b < nb; ++b) {
            dd[b] = tot[b] - touch[k * nb + b];
            dr[b] = tot[nb + b] - touch[(K + k) * nb + b];
            rr[b] = tot[2 * nb + b] - touch[(2 * K + k) * nb + b];
        }
        if ((rc = acf_estimator(estimator, dd.data(), dr.data(), rr.data(), n_d - ndk, n_r - nrk, nbins, w_jk + k * nb)) != ACF_OK) return rc;
    }
    if (cov) {
        std::vector<double> mean(nb, 0.0);
        for (size_t k = 0; k < K; ++k)
            for (size_t b = 0; b < nb; ++b) mean[b] += w_jk[k * nb + b];
        for (size_t b = 0; b < nb; ++b) mean[b] /= (double)n_regions;
        const double f = (double)(n_regions - 1) / (double)n_regions;
        for (size_t a = 0; a < nb; ++a)
            for (size_t b = 0; b < nb; ++b) {
                double sum = 0.0;
                for (size_t k = 0; k < K; ++k) sum += (w_jk[k * nb + a] - mean[a]) * (w_jk[k * nb + b] - mean[b]);
                cov[a * nb + b] = f * sum;
            }
    }
    return ACF_OK;
}

// Monte-Carlo errors from an ensemble of random catalogues (include/acf.h).
extern "C" int acf_random_ensemble(acf_ctx *ctx, const acf_catalog *data, const double *const *d_xyz_r, const size_t *n_r, int n_random,
                                   const double *cos_edges, int nbins, int estimator, uint64_t *dd, uint64_t *dr, uint64_t *rr,
                                   double *w, double *mean, double *cov)
{
    if (!ctx) return ACF_EINVAL;
    ctx->err[0] = 0;
    if (const char *why = check_edges(cos_edges, nbins)) return acf::fail(ctx, ACF_EINVAL, "%s", why);
    if (!data || data->ctx != ctx) return acf::fail(ctx, ACF_EINVAL, "catalogue handle is NULL or of another context");
    if (n_random < 1 || !d_xyz_r || !n_r || !dd || !dr || !rr || !w) return acf::fail(ctx, ACF_EINVAL, "NULL argument or no random catalogue");
    if (cov && n_random < 2) return acf::fail(ctx, ACF_EINVAL, "a covariance needs at least two random catalogues");
    if (estimator < ACF_EST_LANDY_SZALAY || estimator > ACF_EST_HAMILTON) return acf::fail(ctx, ACF_EINVAL, "unknown estimator");
    if (ctx->opt_kernel == ACF_KERNEL_FP64) return acf::fail(ctx, ACF_EINVAL, "the ensemble runs on prepared catalogues: not with the fp64 reference kernel");
    for (int k = 0; k < n_random; ++k) {
        if (n_r[k] && !d_xyz_r[k]) return acf::fail(ctx, ACF_EINVAL, "random catalogue %d is NULL", k);
        if (n_r[k] >= (size_t(1) << 31)) return acf::fail(ctx, ACF_EINVAL, "catalogues are limited to 2^31-1 points");
    }
    ACF_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    const size_t nb = (size_t)nbins, K = (size_t)n_random;
    // device: DD, then DR_k and RR_k; pinned host: the same, then the verdicts
    ACF_CUDA_TRY(ctx, ctx->s_host_stage[4].reserve(sizeof(uint64_t) * (2 * K + 1) * nb));
    uint64_t *d_cnt = ctx->s_host_stage[4].as<uint64_t>();
    const size_t host_bytes = sizeof(uint64_t) * (2 * K + 1) * nb + sizeof(int) * K;
    if (ctx->h_stage_bytes < host_bytes) {
        if (ctx->h_stage) cudaFreeHost(ctx->h_stage);
        ctx->h_stage = nullptr;
        ctx->h_stage_bytes = 0;
        ACF_CUDA_TRY(ctx, cudaHostAlloc(&ctx->h_stage, host_bytes, cudaHostAllocDefault));
        ctx->h_stage_bytes = host_bytes;
    }
    uint64_t *h_cnt = static_cast<uint64_t *>(ctx->h_stage);
    int *h_bad = reinterpret_cast<int *>(h_cnt + (2 * K + 1) * nb);
    // two internal handles, used in turn: the preparation of catalogue k + 1 is enqueued behind the counts of catalogue k
    // (one stream: the buffers of a handle are free again when its counts have run)
    acf_catalog ring[2];
    ring[0].ctx = ring[1].ctx = ctx;
    unsigned long long launches = 0;
    int rc = acf_pair_count_prepared(ctx, data, nullptr, cos_edges, nbins, 0, 1, d_cnt, nullptr);
    launches += ctx->last.kernel_launches;
    for (size_t k = 0; k < K && rc == ACF_OK; ++k) {
        acf_catalog &c = ring[k & 1];
        ctx->last = acf_stats{};
        rc = acf::prepare_catalogue(ctx, c.buf, d_xyz_r[k], n_r[k], 0, n_r[k], nullptr, &c.p);
        launches += ctx->last.kernel_launches;
        if (rc != ACF_OK) break;
        if (cudaMemcpyAsync(&h_bad[k], &c.p.pack->bad, sizeof(int), cudaMemcpyDeviceToHost, st) != cudaSuccess) {
            rc = acf::fail(ctx, ACF_ECUDA, "copy of the verdict failed");
            break;
        }
        rc = acf_pair_count_prepared(ctx, data, &c, cos_edges, nbins, 0, 1, d_cnt + (1 + k) * nb, nullptr);
        launches += ctx->last.kernel_launches;
        if (rc == ACF_OK) rc = acf_pair_count_prepared(ctx, &c, nullptr, cos_edges, nbins, 0, 1, d_cnt + (1 + K + k) * nb, nullptr);
        launches += ctx->last.kernel_launches;
    }
    if (rc == ACF_OK) {
        cudaError_t e = cudaMemcpyAsync(h_cnt, d_cnt, sizeof(uint64_t) * (2 * K + 1) * nb, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) rc = acf::fail(ctx, ACF_ECUDA, "acf_random_ensemble: %s", cudaGetErrorString(e));
    } else {
        cudaStreamSynchronize(st);
    }
    ring[0].buf.release();
    ring[1].buf.release();
    if (rc != ACF_OK) return rc;
    ctx->last.kernel_launches = launches;
    for (size_t k = 0; k < K; ++k)
        if (h_bad[k] != 0)
            return acf::fail(ctx, ACF_EINVAL, "random catalogue %zu: %d points are not finite unit vectors (|r^2 - 1| <= 1e-6)", k, h_bad[k]);
    memcpy(dd, h_cnt, sizeof(uint64_t) * nb);
    memcpy(dr, h_cnt + nb, sizeof(uint64_t) * K * nb);
    memcpy(rr, h_cnt + (1 + K) * nb, sizeof(uint64_t) * K * nb);
    for (size_t k = 0; k < K; ++k)
        if ((rc = acf_estimator(estimator, dd, dr + k * nb, rr + k * nb, data->p.n, n_r[k], nbins, w + k * nb)) != ACF_OK) return rc;
    if (mean || cov) {
        std::vector<double> m(nb, 0.0);
        for (size_t k = 0; k < K; ++k)
            for (size_t b = 0; b < nb; ++b) m[b] += w[k * nb + b];
        for (size_t b = 0; b < nb; ++b) m[b] /= (double)K;
        if (mean) memcpy(mean, m.data(), sizeof(double) * nb);
        if (cov)
            for (size_t a = 0; a < nb; ++a)
                for (size_t b = 0; b < nb; ++b) {
                    double sum = 0.0;
                    for (size_t k = 0; k < K; ++k) sum += (w[k * nb + a] - m[a]) * (w[k * nb + b] - m[b]);
                    cov[a * nb + b] = sum / (double)(K - 1);
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

    // pinned staging: xyz of both catalogues, their weights, then the outputs
    const size_t xyz_bytes = sizeof(double) * 3 * (n_d + n_r);
    const size_t w_bytes = weighted ? ((sizeof(float) * (n_d + n_r) + 15) & ~size_t(15)) : 0;
    const size_t out_bytes = (sizeof(uint64_t) + sizeof(double)) * 3 * (size_t)nbins;
    if (ctx->h_stage_bytes < xyz_bytes + w_bytes + out_bytes) {
        if (ctx->h_stage) cudaFreeHost(ctx->h_stage);
        ctx->h_stage = nullptr;
        ctx->h_stage_bytes = 0;
        ACF_CUDA_TRY(ctx, cudaHostAlloc(&ctx->h_stage, xyz_bytes + w_bytes + out_bytes, cudaHostAllocDefault));
        ctx->h_stage_bytes = xyz_bytes + w_bytes + out_bytes;
    }
    double *h_xyz_d = static_cast<double *>(ctx->h_stage), *h_xyz_r = h_xyz_d + 3 * n_d;
    float *h_wd = reinterpret_cast<float *>(h_xyz_r + 3 * n_r), *h_wr = h_wd + n_d;
    uint64_t *h_cnt = reinterpret_cast<uint64_t *>(reinterpret_cast<char *>(h_wd) + w_bytes);
    double *h_ws = reinterpret_cast<double *>(h_cnt + 3 * (size_t)nbins);

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

    // The data: canonicalise, copy, prepare, and start DD.  The randoms are canonicalised on the host and copied on a
    // second stream while the device counts DD (PAPER.md:128 names the overlap of transfers and kernels as the step the
    // paper's own code did not take); the main stream waits for that copy before it touches them.
    acf_radec_to_xyz(ra_d, dec_d, n_d, h_xyz_d);
    if (weighted && n_d) memcpy(h_wd, w_d, sizeof(float) * n_d);
    if (n_d) ACF_CUDA_TRY(ctx, cudaMemcpyAsync(d_xd, h_xyz_d, sizeof(double) * 3 * n_d, cudaMemcpyHostToDevice, st));
    if (weighted && n_d) ACF_CUDA_TRY(ctx, cudaMemcpyAsync(d_wd, h_wd, sizeof(float) * n_d, cudaMemcpyHostToDevice, st));
    // the two handles live with the context: prepared again on every call, their device memory reused
    auto prepare = [&](int k, const double *x, const float *wt, size_t n) -> int {
        if (!ctx->e2e_cat[k]) return acf_prepare(ctx, x, wt, n, &ctx->e2e_cat[k]);
        return acf_prepare_again(ctx, ctx->e2e_cat[k], x, wt, n, 0, n);
    };
    int rc = prepare(0, d_xd, d_wd, n_d);
    if (rc != ACF_OK) return rc;
    acf_catalog *&cd = ctx->e2e_cat[0], *&cr = ctx->e2e_cat[1];
    auto bail = [&](int code) {
        cudaStreamSynchronize(ctx->copy_stream);
        cudaStreamSynchronize(st);
        return code;
    };
    acf_stats st_sum{};
    auto add_stats = [&]() {
        st_sum.pairs_nominal += ctx->last.pairs_nominal;
        st_sum.kernel_launches += ctx->last.kernel_launches;
    };
    rc = acf_pair_count_prepared(ctx, cd, nullptr, cos_edges, nbins, 0, 1, d_cnt, d_ws);
    if (rc != ACF_OK) return bail(rc);
    add_stats();
    acf_radec_to_xyz(ra_r, dec_r, n_r, h_xyz_r);
    if (weighted && n_r) memcpy(h_wr, w_r, sizeof(float) * n_r);
    if (n_r) ACF_CUDA_TRY(ctx, cudaMemcpyAsync(d_xr, h_xyz_r, sizeof(double) * 3 * n_r, cudaMemcpyHostToDevice, ctx->copy_stream));
    if (weighted && n_r) ACF_CUDA_TRY(ctx, cudaMemcpyAsync(d_wr, h_wr, sizeof(float) * n_r, cudaMemcpyHostToDevice, ctx->copy_stream));
    ACF_CUDA_TRY(ctx, cudaEventRecord(ctx->ev_copy, ctx->copy_stream));
    ACF_CUDA_TRY(ctx, cudaStreamWaitEvent(st, ctx->ev_copy, 0));
    rc = prepare(1, d_xr, d_wr, n_r);
    if (rc != ACF_OK) return bail(rc);
    rc = acf_pair_count_prepared(ctx, cd, cr, cos_edges, nbins, 0, 1, d_cnt + nbins, d_ws ? d_ws + nbins : nullptr);
    if (rc != ACF_OK) return bail(rc);
    add_stats();
    rc = acf_pair_count_prepared(ctx, cr, nullptr, cos_edges, nbins, 0, 1, d_cnt + 2 * nbins, d_ws ? d_ws + 2 * nbins : nullptr);
    if (rc != ACF_OK) return bail(rc);
    add_stats();

    ACF_CUDA_TRY(ctx, cudaMemcpyAsync(h_cnt, d_cnt, sizeof(uint64_t) * 3 * (size_t)nbins, cudaMemcpyDeviceToHost, st));
    if (weighted) ACF_CUDA_TRY(ctx, cudaMemcpyAsync(h_ws, d_ws, sizeof(double) * 3 * (size_t)nbins, cudaMemcpyDeviceToHost, st));
    {
        const cudaError_t e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) return acf::fail(ctx, ACF_ECUDA, "acf_correlate_host: %s", cudaGetErrorString(e));
        ctx->last.pairs_nominal = st_sum.pairs_nominal;
        ctx->last.kernel_launches = st_sum.kernel_launches;
    }
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
