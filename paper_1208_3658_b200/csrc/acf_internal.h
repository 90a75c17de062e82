// acf_internal.h -- context, scratch buffers and kernel entry points shared by the .cu files
// of libacf.  Nothing here is visible through the C ABI (include/acf.h).
#pragma once

#include <cuda_runtime.h>

#include <cstdarg>
#include <cstddef>
#include <cstdint>
#include <cstdio>

#include "acf.h"

namespace acf {

// Device buffer that only ever grows; owned by the context.
struct Scratch {
    void *ptr = nullptr;
    size_t bytes = 0;
    cudaError_t reserve(size_t want)
    {
        if (want <= bytes) return cudaSuccess;
        if (ptr) cudaFree(ptr);
        ptr = nullptr;
        bytes = 0;
        size_t rounded = (want + 255) & ~size_t(255);
        cudaError_t e = cudaMalloc(&ptr, rounded);
        if (e == cudaSuccess) bytes = rounded;
        return e;
    }
    void release()
    {
        if (ptr) cudaFree(ptr);
        ptr = nullptr;
        bytes = 0;
    }
    template <class T>
    T *as() const
    {
        return static_cast<T *>(ptr);
    }
};

// Device-side counters of one call (ACF_OPT_STATS).  Indexes into ctx->d_counters.
enum Counter : int {
    kCtrPairsEvaluated = 0,
    kCtrPairsFp64 = 1,
    kCtrTilePairsTotal = 2,
    kCtrTilePairsPruned = 3,
    kCtrBadInput = 4,   // number of points that failed validation
    kCtrWorkHead = 5,   // persistent-kernel work counter
    kCtrWorkCount = 6,  // number of work items produced on the device
    kCtrPairsWindow = 7,  // pairs classified by the single-edge window path
    kCtrNormDev = 8,      // max over the validated points of |x^2 + y^2 + z^2 - 1|, as the bits of a double
    kCtrPairsChord = 9,   // pairs the fp32 cosine left open and the fp32 chord length decided
    kCtrPairsBulk = 10,   // pairs counted per group of points, not one by one (ACF_OPT_BULK)
    kNumCounters = 11
};

constexpr int kTile = 1024;      // points per tile (both the register-resident i side and the staged j side)
constexpr int kItemTiles = 8;    // at most this many consecutive j-tiles per work item
constexpr int kGroup = 128;      // points per group: a warp's i-points, and the j-points of one window
constexpr int kGroupsPerTile = kTile / kGroup;
constexpr int kSub = 32;         // points per sub-group: the finer caps a window of several edges is split by
constexpr int kSubsPerGroup = kGroup / kSub;

// Bounding cap of one group of kGroup (or sub-group of kSub) consecutive sorted points, in double: every
// point p of the group has centre . p / |p| >= cos_r (a bound on the directions; the points' norms may be
// off 1 by the 1e-6 the validation accepts).  sin_r = sqrt(1 - cos_r^2); wsum = sum of the group's weights.
// A group without points has cos_r = 2.
struct GroupCap {
    double cx, cy, cz, cos_r, sin_r, wsum;
};

// How the window path tallies a catalogue's weights when it is the j side (written on the device by
// the gather kernel from the weight range).  vj[s] = C + w_s when packed: count and weight sum of the
// pairs above an edge share one fp64 accumulator, sum = n * C + sum of w, exact while
// exponent(w_max) - exponent(w_min > 0) <= 13.  Rows are then differences of exact cumulative sums.
// Weights of a wider range do not pack (vj[s] = w_s): their cumulative sums would round at the size of
// the largest weights and a sparsely filled row would inherit that error, so such calls take the table
// path for every pair, which adds each w_i w_j to its row directly (acf_pair.cu).
struct PackInfo {
    double C, inv_C;
    int packed;
    int bad;     // points of the catalogue that failed validation (validate_kernel): its counts are refused
    double eps;  // max over the catalogue's points of | |u|^2 - 1 | (what the chord margins and the cap slack are made of)
};

// One catalogue prepared for the fast path (all device pointers live in ctx scratch).
struct Prepared {
    const double *xyz = nullptr;  // caller's canonical fp64 SoA (not owned)
    const float *w = nullptr;     // caller's weights or nullptr
    size_t stride = 0;            // points in the caller's catalogue (SoA stride)
    size_t n = 0;                 // points prepared
    float4 *pts = nullptr;        // spatially sorted fp32 {x, y, z, w}; padded to a tile multiple
    float *pts2 = nullptr;        // the same points, two by two: {x0, x1, y0, y1, z0, z1, w0, w1} (the staged j side)
    double *vj = nullptr;         // per sorted point: C + w or w (see PackInfo); padded like pts
    PackInfo *pack = nullptr;
    uint32_t *perm = nullptr;     // sorted position -> original index
    double4 *caps = nullptr;      // per tile: unit centre (x, y, z) and cos of the bounding radius
    GroupCap *gcaps = nullptr;    // per group of kGroup points (kGroupsPerTile per tile)
    GroupCap *scaps = nullptr;    // per sub-group of kSub points (kSubsPerGroup per group)
    int n_tiles = 0;
};

// The device buffers of one prepared catalogue (grown lazily, freed with their owner: the context's two slots of
// the calls that prepare on the fly, or an acf_catalog handle).
struct CatBuffers {
    Scratch slab;  // one allocation, carved up by prepare_catalogue
    void release() { slab.release(); }
};

}  // namespace acf

struct acf_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    int num_sms = 0;
    int max_smem_optin = 0;
    char err[512] = {0};

    int opt_kernel = ACF_KERNEL_AUTO;
    int opt_prune = 1;
    int opt_stats = 1;
    int opt_windows = 1;
    int opt_bulk = 0;

    cudaEvent_t ev_start = nullptr, ev_stop = nullptr, ev_flag = nullptr;
    cudaEvent_t ev_k0 = nullptr, ev_k1 = nullptr;  // around the pair kernel(s) of the last call
    bool pair_timed = false;
    unsigned long long *d_counters = nullptr;  // acf::kNumCounters
    unsigned long long *h_counters = nullptr;  // pinned mirror
    int *h_verdict = nullptr;                  // pinned (behind h_counters): bad-point counts of the catalogues of a call
    acf_stats last{};
    bool stats_pending = false;

    // scratch, grown lazily
    acf::Scratch s_edges;            // device copy of cos_edges (+ fp32 tables of the fast path)
    const float *d_sedges = nullptr; // inside s_edges: the edges as squared chord lengths (chord tier)
    acf::CatBuffers cat[2];          // catalogues a / b of the calls that prepare on the fly
    acf::Scratch s_keys;             // sort keys and indices (double-buffered inside): scratch of a preparation
    acf::Scratch s_work;             // work list
    acf::Scratch s_misc;             // radix-sort histograms etc.
    acf::Scratch s_host_stage[6];    // acf_correlate_host: device copies of xyz / weights / outputs
    void *h_stage = nullptr;         // acf_correlate_host: pinned host staging
    size_t h_stage_bytes = 0;
    void *h_tables = nullptr;        // pinned staging of the per-call tables (edges, chord edges, cell table)
    size_t h_tables_bytes = 0;
    cudaEvent_t ev_tables = nullptr; // the last copy out of h_tables
    cudaStream_t copy_stream = nullptr;  // acf_correlate_host: host-to-device copies that overlap the counts
    cudaEvent_t ev_copy = nullptr;
    struct acf_catalog *e2e_cat[2] = {nullptr, nullptr};  // acf_correlate_host: its two handles, kept between calls (no cudaMalloc / cudaFree per call)
    int n_catalogs = 0;              // acf_catalog handles alive (acf_destroy refuses to leave them dangling: it frees them)
    struct acf_catalog *catalogs = nullptr;  // intrusive list of the handles
};

// A catalogue prepared once for any number of counts (include/acf.h: acf_prepare).
struct acf_catalog {
    acf_ctx *ctx = nullptr;
    acf::Prepared p;
    acf::CatBuffers buf;
    bool weighted = false;
    acf_catalog *next = nullptr, *prev = nullptr;
};

namespace acf {

inline int fail(acf_ctx *ctx, int code, const char *fmt, ...)
{
    if (ctx) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(ctx->err, sizeof(ctx->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

#define ACF_CUDA_TRY(ctx, expr)                                                                   \
    do {                                                                                          \
        cudaError_t _e = (expr);                                                                  \
        if (_e != cudaSuccess)                                                                    \
            return acf::fail((ctx), _e == cudaErrorMemoryAllocation ? ACF_ENOMEM : ACF_ECUDA,     \
                             "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), __FILE__,    \
                             __LINE__);                                                           \
    } while (0)

// ---- kernels_ref.cu: the definition, one pair at a time, in double -------------------------
// Adds into d_counts / d_wsums (which the caller has zeroed).  Rows [i_begin, i_end) of a.
cudaError_t launch_pair_count_fp64(acf_ctx *ctx, const double *d_a, const float *d_wa, size_t n_a,
                                   size_t i_begin, size_t i_end, const double *d_b, const float *d_wb,
                                   size_t n_b, const double *d_edges, int nbins, int is_auto,
                                   unsigned long long *d_counts, double *d_wsums);

// ---- acf_pair.cu: the fast path (prep + fp32-certify pair kernel).  Enqueues everything needed
// to add the counts of rows [i_begin, i_end) into d_counts / d_wsums.  Returns an ACF_* code.
int run_pair_count_fast(acf_ctx *ctx, const double *d_a, const float *d_wa, size_t n_a, size_t i_begin,
                        size_t i_end, const double *d_b, const float *d_wb, size_t n_b, const double *h_edges,
                        int nbins, int is_auto, unsigned long long *d_counts, double *d_wsums);

// ---- acf_pair_win.cu: the window kernel on the work items already in ctx->s_work (edges in ctx->s_edges).
int launch_pair_win(acf_ctx *ctx, const Prepared &a, const Prepared &b, int is_auto, const double *h_edges, int nbins, uint32_t capacity,
                    unsigned long long *d_counts, double *d_wsums);

// ---- acf_prep.cu: sort + gather + caps of points [off, off+cnt) of a catalogue with `stride` points;
// and the work list of (i-tile, j-tile run) items for i-tiles [ti_begin, ti_end).
// Validation (finite unit vectors, finite non-negative weights) is part of it: the verdict and the largest norm
// deviation land in the catalogue's PackInfo.
int prepare_catalogue(acf_ctx *ctx, CatBuffers &buf, const double *xyz, size_t stride, size_t off, size_t cnt,
                      const float *w, Prepared *out);
// i-tiles ti_begin + k * ti_stride < ti_end.
int build_worklist(acf_ctx *ctx, const Prepared &a, int ti_begin, int ti_end, int ti_stride, const Prepared &b, int is_auto,
                   double e_first, double e_last, int3 *items, uint32_t capacity);

// Validates points [off, off + cnt) of a catalogue with `stride` points (unit vectors, weights): pack->bad = number of
// bad points, pack->eps = max | |u|^2 - 1 |.
cudaError_t launch_validate(acf_ctx *ctx, const double *d_xyz, size_t stride, size_t off, size_t cnt, const float *d_w, PackInfo *pack);

// ---- acf_pair.cu: the counts of part `part` of `n_parts` (i-tiles t = part mod n_parts) of prepared a against prepared b,
// added into d_counts / d_wsums.  Enqueues only.
int count_prepared_part(acf_ctx *ctx, const Prepared &a, const Prepared &b, int is_auto, const double *h_edges, int nbins,
                        int part, int n_parts, unsigned long long *d_counts, double *d_wsums);

}  // namespace acf
