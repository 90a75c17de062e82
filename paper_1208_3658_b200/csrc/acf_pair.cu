// acf_pair.cu -- the fast path of acf_pair_count*: fp32 pair cosine with certified binning,
// fp64 re-check of every pair the fp32 test cannot certify.
//
// Per pair ("most of their time actually calculating the angular separations"):
//   t32 = K - (x_i x_j + y_i y_j + z_i z_j)   three fp32 FMAs; K = 1 + 2^-18 keeps t32 > 0
//   cell = float bits of t32 >> (23 - m)       log-spaced cells, 2^m per octave of t
//   {thr, row} = LUT[cell]                     the one bin edge (as K - e) that can matter in the cell
//   row += (t32 > thr)                         histogram row: 0 = closer than theta_min, 1..nbins = bins,
//                                              nbins+1 = beyond theta_max (dropped)
//   certified iff |t32 - thr| > G              G bounds |t32 - (K - c64)| + rounding of thr
// A pair that is not certified is re-evaluated exactly as include/acf.h defines it (fp64 fma
// chain on the caller's doubles, clamp, exact edge search) and the histogram is corrected, so
// the counts equal the fp64 definition whatever the fp32 arithmetic did.
//
// Window path.  Points are sorted along a space-filling curve, so the kGroup i-points of a warp and a
// group of kGroup staged j-points each sit in a small cap, and all their pair cosines lie in a window
// [c_lo, c_hi] known from the two caps.  When that window holds at most one bin edge e_m, every pair
// is classified against that single edge, held in a uniform register:
//   d32 = e_m - (x_i x_j + y_i y_j + z_i z_j)  three fp32 FMAs seeded with fp32(e_m)
//   above = d32 > 0                             row m + above
//   certified iff |d32| > G1                    else the exact fp64 row replaces it, as above
// and the tallies (count of `above`, sum of w_j over `above` per i-point) stay in registers until the
// group is done.  Windows with two or more edges, ragged groups and diagonal tiles take the table path.
//
// Histograms are privatised per lane in shared memory (row-major [row][lane]: a lane owns a bank,
// so updates never conflict and need no ordering -- PAPER.md:86 reports 5-50 % loss to atomic
// serialisation), summed per warp with shuffles and flushed with global u64 / f64 atomics.
// j-tiles are staged with cp.async.bulk (TMA, mbarrier completion) into a double buffer while
// each thread holds kR i-points in registers.  Auto-correlations visit the upper triangle only.
#include <cmath>
#include <cstring>
#include <limits>
#include <vector>

#include "acf_device.cuh"
#include "acf_internal.h"
#include "acf_pair_common.cuh"

namespace acf {

namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kR = kTile / kThreads;  // i-points per thread
constexpr float kK = 1.0f + 0x1p-18f;
// |t32 - (K - c64)| <= 2u(1+1e-6) [input rounding, u = 2^-24] + 3 * 2^-23 [three roundings of values < 4]
// = 4.77e-7; thr is K - e rounded to fp32: another 2^-23 at most.
constexpr float kDelta = 5.5e-7f;
constexpr float kGuard = kDelta + 0x1p-23f;
constexpr int kExpLo = -19;  // t32 >= K - (1 + 1e-6) - kDelta > 2^-19
constexpr int kExpHi = 2;    // t32 < 4
constexpr int kMaxPrivateRows = 64;
// Window path: |d32 - (e_m - c64)| <= 2^-25 [fp32(e_m)] + 2u(1+1e-6) [input rounding] + 3 * 2^-24
// [three roundings of values of magnitude <= 2] = 3.3e-7.
constexpr float kGuardWin = 4.5e-7f;
constexpr int kWinUnroll = 4;  // j-points per guard-band vote
static_assert(kGroup == kR * 32, "a warp's i-points are one group");
static_assert(kGroup % kWinUnroll == 0, "");

struct PairParams {
    const float4 *pts_a;
    const float *pts2_b;    // j side, two points per record {x0, x1, y0, y1, z0, z1, w0, w1}
    const double *vj_b;     // j side window-path weights (PackInfo)
    const PackInfo *pack_b;
    const uint32_t *perm_a, *perm_b;
    const GroupCap *gcaps_a, *gcaps_b;
    uint32_t n_a, n_b;
    const double *xyz_a, *xyz_b;
    size_t stride_a, stride_b;
    const int3 *items;
    uint32_t capacity;
    const uint2 *lut;
    int lut_len, key0, shift;
    const double *edges;
    const float *sedges;   // the edges as squared chord lengths (chord_row)
    float chord_margin;    // filled in by the kernel from the validation result
    int nbins;
    unsigned long long *counts;
    double *wsums;
    unsigned long long *counters;
    int is_auto;
    int use_windows;
    int only_unpackable;  // 1: run only if the j side's weights do not pack (the window kernel ran otherwise)
    int prune;
    int n_stages;
};

template <bool kWeighted, bool kPrivate>
struct Hist {
    uint32_t *cnt;  // private: this warp's [rows][32]; shared: the CTA's [rows]
    double *ws;     // same shapes (weighted only)
    int lane;
    __device__ __forceinline__ void add(uint32_t row)
    {
        if constexpr (kPrivate) atomicAdd(&cnt[row * 32 + lane], 1u);  // own bank: conflict-free, result unused -> RED
        else atomicAdd(&cnt[row], 1u);
    }
    __device__ __forceinline__ void add_w(uint32_t row, double w)
    {
        if constexpr (kPrivate) ws[row * 32 + lane] += w;  // the lane owns the word: plain read-modify-write
        else atomicAdd(&ws[row], w);
    }
    __device__ __forceinline__ void add_n(uint32_t row, uint32_t n)
    {
        if constexpr (kPrivate) cnt[row * 32 + lane] += n;
        else atomicAdd(&cnt[row], n);
    }
    __device__ __forceinline__ void move(uint32_t from, uint32_t to)
    {
        if constexpr (kPrivate) {
            cnt[from * 32 + lane] -= 1u;
            cnt[to * 32 + lane] += 1u;
        } else {
            atomicSub(&cnt[from], 1u);
            atomicAdd(&cnt[to], 1u);
        }
    }
};

// One j-tile against the kR register-resident i-points of every thread.
// kMasked: pairs are individually enabled (ragged last i-tile, or the diagonal tile of an auto count
// where only j > i is counted).
// Thread (warp, lane) holds the i-points warp * kGroup + r * 32 + lane of the i-tile, r < kR.
__device__ __forceinline__ uint32_t local_i(int r) { return (threadIdx.x >> 5) * kGroup + r * 32 + (threadIdx.x & 31); }

// Table path: j-points [jj0, jj0 + jn) of the staged tile against the kR register-resident i-points.
template <bool kWeighted, bool kPrivate, bool kMasked>
__device__ __forceinline__ void process_tile(const PairParams &p, Hist<kWeighted, kPrivate> &h, const float *__restrict__ tile2,
                                             int jj0, int jn, const unsigned long long (&nx2)[kR], const unsigned long long (&ny2)[kR], const unsigned long long (&nz2)[kR],
                                             const float (&wi)[kR], const uint2 *__restrict__ lut, uint32_t i_base,
                                             uint32_t j_base, bool diag, uint32_t valid_mask, unsigned long long &n_fp64)
{
    const int shift = p.shift, key0 = p.key0;
#pragma unroll 2
    for (int jj = jj0; jj < jj0 + jn; ++jj) {
        const float4 q = tile_point(tile2, jj);
        bool amb_any = false;
        bool amb[kR];
        uint32_t row[kR];
#pragma unroll
        for (int r = 0; r < kR; ++r) {
            const float t = fmaf(__uint_as_float((uint32_t)nx2[r]), q.x,
                                 fmaf(__uint_as_float((uint32_t)ny2[r]), q.y, fmaf(__uint_as_float((uint32_t)nz2[r]), q.z, kK)));
            const uint2 e = lut[(int)(__float_as_uint(t) >> shift) - key0];
            const float thr = __uint_as_float(e.x);
            row[r] = e.y + (t > thr ? 1u : 0u);
            amb[r] = !(fabsf(t - thr) > kGuard);  // also true for the NaN threshold of a crowded cell
            if constexpr (kMasked) {
                const bool on = ((valid_mask >> r) & 1u) && (!diag || (uint32_t)jj > local_i(r));
                amb[r] = amb[r] && on;
                if (on) h.add(row[r]);
                if constexpr (kWeighted)
                    if (on && !amb[r]) h.add_w(row[r], (double)wi[r] * (double)q.w);
            } else {
                h.add(row[r]);
                if constexpr (kWeighted)
                    if (!amb[r]) h.add_w(row[r], (double)wi[r] * (double)q.w);
            }
            amb_any |= amb[r];
        }
        if (__any_sync(0xffffffffu, amb_any)) {
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                if (amb[r]) {
                    // the chord length decides where the cosine could not; what it leaves open, the definition
                    int exact = chord_row(-__uint_as_float((uint32_t)nx2[r]), -__uint_as_float((uint32_t)ny2[r]),
                                          -__uint_as_float((uint32_t)nz2[r]), q.x, q.y, q.z, p.sedges, p.nbins, p.chord_margin);
                    if (exact < 0) {
                        exact = exact_row(p.xyz_a, p.stride_a, p.perm_a[i_base + local_i(r)], p.xyz_b, p.stride_b,
                                          p.perm_b[j_base + jj], p.edges, p.nbins);
                        ++n_fp64;
                    } else {
                        n_fp64 += 1ull << 32;  // high word: pairs the chord tier decided
                    }
                    if ((uint32_t)exact != row[r]) h.move(row[r], (uint32_t)exact);
                    if constexpr (kWeighted) h.add_w((uint32_t)exact, (double)wi[r] * (double)q.w);
                }
            }
        }
    }
}

// ---- window path --------------------------------------------------------------------------------
struct Window {
    int edge;    // m: the one edge pairs of this window are tested against; -1: take the table path;
                 // -2: every pair of the window is out of range: nothing to evaluate
    float e32;   // fp32(e[m])
    double wsum; // sum of the j-group's weights
};

// All pairs between points of cap a and cap b have c_lo <= cos(theta) <= c_hi; the window is usable
// when rows(c_lo) - rows(c_hi) <= 1.  theta = angle between the centres, rho = sum of the radii:
// cos(theta -+ rho) = cos(theta) cos(rho) +- sin(theta) sin(rho), clamped at the poles.
__device__ __forceinline__ Window make_window(const GroupCap &a, const GroupCap &b, const double *__restrict__ edges, int nbins,
                                              bool prune, double slack)
{
    Window w;
    w.edge = -1;
    w.e32 = 0.f;
    w.wsum = b.wsum;
    double c_lo, c_hi;
    if (!cap_window(a, b, slack, c_lo, c_hi)) return w;
    const int r_lo = row_of_cos(c_hi, edges, nbins), r_hi = row_of_cos(c_lo, edges, nbins);
    if (r_hi - r_lo > 1) return w;
    if (prune && r_hi == r_lo && (r_lo == 0 || r_lo == nbins + 1)) {  // all closer than theta_min or all beyond theta_max
        w.edge = -2;
        return w;
    }
    w.edge = r_lo <= nbins ? r_lo : nbins;  // rows edge (c > e[edge]) and edge + 1
    w.e32 = edge32(edges[w.edge]);
    return w;
}

// One group of kGroup staged j-points against this thread's kR i-points, every pair tested against
// the single edge of the window.  Two j-points per step: d = e_m - c for both in three FFMA2.
// Tallies stay in registers and are added to the histogram rows `edge` and `edge + 1` at the end:
//   weighted: per i-point one fp64 accumulator t += ind * v_j, where ind = 2^-7 [d > 0] is the
//             float 1.0f / 0.0f of the comparison read as the high word of a double, and
//             v_j = C + w_j (packed: 128 t = n C + sum of w_j, both recovered exactly) or v_j = w_j
//             (count kept in a float beside it);
//   unweighted: the sign bits of d are shifted into a word per i-point and counted 32 at a time.
// |d| <= G1 for any pair of a step of kWinUnroll j-points sends that step's pairs to the exact row.
template <bool kWeighted, bool kPacked, bool kPrivate>
__device__ __forceinline__ void window_group(const PairParams &p, Hist<kWeighted, kPrivate> &h, const float *__restrict__ grp2,
                                             const double *__restrict__ vgrp, const unsigned long long (&nx2)[kR],
                                             const unsigned long long (&ny2)[kR], const unsigned long long (&nz2)[kR],
                                             const float (&wi)[kR], const Window win, const double packC, const double inv_packC,
                                             uint32_t i_base, uint32_t j_first, unsigned long long &n_fp64)
{
    const float e32 = win.e32;
    const unsigned long long e2 = pack2(e32, e32);
    double t_above[kR];   // weighted: 2^-7 * sum of v_j over the pairs above the edge, per i-point
    uint32_t sg[kR];      // unweighted: sign bits of d (1 = not above) of the last 32 j-points, per i-point
    uint32_t n_below = 0; // unweighted
    float n_above = 0.f;  // weighted, not packed: exact, at most kGroup * kR = 512
#pragma unroll
    for (int r = 0; r < kR; ++r) {
        t_above[r] = 0.0;
        sg[r] = 0u;
    }
#pragma unroll 1
    for (int jj = 0; jj < kGroup; jj += kWinUnroll) {
        float mn = 1.0f;  // min |d| of the step
#pragma unroll
        for (int u = 0; u < kWinUnroll; u += 2) {
            const ulonglong2 xy = *reinterpret_cast<const ulonglong2 *>(grp2 + (size_t)(jj + u) * 4);
            const unsigned long long zz = *reinterpret_cast<const unsigned long long *>(grp2 + (size_t)(jj + u) * 4 + 4);
            double v0 = 0.0, v1 = 0.0;
            if constexpr (kWeighted) {
                const double2 vv = *reinterpret_cast<const double2 *>(vgrp + jj + u);
                v0 = vv.x;
                v1 = vv.y;
            }
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                const unsigned long long d2 = ffma2(nx2[r], xy.x, ffma2(ny2[r], xy.y, ffma2(nz2[r], zz, e2)));
                const float d0 = __uint_as_float((uint32_t)d2), d1 = __uint_as_float((uint32_t)(d2 >> 32));
                if constexpr (kWeighted) {
                    float i0, i1;  // 1.0f if above else 0.0f (SASS FSET.BF)
                    asm("set.gt.f32.f32 %0, %1, 0f00000000;" : "=f"(i0) : "f"(d0));
                    asm("set.gt.f32.f32 %0, %1, 0f00000000;" : "=f"(i1) : "f"(d1));
                    t_above[r] = fma(v0, __hiloint2double(__float_as_int(i0), 0), t_above[r]);
                    t_above[r] = fma(v1, __hiloint2double(__float_as_int(i1), 0), t_above[r]);
                    if constexpr (!kPacked) n_above += i0 + i1;
                } else {
                    asm("shf.l.wrap.b32 %0, %1, %0, 1;" : "+r"(sg[r]) : "r"(__float_as_uint(d0)));
                    asm("shf.l.wrap.b32 %0, %1, %0, 1;" : "+r"(sg[r]) : "r"(__float_as_uint(d1)));
                }
                asm("min.f32 %0, %0, %1, %2;" : "+f"(mn) : "f"(fabsf(d0)), "f"(fabsf(d1)));
            }
        }
        if (__any_sync(0xffffffffu, !(mn > kGuardWin))) {
            // some pair is within the guard band of the edge: replace its row by the exact one
#pragma unroll 1
            for (int u = 0; u < kWinUnroll; ++u) {
                const float4 q = tile_point(grp2, jj + u);
#pragma unroll
                for (int r = 0; r < kR; ++r) {
                    const float d = fmaf(__uint_as_float((uint32_t)nx2[r]), q.x,
                                         fmaf(__uint_as_float((uint32_t)ny2[r]), q.y, fmaf(__uint_as_float((uint32_t)nz2[r]), q.z, e32)));
                    if (fabsf(d) > kGuardWin) continue;
                    // what the loop above tallied for this pair
                    const bool above = kWeighted ? d > 0.f : (__float_as_uint(d) >> 31) == 0u;
                    const uint32_t fast = (uint32_t)win.edge + (above ? 1u : 0u);
                    int ex = chord_row(-__uint_as_float((uint32_t)nx2[r]), -__uint_as_float((uint32_t)ny2[r]),
                                       -__uint_as_float((uint32_t)nz2[r]), q.x, q.y, q.z, p.sedges, p.nbins, p.chord_margin);
                    if (ex < 0) {
                        ex = exact_row(p.xyz_a, p.stride_a, p.perm_a[i_base + local_i(r)], p.xyz_b, p.stride_b,
                                       p.perm_b[j_first + jj + u], p.edges, p.nbins);
                        ++n_fp64;
                    } else {
                        n_fp64 += 1ull << 32;
                    }
                    const uint32_t exact = (uint32_t)ex;
                    if (exact != fast) {
                        h.move(fast, exact);
                        if constexpr (kWeighted) {
                            const double w = (double)wi[r] * (double)q.w;
                            h.add_w(fast, -w);
                            h.add_w(exact, w);
                        }
                    }
                }
            }
        }
        if constexpr (!kWeighted) {
            if ((jj & 31) == 32 - kWinUnroll) {
#pragma unroll
                for (int r = 0; r < kR; ++r) n_below += __popc(sg[r]);
            }
        }
    }
    const uint32_t total = (uint32_t)(kGroup * kR);
    uint32_t above = total - n_below;
    if constexpr (kWeighted) {
        // sum over this thread's pairs of w_i w_j = sum_r w_i[r] * (sum of w_j above / not above)
        double s_above = 0.0, s_below = 0.0;
        above = kPacked ? 0u : (uint32_t)n_above;
#pragma unroll
        for (int r = 0; r < kR; ++r) {
            double sw = t_above[r] * 128.0;  // undo the 2^-7 of the indicator
            if constexpr (kPacked) {
                const double n = floor(sw * inv_packC);  // C is a power of two and sum of w < C: exact
                sw -= n * packC;
                above += (uint32_t)n;
            }
            s_above = fma((double)wi[r], sw, s_above);
            s_below = fma((double)wi[r], win.wsum - sw, s_below);
        }
        if (above == total) s_below = 0.0;  // nothing below: not even a rounding residue of wsum - sw
        h.add_w((uint32_t)win.edge + 1u, s_above);
        h.add_w((uint32_t)win.edge, s_below);
    }
    h.add_n((uint32_t)win.edge + 1u, above);
    h.add_n((uint32_t)win.edge, total - above);
}

// ---- the kernel ---------------------------------------------------------------------------------
// kWarps consumer warps + one producer warp.  The producer pulls work items {i-tile, first j-tile,
// number of j-tiles} from a global counter and streams their j-tiles through a ring of kStages
// shared-memory buffers with TMA bulk copies (full/empty mbarriers per stage); each stage carries
// {i-tile, j-tile, points}.  Every consumer warp walks the same stream at its own pace -- a warp whose
// windows take the table path does not hold the others back until the ring is full -- holding its
// kGroup i-points of the current i-tile in registers.

template <bool kWeighted, bool kPrivate>
__global__ void __launch_bounds__(kThreads + 32, kWeighted ? 1 : 2) pair_kernel(const PairParams p_in)
{
    if (p_in.counters[kCtrBadInput] != 0) return;  // inputs failed validation: never index the LUT with garbage
    PairParams p = p_in;
    p.chord_margin = chord_margin(p_in.counters);
    if (kWeighted) {
        // Weights that do not pack with the count (PackInfo: range above 2^13) take the table path for every pair:
        // it adds each product w_i w_j to its row directly, where the window tallies would form small rows as
        // differences of large cumulative sums.
        const bool packed = p_in.pack_b->packed != 0;
        if (p_in.only_unpackable && packed) return;
        // This kernel's windows correct a mis-tallied pair by adding its weight to one row and subtracting it from
        // another; a row left with much smaller weights keeps the rounding of the larger one.  Counts are integers and
        // do not mind; weighted sums go pair by pair here (the window kernel corrects its exact accumulators instead).
        p.use_windows = 0;
    }
    extern __shared__ __align__(128) unsigned char smem[];
    const int rows = p.nbins + 2;
    const int n_stages = p.n_stages;
    // layout: [full bars | empty bars | stage meta] (512 B) [tiles][LUT][count rows][weighted rows]
    uint64_t *full = reinterpret_cast<uint64_t *>(smem);
    uint64_t *empty = full + kMaxStages;
    StageMeta *meta = reinterpret_cast<StageMeta *>(smem + 128);
    unsigned char *stages = smem + kSmemHeader;
    constexpr size_t kStage = stage_bytes(kWeighted);
    uint2 *lut = reinterpret_cast<uint2 *>(smem + kSmemHeader + (size_t)n_stages * kStage);
    const size_t cnt_words = kPrivate ? (size_t)kWarps * rows * 32 : (size_t)kWarps * rows;
    size_t off = kSmemHeader + (size_t)n_stages * kStage + (size_t)p.lut_len * sizeof(uint2);
    off = (off + 15) & ~size_t(15);
    uint32_t *cnt_all = reinterpret_cast<uint32_t *>(smem + off);
    off += cnt_words * sizeof(uint32_t);
    off = (off + 15) & ~size_t(15);
    double *ws_all = reinterpret_cast<double *>(smem + off);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    for (int i = tid; i < p.lut_len; i += blockDim.x) lut[i] = p.lut[i];
    for (size_t i = tid; i < cnt_words; i += blockDim.x) cnt_all[i] = 0;
    if constexpr (kWeighted)
        for (size_t i = tid; i < cnt_words; i += blockDim.x) ws_all[i] = 0.0;
    if (tid == 0) {
        for (int s = 0; s < n_stages; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], kWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    unsigned long long n_items = p.counters[kCtrWorkCount];
    if (n_items > p.capacity) n_items = p.capacity;

    if (warp == kWarps) {
        // ---------------- producer
        if (lane != 0) return;
        uint32_t produced = 0;  // stages filled so far: slot = produced % n_stages, round = produced / n_stages
        auto acquire = [&]() -> int {
            const int slot = (int)(produced % (uint32_t)n_stages);
            const uint32_t round = produced / (uint32_t)n_stages;
            mbar_wait(&empty[slot], (round & 1u) ^ 1u);  // round 0 passes at once: nothing to drain yet
            return slot;
        };
        while (true) {
            const unsigned long long item = atomicAdd(&p.counters[kCtrWorkHead], 1ull);
            if (item >= n_items) break;
            const int3 it = p.items[item];
            for (int t = 0; t < it.z; ++t) {
                const int tj = it.y + t;
                const uint32_t j0 = (uint32_t)tj * kTile;
                const uint32_t jn = p.n_b - j0 < (uint32_t)kTile ? p.n_b - j0 : (uint32_t)kTile;
                const int slot = acquire();
                StageMeta m;
                m.ti = it.x;
                m.tj = tj;
                m.jn = (int)jn;
                m.pad = 0;
                meta[slot] = m;
                // the arrays are padded to whole tiles: always a full tile
                mbar_expect_tx(&full[slot], (uint32_t)kStage);
                bulk_load(stages + (size_t)slot * kStage, p.pts2_b + (size_t)j0 * 4, (uint32_t)kTileBytes, &full[slot]);
                if constexpr (kWeighted)
                    bulk_load(stages + (size_t)slot * kStage + kTileBytes, p.vj_b + (size_t)j0, (uint32_t)kVjBytes, &full[slot]);
                ++produced;
            }
        }
        const int slot = acquire();  // end of stream
        StageMeta m;
        m.ti = -1;
        m.tj = m.jn = m.pad = 0;
        meta[slot] = m;
        mbar_arrive(&full[slot]);
        return;
    }

    // ---------------- consumers
    Hist<kWeighted, kPrivate> h;
    h.cnt = kPrivate ? cnt_all + (size_t)warp * rows * 32 : cnt_all + (size_t)warp * rows;
    h.ws = kPrivate ? ws_all + (size_t)warp * rows * 32 : ws_all + (size_t)warp * rows;
    h.lane = lane;

    unsigned long long n_fp64 = 0, n_eval = 0, n_win = 0, n_skip = 0;
    unsigned long long since_flush = 0;  // pairs this warp has tallied in its unflushed shared rows
    float wi[kR];
    unsigned long long nx2[kR], ny2[kR], nz2[kR];  // {-x, -x} etc.: both halves of an FFMA2 see the same i-point
#pragma unroll
    for (int r = 0; r < kR; ++r) {
        wi[r] = 0.f;
        nx2[r] = ny2[r] = nz2[r] = 0ull;
    }
    const PackInfo pack = *p.pack_b;
    uint32_t valid_mask = 0, i_base = 0, n_i = 0;
    bool i_full = false;
    int cur_ti = -1;

    auto flush_rows = [&]() {
        // this warp's rows -> global (u64 / f64 atomics); the rows restart from zero
        __syncwarp();
        if constexpr (kPrivate) {
            for (int row = 1; row <= p.nbins; ++row) {
                const unsigned long long v = warp_sum_u64((unsigned long long)h.cnt[row * 32 + lane]);
                h.cnt[row * 32 + lane] = 0;
                if (lane == 0 && v) atomicAdd(&p.counts[row - 1], v);
                if constexpr (kWeighted) {
                    double w = h.ws[row * 32 + lane];
                    h.ws[row * 32 + lane] = 0.0;
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) w += __shfl_xor_sync(0xffffffffu, w, o);
                    if (lane == 0 && w != 0.0) atomicAdd(&p.wsums[row - 1], w);
                }
            }
            h.cnt[lane] = 0;  // the two out-of-range rows are tallied but never reported
            h.cnt[(p.nbins + 1) * 32 + lane] = 0;
        } else {
            for (int row = lane; row < rows; row += 32) {
                const uint32_t v = h.cnt[row];
                h.cnt[row] = 0;
                if (row >= 1 && row <= p.nbins && v) atomicAdd(&p.counts[row - 1], (unsigned long long)v);
                if constexpr (kWeighted) {
                    const double w = h.ws[row];
                    h.ws[row] = 0.0;
                    if (row >= 1 && row <= p.nbins && w != 0.0) atomicAdd(&p.wsums[row - 1], w);
                }
            }
        }
        __syncwarp();
        since_flush = 0;
    };

    for (uint32_t consumed = 0;; ++consumed) {
        const int slot = (int)(consumed % (uint32_t)n_stages);
        mbar_wait(&full[slot], (consumed / (uint32_t)n_stages) & 1u);
        const StageMeta m = meta[slot];
        if (m.ti < 0) break;
        if (m.ti != cur_ti) {
            cur_ti = m.ti;
            i_base = (uint32_t)m.ti * kTile;
            valid_mask = 0;
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                const uint32_t s = i_base + local_i(r);
                const float4 v = p.pts_a[s];  // the array is padded to a whole tile
                nx2[r] = pack2(-v.x, -v.x);
                ny2[r] = pack2(-v.y, -v.y);
                nz2[r] = pack2(-v.z, -v.z);
                wi[r] = v.w;
                valid_mask |= (s < p.n_a ? 1u : 0u) << r;
            }
            i_full = i_base + kTile <= p.n_a;
            n_i = i_full ? kTile : p.n_a - i_base;
        }
        const float *tile = reinterpret_cast<const float *>(stages + (size_t)slot * kStage);
        const double *vtile = reinterpret_cast<const double *>(stages + (size_t)slot * kStage + kTileBytes);
        const int tj = m.tj, jn = m.jn;
        const bool diag = p.is_auto && tj == m.ti;
        const uint32_t j_base = (uint32_t)tj * kTile;
        // u32 rows: flush before this warp's tallies could wrap (per lane when private, per row otherwise)
        if (since_flush + (unsigned long long)kGroup * kTile > (kPrivate ? (32ull << 31) : (1ull << 31))) flush_rows();
        since_flush += (unsigned long long)kGroup * (unsigned)jn;

        if (diag || !i_full) {
            process_tile<kWeighted, kPrivate, true>(p, h, tile, 0, jn, nx2, ny2, nz2, wi, lut, i_base, j_base, diag, valid_mask, n_fp64);
        } else if (!p.use_windows) {
            process_tile<kWeighted, kPrivate, false>(p, h, tile, 0, jn, nx2, ny2, nz2, wi, lut, i_base, j_base, false, valid_mask, n_fp64);
        } else {
            // lane g works out the window of this warp's i-group against j-group g of the tile
            const int n_groups = (jn + kGroup - 1) / kGroup;
            Window mine;
            mine.edge = -1;
            mine.e32 = 0.f;
            mine.wsum = 0.0;
            if (lane < n_groups && (lane + 1) * kGroup <= jn)
                mine = make_window(p.gcaps_a[(size_t)m.ti * kGroupsPerTile + warp], p.gcaps_b[(size_t)tj * kGroupsPerTile + lane],
                                   p.edges, p.nbins, p.prune != 0, cap_slack(norm_eps(p.counters)));
            for (int g = 0; g < n_groups; ++g) {
                Window win;
                win.edge = __shfl_sync(0xffffffffu, mine.edge, g);
                win.e32 = __shfl_sync(0xffffffffu, mine.e32, g);
                win.wsum = __shfl_sync(0xffffffffu, mine.wsum, g);
                if (win.edge == -2) {  // pruned at the level of groups, like whole tiles in the work list
                    n_skip += (unsigned long long)(kGroup * kR);
                    continue;
                }
                if (win.edge >= 0) {
                    window_group<kWeighted, true, kPrivate>(p, h, tile + (size_t)g * kGroup * 4, vtile + g * kGroup, nx2, ny2, nz2, wi, win,
                                                            pack.C, pack.inv_C, i_base, j_base + g * kGroup, n_fp64);
                    n_win += (unsigned long long)(kGroup * kR);
                } else {
                    const int gn = jn - g * kGroup < kGroup ? jn - g * kGroup : kGroup;
                    process_tile<kWeighted, kPrivate, false>(p, h, tile, g * kGroup, gn, nx2, ny2, nz2, wi, lut, i_base, j_base, false, valid_mask, n_fp64);
                }
            }
        }
        if (tid == 0) n_eval += diag ? (unsigned long long)n_i * (n_i - 1) / 2 : (unsigned long long)n_i * (unsigned)jn;
        __syncwarp();  // every lane has read the stage before it is handed back
        if (lane == 0) mbar_arrive(&empty[slot]);
    }

    flush_rows();
    n_fp64 = warp_sum_u64(n_fp64);  // low word: re-evaluated in fp64; high word: decided by the chord tier
    if (lane == 0 && (n_fp64 & 0xffffffffull)) atomicAdd(&p.counters[kCtrPairsFp64], n_fp64 & 0xffffffffull);
    if (lane == 0 && (n_fp64 >> 32)) atomicAdd(&p.counters[kCtrPairsChord], n_fp64 >> 32);
    n_win = warp_sum_u64(n_win);
    if (lane == 0 && n_win) atomicAdd(&p.counters[kCtrPairsWindow], n_win);
    if (tid == 0 && n_eval) atomicAdd(&p.counters[kCtrPairsEvaluated], n_eval);
    n_skip = warp_sum_u64(n_skip);  // counted in n_eval with their tile, never evaluated
    if (lane == 0 && n_skip) atomicAdd(&p.counters[kCtrPairsEvaluated], 0ull - n_skip);
}

// ---- host: the cell table -------------------------------------------------------------------
// Cells are the float values sharing the top (9 + m) bits; each gets the single edge (as K - e)
// that can separate two rows inside it, or a NaN threshold when two or more edges crowd it.
struct Lut {
    std::vector<uint2> cells;
    int m, shift, key0;
};

float bits_to_float(uint32_t b)
{
    float f;
    memcpy(&f, &b, 4);
    return f;
}
uint32_t float_to_bits(float f)
{
    uint32_t b;
    memcpy(&b, &f, 4);
    return b;
}

Lut build_lut(const double *edges, int nbins, int m)
{
    Lut L;
    L.m = m;
    L.shift = 23 - m;
    L.key0 = (int)(float_to_bits(std::ldexp(1.0f, kExpLo)) >> L.shift);
    const int key1 = (int)(float_to_bits(std::ldexp(1.0f, kExpHi)) >> L.shift);
    L.cells.resize((size_t)(key1 - L.key0));
    std::vector<double> te(nbins + 1);  // edges in the t domain, ascending
    for (int k = 0; k <= nbins; ++k) te[k] = (double)kK - edges[k];
    // The pair cosine is clamped to [-1, 1]: when the range reaches a pole nothing lies beyond it, so
    // that edge must not be tested in fp32 (an unclamped c32 marginally outside would be misfiled).
    if (edges[0] >= 1.0) te[0] = -1.0e300;
    if (edges[nbins] <= -1.0) te[nbins] = 1.0e300;
    const double G = (double)kGuard;
    int crowded = 0;
    for (int key = L.key0; key < key1; ++key) {
        const double lo = (double)bits_to_float((uint32_t)key << L.shift);
        const double hi = (double)bits_to_float((uint32_t)(key + 1) << L.shift);
        int below = 0, inside = 0, first = -1;
        for (int k = 0; k <= nbins; ++k) {
            if (te[k] < lo - G) ++below;
            else if (te[k] <= hi + G) {
                if (!inside) first = k;
                ++inside;
            }
        }
        uint2 c;
        c.y = (uint32_t)below;
        if (inside == 0) c.x = float_to_bits(3.0e38f);
        else if (inside == 1) c.x = float_to_bits((float)te[first]);
        else {
            c.x = 0x7fc00000u;  // NaN: every pair of the cell is re-checked
            ++crowded;
        }
        L.cells[(size_t)(key - L.key0)] = c;
    }
    (void)crowded;
    return L;
}

// number of cells that are crowded although they are wider than a few guard bands (i.e. a finer
// table would resolve them)
int crowded_resolvable(const Lut &L)
{
    int n = 0;
    for (size_t i = 0; i < L.cells.size(); ++i) {
        if (L.cells[i].x != 0x7fc00000u) continue;
        const double lo = (double)bits_to_float((uint32_t)(L.key0 + (int)i) << L.shift);
        const double hi = (double)bits_to_float((uint32_t)(L.key0 + (int)i + 1) << L.shift);
        if (hi - lo > 8.0 * (double)kGuard) ++n;
    }
    return n;
}

template <bool kWeighted, bool kPrivate>
cudaError_t launch(acf_ctx *ctx, const PairParams &p, size_t smem, int grid)
{
    auto kern = pair_kernel<kWeighted, kPrivate>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<grid, kThreads + 32, smem, ctx->stream>>>(p);
    ctx->last.kernel_launches++;
    return cudaGetLastError();
}

// The verdicts of the two catalogues' validations -> the call's counters, where the kernels look for them.
__global__ void seed_counters_kernel(unsigned long long *__restrict__ counters, const PackInfo *__restrict__ pa, const PackInfo *__restrict__ pb)
{
    const int bad = pa->bad + (pb != pa ? pb->bad : 0);
    if (bad) atomicAdd(&counters[kCtrBadInput], (unsigned long long)bad);
    const double eps = fmax(pa->eps, pb->eps);
    atomicMax(&counters[kCtrNormDev], (unsigned long long)__double_as_longlong(eps));
}

int count_prepared(acf_ctx *ctx, const Prepared &a, const Prepared &b, int is_auto, const double *h_edges, int nbins,
                   const Lut &L, const uint2 *d_lut, int part, int n_parts, unsigned long long *d_counts, double *d_wsums)
{
    if (a.n == 0 || b.n == 0 || part >= a.n_tiles) return ACF_OK;
    seed_counters_kernel<<<1, 1, 0, ctx->stream>>>(ctx->d_counters, a.pack, b.pack);
    ctx->last.kernel_launches++;
    const bool weighted = d_wsums != nullptr;
    const int rows = nbins + 2;
    const bool priv = rows <= kMaxPrivateRows;
    // shared memory: header, LUT, histogram rows, and as many j-tile stages as fit (2 CTAs per SM when
    // unweighted and small enough, else 1)
    const size_t cnt_words = priv ? (size_t)kWarps * rows * 32 : (size_t)kWarps * rows;
    auto smem_for = [&](int stages) {
        size_t m = kSmemHeader + (size_t)stages * stage_bytes(weighted) + L.cells.size() * sizeof(uint2);
        m = (m + 15) & ~size_t(15);
        m += cnt_words * sizeof(uint32_t);
        m = (m + 15) & ~size_t(15);
        if (weighted) m += cnt_words * sizeof(double);
        return m;
    };
    const size_t per_sm = (size_t)ctx->max_smem_optin;            // per CTA limit; an SM has 1 KB more per resident CTA
    int ctas_per_sm = (!weighted && smem_for(2) <= (per_sm - 1024) / 2) ? 2 : 1;
    const size_t budget = ctas_per_sm == 2 ? (per_sm - 1024) / 2 : per_sm;
    int n_stages = 2;
    while (n_stages < 4 && smem_for(n_stages + 1) <= budget) ++n_stages;
    const size_t smem = smem_for(n_stages);
    // which kernel: the window kernel; the table kernel on request, and behind the window kernel
    // for weights that do not pack
    bool use_win = ctx->opt_kernel == ACF_KERNEL_WINDOW || ctx->opt_kernel == ACF_KERNEL_AUTO;
    const bool table_fits = smem <= per_sm;
    if (!use_win && !table_fits) {
        if (ctx->opt_kernel != ACF_KERNEL_AUTO) return fail(ctx, ACF_EINVAL, "shared memory need %zu exceeds %d", smem, ctx->max_smem_optin);
        use_win = true;
    }
    // The window kernel tallies weights only when they pack with the count (PackInfo, decided on the device from the
    // weight range); otherwise it returns at once and the table kernel, launched behind it, does the call.  Where the
    // table kernel's histograms do not fit either, the verdict is fetched and the call refused.
    if (use_win && weighted && !table_fits) {
        PackInfo pk{};
        ACF_CUDA_TRY(ctx, cudaMemcpyAsync(&pk, b.pack, sizeof(PackInfo), cudaMemcpyDeviceToHost, ctx->stream));
        ACF_CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
        if (!pk.packed && pk.bad == 0)
            return fail(ctx, ACF_EINVAL, "weights ranging over more than 2^13 cannot be tallied with %d bins (at most about 600)", nbins);
    }

    // i-tiles are handed out in batches so that the item buffer stays bounded
    // (worst case one item per surviving j-tile: survivors may alternate with pruned tiles)
    const uint64_t items_per_ti = (uint64_t)b.n_tiles;
    const uint64_t max_items = 64u << 20;  // 768 MB of items at most (8 M x 8 M points: 61 M tile pairs, one launch)
    const int n_mine = (a.n_tiles - part + n_parts - 1) / n_parts;  // i-tiles part, part + n_parts, ...
    int ti_per_batch = (int)(max_items / items_per_ti);
    if (ti_per_batch < 1) ti_per_batch = 1;
    if (ti_per_batch > n_mine) ti_per_batch = n_mine;
    const uint32_t capacity = (uint32_t)(items_per_ti * (uint64_t)ti_per_batch);
    ACF_CUDA_TRY(ctx, ctx->s_work.reserve(sizeof(int3) * (size_t)capacity));

    PairParams p{};
    p.pts_a = a.pts;
    p.pts2_b = b.pts2;
    p.vj_b = b.vj;
    p.pack_b = b.pack;
    p.perm_a = a.perm;
    p.perm_b = b.perm;
    p.gcaps_a = a.gcaps;
    p.gcaps_b = b.gcaps;
    p.use_windows = ctx->opt_windows;
    p.prune = ctx->opt_prune;
    p.n_a = (uint32_t)a.n;
    p.n_b = (uint32_t)b.n;
    p.xyz_a = a.xyz;
    p.xyz_b = b.xyz;
    p.stride_a = a.stride;
    p.stride_b = b.stride;
    p.items = ctx->s_work.as<int3>();
    p.capacity = capacity;
    p.lut = d_lut;
    p.lut_len = (int)L.cells.size();
    p.key0 = L.key0;
    p.shift = L.shift;
    p.edges = ctx->s_edges.as<double>();
    p.sedges = ctx->d_sedges;
    p.nbins = nbins;
    p.counts = d_counts;
    p.wsums = d_wsums;
    p.counters = ctx->d_counters;
    p.is_auto = is_auto;
    p.n_stages = n_stages;

    const int grid = ctx->num_sms * ctas_per_sm;
    for (int k0 = 0; k0 < n_mine; k0 += ti_per_batch) {
        const int k1 = k0 + ti_per_batch < n_mine ? k0 + ti_per_batch : n_mine;
        const int ti0 = part + k0 * n_parts;
        const int ti1 = part + (k1 - 1) * n_parts + 1;
        ACF_CUDA_TRY(ctx, cudaMemsetAsync(&ctx->d_counters[kCtrWorkHead], 0, 2 * sizeof(unsigned long long), ctx->stream));
        int rc = build_worklist(ctx, a, ti0, ti1, n_parts, b, is_auto, h_edges[0], h_edges[nbins], ctx->s_work.as<int3>(), capacity);
        if (rc != ACF_OK) return rc;
        cudaError_t e;
        if (!ctx->pair_timed) {
            ACF_CUDA_TRY(ctx, cudaEventRecord(ctx->ev_k0, ctx->stream));
            ctx->pair_timed = true;
        }
        if (use_win) {
            rc = launch_pair_win(ctx, a, b, is_auto, h_edges, nbins, capacity, d_counts, d_wsums);
            if (rc != ACF_OK) return rc;
            if (weighted && table_fits) {  // the same work list again, for weights that do not pack
                ACF_CUDA_TRY(ctx, cudaMemsetAsync(&ctx->d_counters[kCtrWorkHead], 0, sizeof(unsigned long long), ctx->stream));
                PairParams q = p;
                q.only_unpackable = 1;
                e = priv ? launch<true, true>(ctx, q, smem, grid) : launch<true, false>(ctx, q, smem, grid);
                ACF_CUDA_TRY(ctx, e);
            }
        } else {
            if (weighted) e = priv ? launch<true, true>(ctx, p, smem, grid) : launch<true, false>(ctx, p, smem, grid);
            else e = priv ? launch<false, true>(ctx, p, smem, grid) : launch<false, false>(ctx, p, smem, grid);
            ACF_CUDA_TRY(ctx, e);
        }
        ACF_CUDA_TRY(ctx, cudaEventRecord(ctx->ev_k1, ctx->stream));
    }
    return ACF_OK;
}

}  // namespace

namespace {

// The device tables of a call: the edges (fp64), the edges as squared chord lengths (fp32, chord tier) and, when the
// table kernel may run (on request, or behind the window kernel for weights that do not pack), its cell table.
int upload_tables(acf_ctx *ctx, const double *h_edges, int nbins, bool weighted, Lut &L, const uint2 *&d_lut)
{
    const bool want_lut = ctx->opt_kernel == ACF_KERNEL_TABLE || weighted;
    if (want_lut) {
        // cell table: the coarsest resolution that leaves no resolvable cell crowded
        L = build_lut(h_edges, nbins, 6);
        for (int m = 7; m <= 9 && crowded_resolvable(L) > 0; ++m) L = build_lut(h_edges, nbins, m);
        // with very many bins a coarser table (more cells left to the re-checks) may be what lets the kernel fit
        const int rows = nbins + 2;
        const size_t words = rows <= kMaxPrivateRows ? (size_t)kWarps * rows * 32 : (size_t)kWarps * rows;
        auto need = [&](const Lut &t) {
            return kSmemHeader + 2 * stage_bytes(weighted) + t.cells.size() * sizeof(uint2) + words * (weighted ? 12 : 4) + 32;
        };
        while (L.m > 6 && need(L) > (size_t)ctx->max_smem_optin) L = build_lut(h_edges, nbins, L.m - 1);
    } else {
        L = Lut{};
        L.m = 6;
        L.shift = 23 - 6;
        L.key0 = 0;
    }
    const size_t edge_bytes = (sizeof(double) * (size_t)(nbins + 1) + 15) & ~size_t(15);
    const size_t sed_bytes = (sizeof(float) * (size_t)(nbins + 1) + 15) & ~size_t(15);
    // staged through pinned memory: the copies are asynchronous and the caller's array may go away at once
    const size_t total = edge_bytes + sed_bytes + L.cells.size() * sizeof(uint2);
    if (ctx->h_tables_bytes < total) {
        if (ctx->h_tables) cudaFreeHost(ctx->h_tables);
        ctx->h_tables = nullptr;
        ctx->h_tables_bytes = 0;
        ACF_CUDA_TRY(ctx, cudaHostAlloc(&ctx->h_tables, total + 4096, cudaHostAllocDefault));
        ctx->h_tables_bytes = total + 4096;
    } else {
        // the previous call's copy out of this buffer must have been made
        ACF_CUDA_TRY(ctx, cudaEventSynchronize(ctx->ev_tables));
    }
    char *h = static_cast<char *>(ctx->h_tables);
    memcpy(h, h_edges, sizeof(double) * (size_t)(nbins + 1));
    float *sed = reinterpret_cast<float *>(h + edge_bytes);
    for (int k = 0; k <= nbins; ++k) sed[k] = (float)(2.0 * (1.0 - h_edges[k]));
    if (h_edges[0] >= 1.0) sed[0] = -1.0f;  // c is clamped: nothing lies beyond a pole
    if (h_edges[nbins] <= -1.0) sed[nbins] = std::numeric_limits<float>::infinity();
    if (!L.cells.empty()) memcpy(h + edge_bytes + sed_bytes, L.cells.data(), L.cells.size() * sizeof(uint2));
    ACF_CUDA_TRY(ctx, ctx->s_edges.reserve(total));
    ACF_CUDA_TRY(ctx, cudaMemcpyAsync(ctx->s_edges.ptr, h, total, cudaMemcpyHostToDevice, ctx->stream));
    ACF_CUDA_TRY(ctx, cudaEventRecord(ctx->ev_tables, ctx->stream));
    ctx->d_sedges = reinterpret_cast<float *>(static_cast<char *>(ctx->s_edges.ptr) + edge_bytes);
    d_lut = reinterpret_cast<const uint2 *>(static_cast<char *>(ctx->s_edges.ptr) + edge_bytes + sed_bytes);
    return ACF_OK;
}

}  // namespace

int count_prepared_part(acf_ctx *ctx, const Prepared &a, const Prepared &b, int is_auto, const double *h_edges, int nbins,
                        int part, int n_parts, unsigned long long *d_counts, double *d_wsums)
{
    Lut L;
    const uint2 *d_lut = nullptr;
    int rc = upload_tables(ctx, h_edges, nbins, d_wsums != nullptr, L, d_lut);
    if (rc != ACF_OK) return rc;
    return count_prepared(ctx, a, b, is_auto, h_edges, nbins, L, d_lut, part, n_parts, d_counts, d_wsums);
}

}  // namespace acf
