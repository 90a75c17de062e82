// acf_pair_win.cu -- the window kernel: every pair classified against the bin edges that can matter
// for its window, tallies in registers, no per-pair shared-memory traffic.
//
// Points are sorted along a space-filling curve, so the kGroup i-points of a warp and a group of kGroup
// staged j-points each sit in a small cap; the two caps bound the cosines of all their pairs to a window
// [c_lo, c_hi] (fp64, rigorous), i.e. to the histogram rows r_lo .. r_hi and the k = r_hi - r_lo edges
// e[r_lo] .. e[r_hi - 1] between them.  The edges are taken kChunk at a time.  Per pair and chunk:
//   d_0 = e_m - (x_i x_j + y_i y_j + z_i z_j)      three fp32 FMAs seeded with fp32(e_m)  (two j-points per FFMA2)
//   d_q = d_0 + fp32(e_{m+q} - e_m)                 one add per further edge of the chunk
//   above_q = d_q > 0                               the pair lies in a row beyond edge m + q
//   certified iff |d_q| > G for every q             else the exact fp64 row of include/acf.h decides
// Per i-point and edge one fp64 accumulator takes t += [above_q] v_j (v_j = C + w_j packs the count and
// the weight sum, see PackInfo: exact sums; weights of too wide a range for that are not tallied here
// but pair by pair in acf_pair.cu; unweighted counts shift the sign bits of d_q into a word instead).
// The accumulators are cumulative in q (above edge m + q implies above edge m + q - 1), so the rows get
// the differences of consecutive edges; they are formed per i-point before anything is summed.
// After a chunk the warp reduces its row tallies with shuffles and lane 0 adds them to the warp's rows in
// shared memory; those go to global memory with u64 / f64 atomics (block histograms summed
// into global memory -- here without a per-pair atomic, the 5-50 % serialisation the paper measures).
// Ragged groups and the diagonal group of an auto-count (i < j) run the same loop with a per-pair mask.
#include <cmath>
#include <cstring>

#include "acf_device.cuh"
#include "acf_internal.h"
#include "acf_pair_common.cuh"

namespace acf {

namespace {

constexpr int kTeams = 2;              // teams of consumer warps: same i-points, alternate j-groups
constexpr int kTeamWarps = kTile / kGroup;  // a team's warps hold the i-tile, kGroup points each
constexpr int kWarps = kTeams * kTeamWarps;  // consumer warps
constexpr int kThreads = 32 * kWarps;  // consumer threads
constexpr int kR = kGroup / 32;        // i-points per thread
#ifndef ACF_WIN_CHUNK
#define ACF_WIN_CHUNK 3
#endif
constexpr int kChunk = ACF_WIN_CHUNK;  // edges per pass over a group
constexpr int kStep = 4;               // j-points per guard-band vote
// Guard bands (u = 2^-24).  A wrong fp32 sign needs |d_0 - (e_m - c64)| >= |d_0|,
// so only pairs with a small |d_0| matter; for those the partial sums of the chain are below 1 + 2e-6 in
// magnitude (they differ from d_0 by products of coordinates whose absolute sum is at most 1 + 2e-6):
//   2^-25 [fp32(e_m)] + 2u (1 + 1e-6) [the six rounded coordinates] + 2 * 2^-24 [the two inner FMAs]
//   + 2^-24 |d_0| [the last FMA] + 4e-16 [c64 itself]  <=  2.69e-7.
// d_q, q >= 1, is the sum of a d_0 that is not small and a rounded offset: partial sums below 4 (three
// roundings of 2^-23), the offset (2^-24) and the six coordinates give 5.7e-7.
constexpr float kGuard1 = 3.0e-7f;
constexpr float kGuardK = 7.0e-7f;
static_assert(kGroup == kR * 32 && (kTeamWarps & (kTeamWarps - 1)) == 0, "a warp's i-points are one group");
static_assert(kGroup % 32 == 0 && 32 % kStep == 0 && kStep % 2 == 0, "");

struct WinParams {
    const float4 *pts_a;
    const float *pts2_b;
    const double *vj_b;
    const PackInfo *pack_b;
    const uint32_t *perm_a, *perm_b;
    const GroupCap *gcaps_a, *gcaps_b;
    uint32_t n_a, n_b;
    const double *xyz_a, *xyz_b;
    size_t stride_a, stride_b;
    const int3 *items;
    uint32_t capacity;
    const double *edges;
    const float *sedges;  // the edges as squared chord lengths (chord_row)
    int nbins;
    unsigned long long *counts;
    double *wsums;
    unsigned long long *counters;
    int is_auto;
    int n_stages;
    int shared_rows;  // 1: one set of histogram rows per CTA instead of one per warp
    int prune;        // 1: groups whose window lies wholly out of range are not evaluated
    int bulk;         // 1: groups whose window lies wholly inside one bin are counted as a whole (ACF_OPT_BULK)
};

__device__ __forceinline__ unsigned long long fadd2(unsigned long long a, unsigned long long b)
{
    unsigned long long d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ float lo32(unsigned long long v) { return __uint_as_float((uint32_t)v); }
__device__ __forceinline__ float hi32(unsigned long long v) { return __uint_as_float((uint32_t)(v >> 32)); }
// 1.0f if v > 0 else 0.0f (SASS FSET.BF); read as the high word of a double it is 2^-7 or 0
__device__ __forceinline__ float ind_gt0(float v)
{
    float r;
    asm("set.gt.f32.f32 %0, %1, 0f00000000;" : "=f"(r) : "f"(v));
    return r;
}

// The same comparison written into the high word of a 64-bit register whose low word is and stays zero:
// the register then reads as the double 2^-7 [v > 0] with no instruction spent on the low word.
__device__ __forceinline__ double ind_gt0_f64(unsigned long long &reg, float v)
{
    asm("{\n\t.reg .b32 lo, hi;\n\tmov.b64 {lo, hi}, %0;\n\tset.gt.f32.f32 hi, %1, 0f00000000;\n\tmov.b64 %0, {lo, hi};\n\t}"
        : "+l"(reg)
        : "f"(v));
    return __longlong_as_double((long long)reg);
}

// This warp's histogram rows in shared memory.  Lane 0 adds the reduced tallies; the rare exact
// corrections come from any lane and are atomic.
struct Rows {
    uint32_t *cnt;
    double *ws;
    const PackInfo *pack;  // the j side's PackInfo, copied to shared memory
    bool shared;  // one set of rows for the whole CTA (many bins): every update is atomic
    template <bool kWeighted>
    __device__ __forceinline__ void add_atomic(int row, uint32_t c, double w) const  // from any lane
    {
        atomicAdd(&cnt[row], c);
        if constexpr (kWeighted) atomicAdd(&ws[row], w);
    }
    template <bool kWeighted>
    __device__ __forceinline__ void add(int row, uint32_t c, double w) const  // lane 0 of the rows' warp
    {
        if (shared) {
            if (c) atomicAdd(&cnt[row], c);
            if constexpr (kWeighted)
                if (w != 0.0) atomicAdd(&ws[row], w);
        } else {
            cnt[row] += c;
            if constexpr (kWeighted) ws[row] += w;
        }
    }
};
// per-CTA statistics kept in shared memory until the kernel ends
enum { kStatFp64 = 0, kStatWindow = 1, kStatEvaluated = 2, kStatChord = 3, kStatBulk = 4, kNumStats = 5 };
// rows and weight of one window, parked in shared memory between its computation and its use
struct WinRows {
    int lo, hi;
    double wsum;
    float e32;  // fp32 of the edge a window with at most one edge is tested against
    int pad;
};

__device__ __forceinline__ double warp_sum_f64(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Thread (warp, lane) holds the i-points (warp % kTeamWarps) * kGroup + r * 32 + lane of the i-tile, r < kR.
__device__ __forceinline__ uint32_t local_i(int r)
{
    return ((threadIdx.x >> 5) & (kTeamWarps - 1)) * kGroup + r * 32 + (threadIdx.x & 31);
}


// Which pairs of a group count: ragged ends of the catalogues and the diagonal group of an auto-count.
struct Mask {
    uint32_t valid;  // bit r: i-point r of this thread exists
    int jn;          // j-points of the group that exist
    int j0;          // index in the tile of the group's first j-point
    bool diag;       // count only pairs with (index in tile of j) > (index in tile of i)
    __device__ __forceinline__ bool on(int r, int jj) const
    {
        return ((valid >> r) & 1u) && jj < jn && (!diag || (uint32_t)(j0 + jj) > local_i(r));
    }
};

// The exact corrections of one chunk of a group, after its loop and before its tallies are read:
// amb_steps has a bit per step of kStep j-points in which some pair came within the guard band of an
// edge.  Every pair of those steps is re-derived bit for bit as the loop computed it; a pair within a
// guard band gets its row from the chord tier or the fp64 definition of include/acf.h, and where that
// disagrees with what the loop tallied, the correction of this thread's accumulators comes back:
//   dt[q * kR + r]  to add to t[q][r]: 2^-7 v_j for a pair that is above edge q after all, minus that for
//                   one that is not (the accumulators are exact sums, so the corrected tally is exactly the
//                   tally of the exact classification: no row ever sees a wrong pair added and taken back);
//   dn[q]           to add to nb[q] (unweighted: pairs not above edge q).
// One copy for all chunk shapes; it reloads the i-points rather than taking them in registers.
template <bool kWeighted>
__device__ __noinline__ void fixup_chunk(const WinParams &p, const float *__restrict__ grp2, const double *__restrict__ vgrp,
                                         uint32_t amb_steps, int K, int m_a, bool masked, const Mask mk, uint32_t i_base,
                                         uint32_t j_first, unsigned long long *stat, double *__restrict__ dt, int *__restrict__ dn)
{
    float4 pi[kR];
#pragma unroll
    for (int r = 0; r < kR; ++r) pi[r] = p.pts_a[i_base + local_i(r)];  // the array is padded to a whole tile
    for (int i = 0; i < kChunk * kR; ++i) dt[i] = 0.0;
    for (int i = 0; i < kChunk; ++i) dn[i] = 0;
    const double e0 = p.edges[m_a];
    const float e32 = (float)e0;
    const float G = K == 1 ? kGuard1 : kGuardK;
    const float margin = chord_margin(p.counters);
    float dl[kChunk];
#pragma unroll
    for (int q = 0; q < kChunk; ++q) dl[q] = q > 0 && q < K ? (float)(p.edges[m_a + q] - e0) : 0.f;
    while (amb_steps) {
        const int jj0 = (__ffs(amb_steps) - 1) * kStep;
        amb_steps &= amb_steps - 1;
        for (int u = 0; u < kStep; ++u) {
            const float4 pj = tile_point(grp2, jj0 + u);
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                if (masked && !mk.on(r, jj0 + u)) continue;
                const float d0 = fmaf(-pi[r].x, pj.x, fmaf(-pi[r].y, pj.y, fmaf(-pi[r].z, pj.z, e32)));
                bool amb = false;
#pragma unroll
                for (int q = 0; q < kChunk; ++q) amb |= q < K && !(fabsf(q == 0 ? d0 : __fadd_rn(d0, dl[q])) > G);
                if (!amb) continue;
                // the chord length decides where the cosine could not; what it leaves open, the definition
                int exact = chord_row(pi[r].x, pi[r].y, pi[r].z, pj.x, pj.y, pj.z, p.sedges, p.nbins, margin);
                if (exact < 0) {
                    exact = exact_row(p.xyz_a, p.stride_a, p.perm_a[i_base + local_i(r)], p.xyz_b, p.stride_b,
                                      p.perm_b[j_first + jj0 + u], p.edges, p.nbins);
                    atomicAdd(&stat[kStatFp64], 1ull);
                } else {
                    atomicAdd(&stat[kStatChord], 1ull);
                }
#pragma unroll
                for (int q = 0; q < kChunk; ++q) {
                    if (q >= K) break;
                    const float dq = q == 0 ? d0 : __fadd_rn(d0, dl[q]);
                    // what the loop tallied for this pair and edge
                    const bool fast_above = kWeighted ? dq > 0.f : (__float_as_uint(dq) >> 31) == 0u;
                    const bool exact_above = exact > m_a + q;
                    if (fast_above != exact_above) {
                        if constexpr (kWeighted) dt[q * kR + r] += (exact_above ? 0.0078125 : -0.0078125) * vgrp[jj0 + u];
                        else dn[q] += exact_above ? -1 : 1;
                    }
                }
            }
        }
    }
}

// What a thread carries from one chunk of a group's edges to the next (registers of window_group): its
// pairs above the last edge done and, per i-point, the sum of their w_j.
struct Carry {
    uint32_t c;
    double s[kGroup / 32];
};

// One thread's tallies of the two rows around an edge, kept in registers over consecutive groups that
// are tested against the same edge (the common single-edge groups of the kernel's own loop).
struct LaneTally {
    uint32_t c_lo, c_hi;  // pairs in row m / row m + 1
    double w_lo, w_hi;    // and their weight
};

// Edges m_a .. m_a + K - 1 against one group of kGroup staged j-points and this thread's kR i-points.
// A chunk fills rows m_a .. m_a + K - 1 (and m_a + K if it is the last of its group); the tallies above
// its last edge go to the next chunk through `carry`.
template <int K, bool kWeighted, bool kMasked, bool kDeferFix = false>
__device__ __forceinline__ uint32_t window_chunk(const WinParams &p, const Rows rows, const float *__restrict__ grp2,
                                             const double *__restrict__ vgrp, const float (&nx)[kR],
                                             const float (&ny)[kR], const float (&nz)[kR],
                                             const float (&wi)[kR], const int m_a, const bool first, const bool last, const double wsum_j,
                                             const Mask &mk, uint32_t i_base, uint32_t j_first, unsigned long long *stat,
                                             LaneTally *tally = nullptr, Carry *carry = nullptr, float e32_known = 0.f)
{
    const int lane = threadIdx.x & 31;
    const double e0 = kDeferFix ? 0.0 : p.edges[m_a];               // (the kernel's own loop has the edge at hand)
    const float e32 = kDeferFix ? e32_known : (float)e0;
    const unsigned long long e2 = pack2(e32, e32);
    float dl[K];
    unsigned long long dl2[K];
    dl[0] = 0.f;
    dl2[0] = 0ull;
#pragma unroll
    for (int q = 1; q < K; ++q) {
        dl[q] = (float)(p.edges[m_a + q] - e0);
        dl2[q] = pack2(dl[q], dl[q]);
    }
    const float G = K == 1 ? kGuard1 : kGuardK;

    double t[K][kR];     // weighted: 2^-7 * sum of v_j over the pairs above edge q, per i-point
    uint32_t sg[K][kR];  // unweighted: sign bits of d_q (1 = not above) of the last 32 j-points
    uint32_t nb[K];      // unweighted: pairs not above edge q
    double tall[kR];     // masked: 2^-7 * sum of v_j over the enabled pairs
    uint32_t call = 0;   // masked: enabled pairs
#pragma unroll
    for (int q = 0; q < K; ++q) {
        nb[q] = 0u;
#pragma unroll
        for (int r = 0; r < kR; ++r) {
            t[q][r] = 0.0;
            sg[q][r] = 0u;
        }
    }
#pragma unroll
    for (int r = 0; r < kR; ++r) tall[r] = 0.0;
    constexpr int kInd = (K == 1 ? kStep : 2) * kR;  // indicator registers: low words zero for the whole loop
    unsigned long long ind[kInd];
#pragma unroll
    for (int i = 0; i < kInd; ++i) ind[i] = 0ull;

    uint32_t amb_steps = 0;  // warp-uniform
    static_assert(kGroup / kStep <= 32, "one bit per step");
#pragma unroll 1
    for (int jj = 0; jj < kGroup; jj += kStep) {
        float mn = 1.0f;  // min |d_q| over the enabled pairs of the step
#pragma unroll
        for (int u = 0; u < kStep; u += 2) {
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
                // {n, n} packed at the use: the FFMA2 takes the one register for both halves
                const unsigned long long d2 = ffma2(pack2(nx[r], nx[r]), xy.x,
                                                    ffma2(pack2(ny[r], ny[r]), xy.y, ffma2(pack2(nz[r], nz[r]), zz, e2)));
                bool on0 = true, on1 = true;
                if constexpr (kMasked) {
                    on0 = mk.on(r, jj + u);
                    on1 = mk.on(r, jj + u + 1);
                    call += (on0 ? 1u : 0u) + (on1 ? 1u : 0u);
                    if constexpr (kWeighted) {
                        tall[r] = fma(v0, __hiloint2double(on0 ? 0x3f800000 : 0, 0), tall[r]);
                        tall[r] = fma(v1, __hiloint2double(on1 ? 0x3f800000 : 0, 0), tall[r]);
                    }
                }
#pragma unroll
                for (int q = 0; q < K; ++q) {
                    const unsigned long long dq2 = q == 0 ? d2 : fadd2(d2, dl2[q]);
                    const float a = lo32(dq2), b = hi32(dq2);
                    if constexpr (kWeighted && !kMasked) {
                        unsigned long long &g0 = ind[(u * kR + 2 * r) % kInd], &g1 = ind[(u * kR + 2 * r + 1) % kInd];
                        t[q][r] = fma(v0, ind_gt0_f64(g0, a), t[q][r]);
                        t[q][r] = fma(v1, ind_gt0_f64(g1, b), t[q][r]);
                    } else if constexpr (kWeighted) {
                        float i0 = ind_gt0(a), i1 = ind_gt0(b);
                        i0 = on0 ? i0 : 0.f;
                        i1 = on1 ? i1 : 0.f;
                        t[q][r] = fma(v0, __hiloint2double(__float_as_int(i0), 0), t[q][r]);
                        t[q][r] = fma(v1, __hiloint2double(__float_as_int(i1), 0), t[q][r]);
                    } else {
                        uint32_t ba = __float_as_uint(a), bb = __float_as_uint(b);
                        if constexpr (kMasked) {
                            ba = on0 ? ba : 0x80000000u;
                            bb = on1 ? bb : 0x80000000u;
                        }
                        asm("shf.l.wrap.b32 %0, %1, %0, 1;" : "+r"(sg[q][r]) : "r"(ba));
                        asm("shf.l.wrap.b32 %0, %1, %0, 1;" : "+r"(sg[q][r]) : "r"(bb));
                    }
                    float aa = fabsf(a), ab = fabsf(b);
                    if constexpr (kMasked) {
                        aa = on0 ? aa : 1.0f;
                        ab = on1 ? ab : 1.0f;
                    }
                    asm("min.f32 %0, %0, %1, %2;" : "+f"(mn) : "f"(aa), "f"(ab));
                }
            }
        }
        // a pair within the guard band of an edge: the step is noted and redone exactly after the loop
        if (__any_sync(0xffffffffu, !(mn > G))) amb_steps |= 1u << (jj / kStep);
        if constexpr (!kWeighted) {
            if ((jj & 31) == 32 - kStep) {
#pragma unroll
                for (int q = 0; q < K; ++q)
#pragma unroll
                    for (int r = 0; r < kR; ++r) nb[q] += __popc(sg[q][r]);
            }
        }
    }

    if (amb_steps) {
        // exact corrections, applied to the (exact) accumulators before anything is read from them
        double dt[kChunk * kR];
        int dn[kChunk];
        fixup_chunk<kWeighted>(p, grp2, vgrp, amb_steps, K, m_a, kMasked, mk, i_base, j_first, stat, dt, dn);
#pragma unroll
        for (int q = 0; q < K; ++q) {
            if constexpr (kWeighted) {
#pragma unroll
                for (int r = 0; r < kR; ++r) t[q][r] += dt[q * kR + r];
            } else {
                nb[q] += (uint32_t)dn[q];
            }
        }
    }
    // ---- this thread's tallies -> row contributions -> the warp's rows
    auto unpack = [&](double tt, uint32_t &n) -> double {  // 2^-7 (n C + sum of w) -> sum of w, n += count
        double sw = tt * 128.0;
        if constexpr (kWeighted) {
            const double nn = floor(sw * rows.pack->inv_C);  // C is a power of two and the sum of w is below C: exact
            sw -= nn * rows.pack->C;
            n += (uint32_t)nn;
        }
        return sw;
    };
    if constexpr (kDeferFix) {
        // the kernel's own loop: one edge, nothing masked; the two rows' tallies stay with the thread
        static_assert(K == 1 && !kMasked, "");
        uint32_t c_hi = kWeighted ? 0u : (uint32_t)(kGroup * kR) - nb[0];
        double w_lo = 0.0, w_hi = 0.0;
        if constexpr (kWeighted) {
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                const double sw = unpack(t[0][r], c_hi);
                w_lo = fma((double)wi[r], wsum_j - sw, w_lo);
                w_hi = fma((double)wi[r], sw, w_hi);
            }
        }
        const uint32_t c_lo = (uint32_t)(kGroup * kR) - c_hi;
        tally->c_lo += c_lo;
        tally->c_hi += c_hi;
        if (c_lo != 0u) tally->w_lo += w_lo;  // no pair of this thread in the row: not even a rounding residue
        if (c_hi != 0u) tally->w_hi += w_hi;
        return 0u;
    }
    uint32_t c_prev = 0;  // this thread's pairs above the previous edge (all its pairs before the first)
    double s_prev[kR];    // and, per i-point, the sum of their w_j
    if (first) {
        if constexpr (kMasked) {
            uint32_t n_unused = 0;
            c_prev = call;
#pragma unroll
            for (int r = 0; r < kR; ++r) s_prev[r] = kWeighted ? unpack(tall[r], n_unused) : 0.0;
        } else {
            c_prev = (uint32_t)(kGroup * kR);
#pragma unroll
            for (int r = 0; r < kR; ++r) s_prev[r] = wsum_j;
        }
    } else {
        c_prev = carry->c;
#pragma unroll
        for (int r = 0; r < kR; ++r) s_prev[r] = carry->s[r];
    }
    __syncwarp();
#pragma unroll
    for (int q = 0; q <= K; ++q) {
        if (q == K && !last) break;
        uint32_t c_q = 0;  // pairs above edge q (q == K: nothing lies above the row after the last edge)
        double rw = 0.0;   // weight of this thread's pairs in row m_a + q
        if (q < K) {
            if constexpr (kWeighted) {
                c_q = 0u;
#pragma unroll
                for (int r = 0; r < kR; ++r) {
                    const double sw = unpack(t[q][r], c_q);
                    rw = fma((double)wi[r], s_prev[r] - sw, rw);
                    s_prev[r] = sw;
                }
            } else {
                c_q = (uint32_t)(kGroup * kR) - nb[q];
            }
        } else if constexpr (kWeighted) {
#pragma unroll
            for (int r = 0; r < kR; ++r) rw = fma((double)wi[r], s_prev[r], rw);
        }
        const uint32_t rc = c_prev - c_q;
        c_prev = c_q;
        if (rc == 0u) rw = 0.0;  // no pair of this thread in the row: not even a rounding residue
        const uint32_t rc_warp = __reduce_add_sync(0xffffffffu, rc);
        if constexpr (kWeighted) rw = warp_sum_f64(rw);
        if (lane == 0) {
            rows.template add<kWeighted>(m_a + q, rc_warp, rw);
        }
    }
    if (!last) {
        carry->c = c_prev;
#pragma unroll
        for (int r = 0; r < kR; ++r) carry->s[r] = s_prev[r];
    }
    __syncwarp();
    return 0u;
}

// One group: all edges r_lo .. r_hi - 1 of its window, kChunk at a time.
#define ACF_WIN_CHUNK_CALL(K, MASKED) \
    window_chunk<K, kWeighted, MASKED>(p, rows, grp2, vgrp, nx, ny, nz, wi, m, m == r_lo, left <= K, wsum_j, mk, i_base, j_first, stat, \
                                                nullptr, &carry)
// Not inlined: only the common case (one edge, nothing masked) lives in the kernel's own loop, so that
// the register allocation of that loop is not set by the rare variants.  It reloads the i-points.
template <bool kWeighted>
__device__ __noinline__ void window_group(const WinParams &p, const Rows rows, const float *__restrict__ grp2,
                                          const double *__restrict__ vgrp, int r_lo, int r_hi,
                                          double wsum_j, bool masked, const Mask mk, uint32_t i_base, uint32_t j_first,
                                          unsigned long long *stat)
{
    float nx[kR], ny[kR], nz[kR], wi[kR];
#pragma unroll
    for (int r = 0; r < kR; ++r) {
        const float4 v = p.pts_a[i_base + local_i(r)];  // the array is padded to a whole tile
        nx[r] = -v.x;
        ny[r] = -v.y;
        nz[r] = -v.z;
        wi[r] = v.w;
    }
    static_assert(kChunk == 3, "the dispatch below spells the chunk sizes out");
    if (r_hi == r_lo) {  // one row: still every pair is evaluated, against the edge that bounds the row
        if (r_lo > p.nbins) r_lo = p.nbins;
        r_hi = r_lo + 1;
    }
    Carry carry;
    carry.c = 0u;
#pragma unroll
    for (int r = 0; r < kR; ++r) carry.s[r] = 0.0;
    int m = r_lo;  // edges below m are done
    while (m < r_hi) {
        const int left = r_hi - m;
        if (masked) {
            if (left == 1) ACF_WIN_CHUNK_CALL(1, true);
            else if (left == 2) ACF_WIN_CHUNK_CALL(2, true);
            else ACF_WIN_CHUNK_CALL(3, true);
        } else {
            if (left == 1) ACF_WIN_CHUNK_CALL(1, false);
            else if (left == 2) ACF_WIN_CHUNK_CALL(2, false);
            else ACF_WIN_CHUNK_CALL(3, false);
        }
        m += left < kChunk ? left : kChunk;
    }
}
#undef ACF_WIN_CHUNK_CALL

// ---- the kernel ---------------------------------------------------------------------------------
// kWarps consumer warps and no producer warp (16 warps leave each thread 128 registers; a 17th would cost
// 32 of them).  The j-tiles of the work items {i-tile, first j-tile, number of j-tiles} stream through a
// ring of shared-memory stages filled by TMA bulk copies (full / empty mbarriers per stage).  Whichever
// warp finds the ring's lock free refills the drained stages -- after it hands a stage back, and while it
// waits for one -- pulling work items from a global counter.  Every warp walks the stream at its own
// pace, holding its kGroup i-points of the current i-tile in registers.
struct ProdState {
    uint32_t lock;      // 0 free, 1 held
    uint32_t produced;  // stages filled so far: slot = produced % n_stages, round = produced / n_stages
    int ti, tj, left;   // the work item being streamed: its i-tile, next j-tile, j-tiles left
    int done;           // the end-of-stream stage has been posted
    unsigned long long n_items;
};

template <bool kWeighted>
__device__ __forceinline__ void try_produce(const WinParams &p, volatile ProdState *ps, uint64_t *full, uint64_t *empty,
                                            StageMeta *meta, unsigned char *stages, int n_stages)
{
    constexpr size_t kStage = stage_bytes(kWeighted);
    if (ps->done || atomicCAS(const_cast<uint32_t *>(&ps->lock), 0u, 1u) != 0u) return;
    while (!ps->done) {
        const uint32_t produced = ps->produced;
        const int slot = (int)(produced % (uint32_t)n_stages);
        const uint32_t round = produced / (uint32_t)n_stages;
        if (!mbar_test(&empty[slot], (round & 1u) ^ 1u)) break;  // not drained yet (round 0 passes at once)
        if (ps->left == 0) {
            const unsigned long long item = atomicAdd(&p.counters[kCtrWorkHead], 1ull);
            if (item >= ps->n_items) {  // end of stream
                StageMeta m;
                m.ti = -1;
                m.tj = m.jn = m.pad = 0;
                meta[slot] = m;
                ps->done = 1;
                ps->produced = produced + 1;
                mbar_arrive(&full[slot]);
                break;
            }
            const int3 it = p.items[item];
            ps->ti = it.x;
            ps->tj = it.y;
            ps->left = it.z;
        }
        const int tj = ps->tj;
        const uint32_t j0 = (uint32_t)tj * kTile;
        const uint32_t jn = p.n_b - j0 < (uint32_t)kTile ? p.n_b - j0 : (uint32_t)kTile;
        StageMeta m;
        m.ti = ps->ti;
        m.tj = tj;
        m.jn = (int)jn;
        m.pad = 0;
        meta[slot] = m;
        ps->tj = tj + 1;
        ps->left = ps->left - 1;
        ps->produced = produced + 1;
        // the arrays are padded to whole tiles: always a full tile
        mbar_expect_tx(&full[slot], (uint32_t)kStage);
        bulk_load(stages + (size_t)slot * kStage, p.pts2_b + (size_t)j0 * 4, (uint32_t)kTileBytes, &full[slot]);
        if constexpr (kWeighted)
            bulk_load(stages + (size_t)slot * kStage + kTileBytes, p.vj_b + (size_t)j0, (uint32_t)kVjBytes, &full[slot]);
    }
    __threadfence_block();
    atomicExch(const_cast<uint32_t *>(&ps->lock), 0u);
}

template <bool kWeighted>
__global__ void __launch_bounds__(kThreads, 1) pair_win_kernel(const WinParams p)
{
    if (p.counters[kCtrBadInput] != 0) return;  // inputs failed validation
    if (kWeighted && p.pack_b->packed == 0) return;  // weights that do not pack: the table kernel does the call
    extern __shared__ __align__(128) unsigned char smem[];
    const int rows_n = p.nbins + 2;
    const int n_stages = p.n_stages;
    constexpr size_t kStage = stage_bytes(kWeighted);
    // layout: [full bars | empty bars | stage meta | producer state] (512 B) [stages][count rows per warp][weight rows per warp]
    uint64_t *full = reinterpret_cast<uint64_t *>(smem);
    uint64_t *empty = full + kMaxStages;
    StageMeta *meta = reinterpret_cast<StageMeta *>(smem + 128);
    volatile ProdState *ps = reinterpret_cast<volatile ProdState *>(smem + 128 + kMaxStages * sizeof(StageMeta));
    unsigned long long *stat = reinterpret_cast<unsigned long long *>(smem + 128 + kMaxStages * sizeof(StageMeta) + sizeof(ProdState));
    PackInfo *pack_sm = reinterpret_cast<PackInfo *>(stat + kNumStats);
    static_assert(sizeof(ProdState) % 8 == 0 &&
                      128 + kMaxStages * sizeof(StageMeta) + sizeof(ProdState) + kNumStats * 8 + sizeof(PackInfo) <= kSmemHeader,
                  "header");
    unsigned char *stages = smem + kSmemHeader;
    size_t off = kSmemHeader + (size_t)n_stages * kStage;
    uint32_t *cnt_all = reinterpret_cast<uint32_t *>(smem + off);
    const int row_sets = p.shared_rows ? 1 : kWarps;
    off += (size_t)row_sets * rows_n * sizeof(uint32_t);
    off = (off + 15) & ~size_t(15);
    double *ws_all = reinterpret_cast<double *>(smem + off);
    if constexpr (kWeighted) off += (size_t)row_sets * rows_n * sizeof(double);
    WinRows *win_all = reinterpret_cast<WinRows *>(smem + off);
    off += (size_t)kWarps * kGroupsPerTile * sizeof(WinRows);
    double *edges_sm = reinterpret_cast<double *>(smem + off);  // the edges, for the windows' row searches

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int igrp = warp & (kTeamWarps - 1), team = warp / kTeamWarps;
    for (int i = tid; i < row_sets * rows_n; i += blockDim.x) {
        cnt_all[i] = 0;
        if constexpr (kWeighted) ws_all[i] = 0.0;
    }
    for (int i = tid; i <= p.nbins; i += blockDim.x) edges_sm[i] = p.edges[i];
    if (tid == 0) {
        for (int s = 0; s < n_stages; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], kWarps);
        }
        ps->lock = 0;
        ps->produced = 0;
        ps->ti = ps->tj = ps->left = 0;
        ps->done = 0;
        unsigned long long n_items = p.counters[kCtrWorkCount];
        ps->n_items = n_items > p.capacity ? p.capacity : n_items;
        for (int i = 0; i < kNumStats; ++i) stat[i] = 0ull;
        *pack_sm = *p.pack_b;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (tid == 0) try_produce<kWeighted>(p, ps, full, empty, meta, stages, n_stages);

    // ---------------- consumers
    Rows rows;
    rows.shared = p.shared_rows != 0;
    rows.pack = pack_sm;
    rows.cnt = cnt_all + (rows.shared ? 0 : (size_t)warp * rows_n);
    rows.ws = ws_all + (rows.shared ? 0 : (size_t)warp * rows_n);
    WinRows *win = win_all + (size_t)warp * kGroupsPerTile;
    uint32_t since_flush = 0;  // j-tiles this warp has tallied in its unflushed rows
    // u32 rows: flush before the tallies could wrap (shared rows take the pairs of all the CTA's warps)
    // (the rows are read as signed 32-bit numbers when flushed: half the range)
    const uint32_t flush_every = (1u << 30) / (uint32_t)(kGroup * kTile) / (rows.shared ? (uint32_t)kWarps : 1u);
    float wi[kR];
    float nx[kR], ny[kR], nz[kR];  // the i-points, negated
#pragma unroll
    for (int r = 0; r < kR; ++r) wi[r] = nx[r] = ny[r] = nz[r] = 0.f;
    uint32_t valid_mask = 0, i_base = 0, n_i = 0;
    bool warp_full = false, warp_any = false;
    int cur_ti = -1;

    LaneTally tally{0u, 0u, 0.0, 0.0};
    int tally_m = -1;  // the edge the tally belongs to (warp-uniform)
    auto flush_tally = [&]() {
        // the threads' tallies of rows tally_m and tally_m + 1 -> the warp's rows
        if (tally_m >= 0) {
            const uint32_t c_lo = __reduce_add_sync(0xffffffffu, tally.c_lo), c_hi = __reduce_add_sync(0xffffffffu, tally.c_hi);
            double w_lo = 0.0, w_hi = 0.0;
            if constexpr (kWeighted) {
                w_lo = warp_sum_f64(tally.w_lo);
                w_hi = warp_sum_f64(tally.w_hi);
            }
            if (lane == 0) {
                rows.template add<kWeighted>(tally_m, c_lo, w_lo);
                rows.template add<kWeighted>(tally_m + 1, c_hi, w_hi);
            }
            tally = LaneTally{0u, 0u, 0.0, 0.0};
            tally_m = -1;
        }
    };
    auto flush_rows = [&]() {
        // this warp's rows -> global (u64 / f64 atomics); the rows restart from zero
        flush_tally();
        __syncwarp();
        for (int row = lane; row < rows_n; row += 32) {
            // (shared rows: other warps add while this one takes the value and leaves zero)
            const uint32_t v = rows.shared ? atomicExch(&rows.cnt[row], 0u) : rows.cnt[row];
            if (!rows.shared) rows.cnt[row] = 0;
            // read as signed: with shared rows another warp's exact correction (-1 now, its tally later) may be
            // caught in between; the two's-complement sum in global memory comes out the same
            if (row >= 1 && row <= p.nbins && v) atomicAdd(&p.counts[row - 1], (unsigned long long)(long long)(int32_t)v);
            if constexpr (kWeighted) {
                const double w = rows.shared ? __longlong_as_double((long long)atomicExch(reinterpret_cast<unsigned long long *>(&rows.ws[row]), 0ull))
                                             : rows.ws[row];
                if (!rows.shared) rows.ws[row] = 0.0;
                if (row >= 1 && row <= p.nbins && w != 0.0) atomicAdd(&p.wsums[row - 1], w);
            }
        }
        __syncwarp();
        since_flush = 0;
    };

    for (uint32_t consumed = 0;; ++consumed) {
        const int slot = (int)(consumed % (uint32_t)n_stages);
        const uint32_t parity = (consumed / (uint32_t)n_stages) & 1u;
        if (lane == 0)
            while (!mbar_test(&full[slot], parity)) {
                try_produce<kWeighted>(p, ps, full, empty, meta, stages, n_stages);
                if (!mbar_test(&full[slot], parity)) __nanosleep(100);  // leave the issue slots to the warps that have work
            }
        __syncwarp();
        mbar_wait(&full[slot], parity);  // every lane observes the completed phase
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
                nx[r] = -v.x;
                ny[r] = -v.y;
                nz[r] = -v.z;
                wi[r] = v.w;
                valid_mask |= (s < p.n_a ? 1u : 0u) << r;
            }
            n_i = i_base + kTile <= p.n_a ? kTile : p.n_a - i_base;
            warp_full = (uint32_t)(igrp + 1) * kGroup <= n_i;
            warp_any = (uint32_t)igrp * kGroup < n_i;
        }
        const float *tile = reinterpret_cast<const float *>(stages + (size_t)slot * kStage);
        const double *vtile = reinterpret_cast<const double *>(stages + (size_t)slot * kStage + kTileBytes);
        const int tj = m.tj, jn = m.jn;
        const bool diag = p.is_auto && tj == m.ti;
        const uint32_t j_base = (uint32_t)tj * kTile;
        // u32 rows: flush before this warp's tallies could wrap
        if (since_flush >= flush_every) flush_rows();
        ++since_flush;

        if (warp_any) {
            // lane l bounds the rows of this warp's i-group against the team's l-th j-group of the tile
            const int n_groups = (jn + kGroup - 1) / kGroup;
            __syncwarp();
            const int my_g = lane * kTeams + team;
            if (lane < kGroupsPerTile / kTeams && my_g < n_groups) {
                WinRows wr;
                wr.lo = 0;
                wr.hi = p.nbins + 1;
                const GroupCap gb = p.gcaps_b[(size_t)tj * kGroupsPerTile + my_g];
                double c_lo, c_hi;
                if (cap_window(p.gcaps_a[(size_t)m.ti * kGroupsPerTile + igrp], gb, c_lo, c_hi)) {
                    // rows of the two ends; the far end is a few rows on at most: walk there
                    int hi = wr.lo = row_of_cos(c_hi, edges_sm, p.nbins);
                    while (hi < p.nbins && c_lo <= edges_sm[hi]) ++hi;
                    if (hi == p.nbins && c_lo < edges_sm[p.nbins]) ++hi;
                    wr.hi = hi;
                }
                if (p.prune && wr.hi == wr.lo && (wr.lo == 0 || wr.lo > p.nbins) && !(diag && my_g < igrp)) {
                    // all closer than theta_min or all beyond theta_max: pruned at the level of groups, like whole
                    // tiles in the work list; the tile's pair count in the statistics loses them
                    const uint32_t gi = n_i - (uint32_t)igrp * kGroup < (uint32_t)kGroup ? n_i - (uint32_t)igrp * kGroup : (uint32_t)kGroup;
                    const uint32_t gj = (uint32_t)(jn - my_g * kGroup < kGroup ? jn - my_g * kGroup : kGroup);
                    const unsigned long long gone = diag && my_g == igrp ? (unsigned long long)gi * (gi - 1) / 2 : (unsigned long long)gi * gj;
                    atomicAdd(&stat[kStatEvaluated], 0ull - gone);
                    wr.lo = wr.hi = -1;
                }
                if (p.bulk && wr.lo >= 0 && wr.hi == wr.lo && warp_full && jn - my_g * kGroup >= kGroup && !(diag && my_g <= igrp)) {
                    // all pairs of two full groups in one bin: the bin gets the groups' pair count and the product of
                    // their weight sums, and nothing is evaluated (ACF_OPT_BULK)
                    const unsigned long long all = (unsigned long long)kGroup * kGroup;
                    rows.template add_atomic<kWeighted>(wr.lo, (uint32_t)all, p.gcaps_a[(size_t)m.ti * kGroupsPerTile + igrp].wsum * gb.wsum);
                    atomicAdd(&stat[kStatEvaluated], 0ull - all);
                    atomicAdd(&stat[kStatBulk], all);
                    wr.lo = wr.hi = -1;
                }
                const int m_one = wr.hi > wr.lo ? wr.lo : (wr.lo > p.nbins ? p.nbins : (wr.lo < 0 ? 0 : wr.lo));
                wr.e32 = (float)edges_sm[m_one];
                wr.pad = 0;
                wr.wsum = gb.wsum;
                win[my_g] = wr;
            }
            __syncwarp();
            // pass 1: the common groups (one edge, nothing masked), inline; the others are noted in slow_groups
            uint32_t slow_groups = 0;
            for (int g = diag ? igrp : 0; g < n_groups; ++g) {
                if ((g & (kTeams - 1)) != team) continue;  // the other team's group
                const int r_lo = win[g].lo, r_hi = win[g].hi;
                if (r_lo < 0) continue;  // pruned (see where the windows are bounded)
                const bool masked = !warp_full || jn - g * kGroup < kGroup || (diag && g == igrp);
                if (masked || r_hi - r_lo > 1) {
                    slow_groups |= 1u << g;
                    continue;
                }
                // a window inside one row is tested against the edge that bounds the row
                const int m_edge = r_hi > r_lo ? r_lo : (r_lo > p.nbins ? p.nbins : r_lo);
                Mask mk{};
                if (m_edge != tally_m) {
                    flush_tally();
                    tally_m = m_edge;
                }
                window_chunk<1, kWeighted, false, true>(p, rows, tile + (size_t)g * kGroup * 4, vtile + g * kGroup,
                                                                                      nx, ny, nz, wi, m_edge, true, true, win[g].wsum, mk,
                                                                                      i_base, j_base + g * kGroup, stat, &tally, nullptr,
                                                                                      win[g].e32);
                if (lane == 0) atomicAdd(&stat[kStatWindow], (unsigned long long)(kGroup * kGroup));
            }
            // pass 2: the rest through the function; it reloads the i-points, and so does this loop afterwards
            // (they are not kept in registers across the calls)
            if (slow_groups) {
                for (int g = 0; g < n_groups; ++g) {
                    if (!((slow_groups >> g) & 1u)) continue;
                    const int r_lo = win[g].lo, r_hi = win[g].hi;
                    Mask mk;
                    mk.valid = valid_mask;
                    mk.jn = jn - g * kGroup < kGroup ? jn - g * kGroup : kGroup;
                    mk.j0 = g * kGroup;
                    mk.diag = diag && g == igrp;
                    const bool masked = !warp_full || mk.jn < kGroup || mk.diag;
                    window_group<kWeighted>(p, rows, tile + (size_t)g * kGroup * 4, vtile + g * kGroup, r_lo, r_hi, win[g].wsum,
                                                     masked, mk, i_base, j_base + g * kGroup, stat);
                    if (lane == 0 && !masked && r_hi - r_lo <= 1) atomicAdd(&stat[kStatWindow], (unsigned long long)(kGroup * kGroup));
                }
#pragma unroll
                for (int r = 0; r < kR; ++r) {
                    const float4 v = p.pts_a[i_base + local_i(r)];
                    nx[r] = -v.x;
                    ny[r] = -v.y;
                    nz[r] = -v.z;
                    wi[r] = v.w;
                }
            }
        }
        if (tid == 0) atomicAdd(&stat[kStatEvaluated], diag ? (unsigned long long)n_i * (n_i - 1) / 2 : (unsigned long long)n_i * (unsigned)jn);
        __syncwarp();  // every lane has read the stage before it is handed back
        if (lane == 0) {
            mbar_arrive(&empty[slot]);
            try_produce<kWeighted>(p, ps, full, empty, meta, stages, n_stages);
        }
    }

    flush_rows();
    __syncthreads();
    if (tid == 0) {
        if (stat[kStatFp64]) atomicAdd(&p.counters[kCtrPairsFp64], stat[kStatFp64]);
        if (stat[kStatWindow]) atomicAdd(&p.counters[kCtrPairsWindow], stat[kStatWindow]);
        if (stat[kStatEvaluated]) atomicAdd(&p.counters[kCtrPairsEvaluated], stat[kStatEvaluated]);
        if (stat[kStatChord]) atomicAdd(&p.counters[kCtrPairsChord], stat[kStatChord]);
        if (stat[kStatBulk]) atomicAdd(&p.counters[kCtrPairsBulk], stat[kStatBulk]);
    }
}

}  // namespace

// Launches the window kernel on the work items of the context's work list.
int launch_pair_win(acf_ctx *ctx, const Prepared &a, const Prepared &b, int is_auto, int nbins, uint32_t capacity,
                    unsigned long long *d_counts, double *d_wsums)
{
    const bool weighted = d_wsums != nullptr;
    const int rows_n = nbins + 2;
    int row_sets = kWarps;  // a set of rows per warp, or one per CTA when that leaves no room for the ring
    auto smem_for = [&](int stages) {
        size_t m = kSmemHeader + (size_t)stages * stage_bytes(weighted);
        m += (size_t)row_sets * rows_n * sizeof(uint32_t);
        m = (m + 15) & ~size_t(15);
        if (weighted) m += (size_t)row_sets * rows_n * sizeof(double);
        m += (size_t)kWarps * kGroupsPerTile * sizeof(WinRows);
        m += sizeof(double) * (size_t)(nbins + 1);
        return m;
    };
    // one CTA of 16 warps per SM: 128 registers a thread
    const int ctas_per_sm = 1;
    const size_t budget = (size_t)ctx->max_smem_optin;
    if (smem_for(4) > budget) row_sets = 1;
    if (smem_for(2) > budget) return fail(ctx, ACF_EINVAL, "too many bins for the window kernel (%d)", nbins);
    int n_stages = 2;
    while (n_stages < kMaxStages && smem_for(n_stages + 1) <= budget) ++n_stages;
    const size_t smem = smem_for(n_stages);

    WinParams p{};
    p.pts_a = a.pts;
    p.pts2_b = b.pts2;
    p.vj_b = b.vj;
    p.pack_b = b.pack;
    p.perm_a = a.perm;
    p.perm_b = b.perm;
    p.gcaps_a = a.gcaps;
    p.gcaps_b = b.gcaps;
    p.n_a = (uint32_t)a.n;
    p.n_b = (uint32_t)b.n;
    p.xyz_a = a.xyz;
    p.xyz_b = b.xyz;
    p.stride_a = a.stride;
    p.stride_b = b.stride;
    p.items = ctx->s_work.as<int3>();
    p.capacity = capacity;
    p.edges = ctx->s_edges.as<double>();
    p.sedges = ctx->d_sedges;
    p.nbins = nbins;
    p.counts = d_counts;
    p.wsums = d_wsums;
    p.counters = ctx->d_counters;
    p.is_auto = is_auto;
    p.n_stages = n_stages;
    p.shared_rows = row_sets == 1 ? 1 : 0;
    p.prune = ctx->opt_prune;
    p.bulk = ctx->opt_bulk;

    const int grid = ctx->num_sms * ctas_per_sm;
    cudaError_t e = cudaSuccess;
    auto launch = [&](auto kern) {
        if (e != cudaSuccess) return;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) kern<<<grid, kThreads, smem, ctx->stream>>>(p);
        ctx->last.kernel_launches++;
    };
    if (weighted) {
        launch(pair_win_kernel<true>);  // returns at once if the j side's weights do not pack (acf_pair.cu)
    } else {
        launch(pair_win_kernel<false>);
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    ACF_CUDA_TRY(ctx, e);
    return ACF_OK;
}

}  // namespace acf
