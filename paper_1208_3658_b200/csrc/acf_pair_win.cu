// acf_pair_win.cu -- the window kernel: every pair classified against the bin edges that can matter
// for its window, tallies in registers, no per-pair shared-memory traffic.
//
// Points are sorted along a space-filling curve, so the kGroup i-points a warp holds and a group of kGroup
// (or a sub-group of kSub) j-points each sit in a small cap; the two caps bound the cosines of all their
// pairs to a window [c_lo, c_hi] (fp64, rigorous), i.e. to the histogram rows r_lo .. r_hi and the
// k = r_hi - r_lo edges e[r_lo] .. e[r_hi - 1] between them.  The edges are taken kChunk at a time.  Per
// pair and chunk, on the cosine:
//   d_0 = e_m - (x_i x_j + y_i y_j + z_i z_j)      three fp32 FMAs seeded with fp32(e_m)  (two j-points per FFMA2)
//   d_q = d_0 + fp32(e_{m+q} - e_m)                 one add per further edge of the chunk
//   above_q = d_q > 0                               the pair lies in a row beyond edge m + q
//   certified iff |d_q| > G for every q             else the exact fp64 row of include/acf.h decides
// or, for windows at small separations (1 - c_lo <= 2^-12, where the fp32 cosine cannot tell the edges
// apart: SURVEY.md section 7, hard part 2), on the squared chord length s = |u_i - u_j|^2 = 2 (1 - c) up to
// the norms, which does not cancel:
//   d_0 = (x_j - x_i)^2 + (y_j - y_i)^2 + (z_j - z_i)^2 - s_m      s_m = fp32(2 (1 - e_m)); three adds, three FMAs
//   d_q = d_0 + fp32(s_m - s_{m+q}),  above_q and the guard band as before, G = G(s_m) relative (chord_guard)
// Per i-point and edge one fp64 accumulator takes t += [above_q] v_j (v_j = C + w_j packs the count and
// the weight sum, see PackInfo: exact sums; weights of too wide a range for that are not tallied here
// but pair by pair in acf_pair.cu; unweighted counts shift the sign bits of d_q into a word instead).
// The accumulators are cumulative in q (above edge m + q implies above edge m + q - 1), so the rows get
// the differences of consecutive edges; they are formed per i-point before anything is summed.
// After a chunk the warp reduces its row tallies with shuffles and lane 0 adds them to the warp's rows in
// shared memory; those go to global memory with u64 / f64 atomics (block histograms summed
// into global memory -- here without a per-pair atomic, the 5-50 % serialisation the paper measures).
//
// Every warp works on its own: it takes jobs {i-group, run of work items} from a global counter, bounds the
// windows of its i-group against 16 j-groups at a time (one lane per j-group, fp64), drops the groups whose
// window lies out of range without loading them, splits a window of several edges by the
// j-side sub-group caps, and streams the surviving j-groups through its own ring of shared-memory stages with
// TMA bulk copies (one mbarrier per stage).  No barrier is shared between warps: a warp whose groups are all
// pruned runs ahead, one with many near-field groups takes its time, and neither waits for the other.
#include <cmath>
#include <cstring>

#include "acf_device.cuh"
#include "acf_internal.h"
#include "acf_pair_common.cuh"

namespace acf {

namespace {

constexpr int kWarps = 16;             // warps per CTA, each on its own stream of j-groups
constexpr int kThreads = 32 * kWarps;
constexpr int kR = kGroup / 32;        // i-points per thread
constexpr int kChunk = 3;              // edges per pass over a group
// j-points per guard-band vote (8 for unweighted counts saves 0.7 instructions per pair in the loop and measured
// 5 to 15 % slower on the clustered configurations: every flagged step re-derives twice the pairs)
__host__ __device__ constexpr int step_of(bool) { return 4; }
constexpr int kWStages = 2;            // staged j-groups per warp
constexpr int kQueue = 32;             // surviving j-groups a warp has bounded and not yet evaluated
constexpr int kScan = 16;              // j-groups bounded at a time (two tiles, one lane each)
constexpr int kMaxPassEdges = 3;       // unweighted: windows of more edges than this go pair by pair (general_span); weighted ones
                                       // take as many passes as it needs (their pair-by-pair tallies are fp64 atomics on shared memory)
// The cell table of the pair-by-pair path: the values of the fp32 squared chord length s that share their sign,
// exponent and top `bits` mantissa bits form a cell; 2^bits cells per octave from 2^exp_lo to 4.  The host picks both
// per call (cell_shape): exp_lo just below the first edge, and as many cells per octave as the narrowest bin needs to
// have a cell to itself, between 64 and 1024 for unweighted counts (which send the windows of more than kMaxPassEdges
// edges through the table) as far as the table stays within kCellBudget; weighted counts use the table for ragged and
// diagonal groups only and keep 16 cells per octave: their shared memory goes to their wider stages.
constexpr int kCellExpMin = -40;       // s below 2^-40 (0.2 arc seconds): never a cell, the edges are searched
constexpr size_t kCellBudget = 48 << 10;
struct CellShape {
    int bits, exp_lo, count;  // count = (2 - exp_lo) << bits cells; slot `count` stands for the values outside the table
    __host__ __device__ int slots() const { return count + 2; }  // (one more for 16-byte alignment)
};
struct Cell {
    float thr;      // the one edge s_k (as stored, fp32) that can separate two rows inside the cell; +big if none; NaN: the cell
                    // holds several edges (or is the slot of the values outside the table) and certifies nothing
    uint32_t word;  // bits 16..31: the guard band of that edge (the bound of chord_row) as the upper half of a float, rounded up:
                    // a pair is certified iff |s - thr| > guard;  bits 0..15: the row of s >= thr (s < thr is the row before)
};
static_assert(sizeof(Cell) == 8, "one LDS.64 per pair");
// What the pair loops keep of a CellShape: the shift of the float bits, the key of the first cell, the number of cells.
struct CellKey {
    uint32_t shift, key0, count;
    __device__ __forceinline__ explicit CellKey(const CellShape c)
        : shift((uint32_t)(23 - c.bits)), key0((uint32_t)(127 + c.exp_lo) << c.bits), count((uint32_t)c.count)
    {
    }
};
// The cell of the squared chord length s32 ...
__device__ __forceinline__ void cell_load(uint32_t cells, const CellKey ck, float s32, float &thr, uint32_t &word)
{
    // (zero, values below 2^exp_lo and NaN wrap or run past the table: all of them land in the slot after it)
    const uint32_t key = min((__float_as_uint(s32) >> ck.shift) - ck.key0, ck.count);
    asm volatile("ld.shared.v2.b32 {%0, %1}, [%2];" : "=f"(thr), "=r"(word) : "r"(cells + 8u * key));
}
// ... and its row by that cell; false if the cell does not certify it.
__device__ __forceinline__ bool cell_decide(float s32, float thr, uint32_t word, int &row)
{
    const float d = s32 - thr;
    row = (int)(word & 0xffffu) + (__float_as_int(d) >> 31);
    // (the whole word as the float: the row in its low half adds less than 2^-7 of the guard band to it, on the safe side)
    return fabsf(d) > __uint_as_float(word);
}
__device__ __forceinline__ bool cell_row(uint32_t cells, const CellKey ck, float s32, int &row)
{
    float thr;
    uint32_t word;
    cell_load(cells, ck, s32, thr, word);
    return cell_decide(s32, thr, word, row);
}
// Guard bands on the cosine (u = 2^-24).  A wrong fp32 sign needs
// |d_0 - (e_m - c64)| >= |d_0|, so only pairs with a small |d_0| matter; for those the partial sums of the
// chain are below 1 + 2e-6 in magnitude (they differ from d_0 by products of coordinates whose absolute sum is
// at most 1 + 2e-6):
//   2^-25 [fp32(e_m)] + 2u (1 + 1e-6) [the six rounded coordinates] + 2 * 2^-24 [the two inner FMAs]
//   + 2^-24 |d_0| [the last FMA] + 4e-16 [c64 itself]  <=  2.69e-7.
// d_q, q >= 1, is the sum of a d_0 that is not small and a rounded offset: partial sums below 4 (three
// roundings of 2^-23), the offset (2^-24) and the six coordinates give 5.7e-7.
constexpr float kGuard1 = 3.0e-7f;
constexpr float kGuardK = 7.0e-7f;
// A window with an edge inside it is classified on the chord length when it is narrower than this in the cosine
// (and closer than 45 degrees).  A pair comes within the guard band of the edge with probability about 2 G / width --
// 6e-7 / width on the cosine, (2.5e-7 sqrt(s) + 6e-7 s) / width on the chord, s = 2 (1 - c) -- and costs some
// 1e4 thread-instructions of exact re-evaluation when it does, against 1.5 per pair for the chord's three extra adds:
// below a width of 4e-3 the chord is the cheaper test.  Windows that hold no edge are tested on the cosine: their
// pairs are near the edge that bounds their row only if the window itself is.
constexpr double kChordWidth = 4.0e-3;
constexpr double kChordCosMin = 0.7071;
static_assert(kGroup == kR * 32 && kSub == 32 && kR == kSubsPerGroup, "register slot r of a warp is sub-group r of its i-group");
static_assert(kGroup % 32 == 0 && 32 % step_of(false) == 0 && 32 % step_of(true) == 0 && kScan == 2 * kGroupsPerTile, "");

constexpr size_t kGroupBytes = (size_t)kGroup * sizeof(float4);   // a staged j-group: the paired fp32 records
constexpr size_t kGroupVjBytes = (size_t)kGroup * sizeof(double);  // and (weighted) its fp64 window weights
__host__ __device__ constexpr size_t wstage_bytes(bool weighted) { return kGroupBytes + (weighted ? kGroupVjBytes : 0); }

struct WinParams {
    const float4 *pts_a;
    const float *pts2_b;
    const double *vj_b;
    const PackInfo *pack_b;
    const uint32_t *perm_a, *perm_b;
    const GroupCap *gcaps_a, *gcaps_b, *scaps_b;
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
    int shared_rows;  // 1: one set of histogram rows per CTA instead of one per warp
    int prune;        // 1: groups whose window lies wholly out of range are not evaluated
    int bulk;         // 1: groups whose window lies wholly inside one bin are counted as a whole (ACF_OPT_BULK)
    int refine;       // 1: windows of two or more edges are split by the j side's sub-group caps
    CellShape cell;   // the cell table of the pair-by-pair path
};

// chord_row out of line: the exact corrections and the pair-by-pair paths call it from unrolled loops, and one copy of
// its search is what should be resident.
__device__ __noinline__ int chord_row_ool(float xi, float yi, float zi, float xj, float yj, float zj, const float *sed, int nbins, float margin)
{
    return chord_row(xi, yi, zi, xj, yj, zj, sed, nbins, margin);
}

// Shared-memory loads by 32-bit shared address: the loads of the pair loops are LDS whatever the compiler can
// prove about a pointer, and an address costs one register.
__device__ __forceinline__ ulonglong2 lds_u64x2(uint32_t a)
{
    ulonglong2 v;
    asm volatile("ld.shared.v2.u64 {%0, %1}, [%2];" : "=l"(v.x), "=l"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ unsigned long long lds_u64(uint32_t a)
{
    unsigned long long v;
    asm volatile("ld.shared.u64 %0, [%1];" : "=l"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ double2 lds_f64x2(uint32_t a)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ double lds_f64(uint32_t a)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ float lds_f32(uint32_t a)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
    return v;
}

// Tables of a launch in shared memory (per CTA): nbins + 1 cosine edges (fp64), then four fp32 arrays of the same
// length: the edges as squared chord lengths s_m (-1 / +inf at the poles), -s_m (the seed of the chord test), the
// guard band of the chord test against edge m alone, and against edge m inside a chunk of several.
struct Tables {
    uint32_t base;  // shared address of the edges
    int nbins;
    const unsigned long long *counters;  // for chord_margin, on the rare paths that need it
    __device__ __forceinline__ float margin() const { return chord_margin(counters); }
    __device__ __forceinline__ const double *edges_ptr() const
    {
        return reinterpret_cast<const double *>(__cvta_shared_to_generic(base));
    }
    __device__ __forceinline__ const float *sed_ptr() const { return reinterpret_cast<const float *>(edges_ptr() + (nbins + 1)); }
    __device__ __forceinline__ double edge(int m) const { return lds_f64(base + 8u * (uint32_t)m); }
    __device__ __forceinline__ uint32_t f32_base(int k) const { return base + 8u * (uint32_t)(nbins + 1) + 4u * (uint32_t)(k * (nbins + 1)); }
    __device__ __forceinline__ float sneg(int m) const { return lds_f32(f32_base(1) + 4u * (uint32_t)m); }
    __device__ __forceinline__ float gs1(int m) const { return lds_f32(f32_base(2) + 4u * (uint32_t)m); }
    __device__ __forceinline__ float gsk(int m) const { return lds_f32(f32_base(3) + 4u * (uint32_t)m); }
    // the cell table of general_span, after the four fp32 arrays (16-byte aligned)
    __device__ __forceinline__ uint32_t cells() const { return (f32_base(4) + 15u) & ~15u; }
};

__device__ __forceinline__ unsigned long long fadd2(unsigned long long a, unsigned long long b)
{
    unsigned long long d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ float lo32(unsigned long long v) { return __uint_as_float((uint32_t)v); }
__device__ __forceinline__ float hi32(unsigned long long v) { return __uint_as_float((uint32_t)(v >> 32)); }

// The comparison v > 0 written as 1.0f / 0.0f (SASS FSET.BF) into the high word of a 64-bit register whose low
// word is and stays zero: the register then reads as the double 2^-7 [v > 0] with no instruction spent on
// the low word.
__device__ __forceinline__ double ind_gt0_f64(unsigned long long &reg, float v)
{
    asm("{\n\t.reg .b32 lo, hi;\n\tmov.b64 {lo, hi}, %0;\n\tset.gt.f32.f32 hi, %1, 0f00000000;\n\tmov.b64 %0, {lo, hi};\n\t}"
        : "+l"(reg)
        : "f"(v));
    return __longlong_as_double((long long)reg);
}

// Guard band of the chord test against the stored s_m (acf_pair_common.cuh "chord tier"): |s32 - s| <=
// 2.4e-7 sqrt(s) + 3.1e-7 s + 6e-14 for the chain of chord_row; the chains here are seeded with -s_m (three
// roundings of partial sums no larger than max(s, s_m)) and, inside a chunk, add a rounded offset to a d_0 that
// is not small (2^-24 s_m each for the offset and the sum): 6e-7 s and 9e-7 s take that and the rounding of the
// stored s_m; the edge's own uncertainty (norms, fp64 chain) is `margin` on both sides, as in chord_row.
__device__ __forceinline__ float chord_guard(float se, float margin, bool in_chunk)
{
    if (!(se >= 0.f) || se > 3.0e38f) return 0.f;  // a pole: never within reach
    const float sm = se + margin;
    return 1.02f * (2.5e-7f * sqrtf(sm) + (in_chunk ? 9.0e-7f : 6.0e-7f) * sm + 1.0e-13f) + margin;
}

// This warp's histogram rows in shared memory.  Lane 0 adds the reduced tallies; the exact corrections, the
// bulk counts and the pair-by-pair path come from any lane and are atomic.
struct Rows {
    uint32_t *cnt;
    double *ws;
    const PackInfo *pack;  // the j side's PackInfo, copied to shared memory
    bool shared;  // one set of rows for the whole CTA (many bins): every update is atomic
    template <bool kWeighted>
    __device__ __forceinline__ void add_atomic(int row, uint32_t c, double w) const  // from any lane
    {
        // (by shared address: through the generic pointer the compiler emits a generic ATOM, ten times slower)
        asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(smem_u32(cnt + row)), "r"(c) : "memory");
        if constexpr (kWeighted) asm volatile("red.shared.add.f64 [%0], %1;" ::"r"(smem_u32(ws + row)), "d"(w) : "memory");
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

// One surviving j-group in a warp's queue: where it is, and the rows of its window (or of the windows of its
// kSubsPerGroup sub-groups).
struct Unit {
    uint32_t i_first;      // index in catalogue a of the first point of the i-group the window was bounded for
    uint32_t j_first;      // index in catalogue b of the group's first point
    int16_t lo[kSubsPerGroup], hi[kSubsPerGroup];  // rows; nsub == 1: of the whole group, in [0]; lo < 0: nothing to evaluate
    uint8_t nsub;          // 1 or kSubsPerGroup
    uint8_t masked;        // ragged group on either side, or the diagonal group of an auto-count
    uint8_t diag;          // count only pairs with (index of j) > (index of i)
    uint8_t chord;         // bit s: (sub-)window s is classified on the chord length
    int32_t jn;            // points of the j-group that exist
    double wsum[kSubsPerGroup];  // weight sums of the (sub-)groups
};
static_assert(sizeof(Unit) == 64, "");

__device__ __forceinline__ double warp_sum_f64(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// The j-points [jj0, jj1) of a staged group against this warp's i-group: what one pass works on.
// Thread `lane` holds the i-points i_first + r * 32 + lane, r < kR.
struct Span {
    uint32_t grp2;       // shared address of the staged group, paired layout
    uint32_t vgrp;       // shared address of its window weights
    int jj0, jj1;        // multiples of kSub
    double wsum;         // sum of the weights of the span's j-points
    uint32_t i_first;    // index in catalogue a of the i-group's first point
    uint32_t j_first;    // index in catalogue b of the staged group's first point
    uint32_t ipts;       // shared address of the warp's i-points {-x, -y, -z, w}, kGroup float4: thread `lane` reads r * 32 + lane
    // i-point r of this thread, negated
    __device__ __forceinline__ float4 ipoint(int r) const
    {
        const uint32_t a = ipts + 16u * (uint32_t)(r * 32 + (int)(threadIdx.x & 31u));
        float4 v;
        asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
        return v;
    }
    // point jj of the staged group
    __device__ __forceinline__ float4 point(int jj) const
    {
        const uint32_t a = grp2 + 32u * (uint32_t)(jj >> 1) + 4u * (uint32_t)(jj & 1);
        return make_float4(lds_f32(a), lds_f32(a + 8u), lds_f32(a + 16u), lds_f32(a + 24u));
    }
};

// Which pairs of a span count: ragged ends of the catalogues and the diagonal group of an auto-count.
struct Mask {
    uint32_t gi;  // i-points of the group that exist
    int jn;       // j-points of the group that exist
    bool diag;    // count only pairs with (index of j) > (index of i); both catalogues are the same then
    __device__ __forceinline__ bool on(const Span &sp, int r, int jj) const
    {
        const uint32_t il = (uint32_t)r * 32u + (threadIdx.x & 31u);
        return il < gi && jj < jn && (!diag || sp.j_first + (uint32_t)jj > sp.i_first + il);
    }
};

// The exact corrections of one chunk of a span, after its loop and before its tallies are read:
// amb_steps has a bit per step of kStep j-points in which some pair came within the guard band of an
// edge.  Every pair of those steps is re-derived bit for bit as the loop computed it; a pair within a
// guard band gets its row from the chord tier or the fp64 definition of include/acf.h, and where that
// disagrees with what the loop tallied, the correction of this thread's accumulators comes back:
//   dt[q * kR + r]  to add to t[q][r]: 2^-7 v_j for a pair that is above edge q after all, minus that for
//                   one that is not (the accumulators are exact sums, so the corrected tally is exactly the
//                   tally of the exact classification: no row ever sees a wrong pair added and taken back);
//   dn[q]           to add to nb[q] (unweighted: pairs not above edge q).
// One copy for all chunk shapes; it reloads the i-points rather than taking them in registers.
template <bool kWeighted, bool kChord>
__device__ __noinline__ void fixup_chunk(const WinParams &p, const Tables tb, const Span sp, uint32_t amb_steps, int K, int m_a,
                                         float G, unsigned long long *stat, double *__restrict__ dt, int *__restrict__ dn)
{
    const int lane = threadIdx.x & 31;
    for (int i = 0; i < kChunk * kR; ++i) dt[i] = 0.0;
    for (int i = 0; i < kChunk; ++i) dn[i] = 0;
    float e32, dl[kChunk];
    if constexpr (kChord) {
        e32 = tb.sneg(m_a);
#pragma unroll
        for (int q = 0; q < kChunk; ++q) dl[q] = q > 0 && q < K ? __fsub_rn(tb.sneg(m_a + q), e32) : 0.f;
    } else {
        const double e0 = tb.edge(m_a);
        e32 = edge32(e0);
#pragma unroll
        for (int q = 0; q < kChunk; ++q) dl[q] = q > 0 && q < K ? (tb.edge(m_a + q) <= -1.0 ? -8.0f : (float)(tb.edge(m_a + q) - e0)) : 0.f;
    }
    while (amb_steps) {
        constexpr int kStep = step_of(kWeighted);
        const int jj0 = sp.jj0 + (__ffs(amb_steps) - 1) * kStep;
        amb_steps &= amb_steps - 1;
        // (rolled loops: this code runs for one unit in three and should be short)
#pragma unroll 1
        for (int u = 0; u < kStep; ++u) {
            const float4 pj = sp.point(jj0 + u);
#pragma unroll 1
            for (int r = 0; r < kR; ++r) {
                float4 pir = sp.ipoint(r);  // negated in the stash
                pir.x = -pir.x;
                pir.y = -pir.y;
                pir.z = -pir.z;
                float d0;
                if constexpr (kChord) {
                    const float dx = __fadd_rn(pj.x, -pir.x), dy = __fadd_rn(pj.y, -pir.y), dz = __fadd_rn(pj.z, -pir.z);
                    d0 = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, e32)));
                } else {
                    d0 = fmaf(-pir.x, pj.x, fmaf(-pir.y, pj.y, fmaf(-pir.z, pj.z, e32)));
                }
                bool amb = false;
#pragma unroll
                for (int q = 0; q < kChunk; ++q) amb |= q < K && !(fabsf(q == 0 ? d0 : __fadd_rn(d0, dl[q])) > G);
                if (!amb) continue;
                // on the cosine, the chord length decides where it can; what is left open, the definition does
                int exact = kChord ? -1 : chord_row_ool(pir.x, pir.y, pir.z, pj.x, pj.y, pj.z, tb.sed_ptr(), tb.nbins, tb.margin());
                if (exact < 0) {
                    exact = exact_row(p.xyz_a, p.stride_a, p.perm_a[sp.i_first + r * 32 + lane], p.xyz_b, p.stride_b,
                                      p.perm_b[sp.j_first + jj0 + u], p.edges, p.nbins);
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
                        if constexpr (kWeighted) dt[q * kR + r] += (exact_above ? 0.0078125 : -0.0078125) * lds_f64(sp.vgrp + 8u * (uint32_t)(jj0 + u));
                        else dn[q] += exact_above ? -1 : 1;
                    }
                }
            }
        }
    }
}

// What a thread carries from one chunk of a window's edges to the next (registers of window_multi): its
// pairs above the last edge done and, per i-point, the sum of their w_j.
struct Carry {
    uint32_t c;
    double s[kR];
};

// One thread's tallies of the two rows around an edge, kept in registers over consecutive spans that
// are tested against the same edge (the common single-edge windows of the kernel's own loop).
struct LaneTally {
    uint32_t c_lo, c_hi;  // pairs in row m / row m + 1
    double w_lo, w_hi;    // and their weight
};

// The pair loop: n_j staged j-points (a multiple of 32, paired layout at shared address grp2, window weights at
// vgrp) against this thread's kR i-points and the K edges seeded by e32 and the offsets dl.  Returns the steps of
// kStep j-points in which some pair came within the guard band G of an edge, one bit each (warp-uniform).
//   t[q][r]  weighted: 2^-7 * sum of v_j over the pairs above edge q, per i-point
//   nb[q]    unweighted: pairs not above edge q
template <int K, bool kWeighted, bool kChord>
__device__ __forceinline__ uint32_t pair_loop(const uint32_t grp2, const uint32_t vgrp, const int n_j, const float (&nx)[kR],
                                              const float (&ny)[kR], const float (&nz)[kR], const float e32, const float (&dl)[K],
                                              const float G, double (&t)[K][kR], uint32_t (&nb)[K])
{
    const unsigned long long e2 = pack2(e32, e32);
    unsigned long long dl2[K];
#pragma unroll
    for (int q = 0; q < K; ++q) dl2[q] = pack2(dl[q], dl[q]);
    uint32_t sg[K][kR];  // unweighted: sign bits of d_q (1 = not above) of the last 32 j-points
#pragma unroll
    for (int q = 0; q < K; ++q) {
        nb[q] = 0u;
#pragma unroll
        for (int r = 0; r < kR; ++r) {
            t[q][r] = 0.0;
            sg[q][r] = 0u;
        }
    }
    constexpr int kInd = (K == 1 ? 4 : 2) * kR;  // indicator registers: low words zero for the whole loop
    unsigned long long ind[kInd];
#pragma unroll
    for (int i = 0; i < kInd; ++i) ind[i] = 0ull;

    uint32_t amb_steps = 0;  // warp-uniform
    constexpr int kStep = step_of(kWeighted);
    static_assert(kGroup / kStep <= 32, "one bit per step");
#pragma unroll 1
    for (int jj = 0; jj < n_j; jj += kStep) {
        float mn = 1.0f;  // min |d_q| over the pairs of the step
        // (the loops of several edges are not unrolled over the step's two pairs of j-points: they are the rare shapes,
        // and half their code is what the instruction cache has for the common one)
#pragma unroll(K == 1 ? kStep / 2 : 1)
        for (int u = 0; u < kStep; u += 2) {
            const ulonglong2 xy = lds_u64x2(grp2 + 16u * (uint32_t)(jj + u));
            const unsigned long long zz = lds_u64(grp2 + 16u * (uint32_t)(jj + u) + 16u);
            double v0 = 0.0, v1 = 0.0;
            if constexpr (kWeighted) {
                const double2 vv = lds_f64x2(vgrp + 8u * (uint32_t)(jj + u));
                v0 = vv.x;
                v1 = vv.y;
            }
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                unsigned long long d2;
                if constexpr (kChord) {
                    const unsigned long long dx = fadd2(xy.x, pack2(nx[r], nx[r])), dy = fadd2(xy.y, pack2(ny[r], ny[r])),
                                             dz = fadd2(zz, pack2(nz[r], nz[r]));
                    d2 = ffma2(dx, dx, ffma2(dy, dy, ffma2(dz, dz, e2)));
                } else {
                    // {n, n} packed at the use: the FFMA2 takes the one register for both halves
                    d2 = ffma2(pack2(nx[r], nx[r]), xy.x, ffma2(pack2(ny[r], ny[r]), xy.y, ffma2(pack2(nz[r], nz[r]), zz, e2)));
                }
#pragma unroll
                for (int q = 0; q < K; ++q) {
                    const unsigned long long dq2 = q == 0 ? d2 : fadd2(d2, dl2[q]);
                    const float a = lo32(dq2), b = hi32(dq2);
                    if constexpr (kWeighted) {
                        unsigned long long &g0 = ind[(u * kR + 2 * r) % kInd], &g1 = ind[(u * kR + 2 * r + 1) % kInd];
                        t[q][r] = fma(v0, ind_gt0_f64(g0, a), t[q][r]);
                        t[q][r] = fma(v1, ind_gt0_f64(g1, b), t[q][r]);
                    } else {
                        asm("shf.l.wrap.b32 %0, %1, %0, 1;" : "+r"(sg[q][r]) : "r"(__float_as_uint(a)));
                        asm("shf.l.wrap.b32 %0, %1, %0, 1;" : "+r"(sg[q][r]) : "r"(__float_as_uint(b)));
                    }
                    asm("min.f32 %0, %0, %1, %2;" : "+f"(mn) : "f"(fabsf(a)), "f"(fabsf(b)));
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
    return amb_steps;
}

// The pair loop of a window that holds no edge: its caps prove that every pair lies in one row, on the near side of the
// edge e_m that bounds the row.  Every pair's d = e_m - c (or s - s_m) is still computed and must come out below -G --
// certified on that side -- but nothing is tallied pair by pair: the row gets the span's pair count and weight at once.
// Returns false if some pair is not certified (the span is then redone by pair_loop and its exact corrections).
template <bool kChord>
__device__ __forceinline__ bool verify_loop(const uint32_t grp2, const int n_j, const float (&nx)[kR], const float (&ny)[kR],
                                            const float (&nz)[kR], const float e32, const float G)
{
    const unsigned long long e2 = pack2(e32, e32);
    float mx0 = -3.0e38f, mx1 = -3.0e38f;  // max d over the pairs, two chains
#pragma unroll 1
    for (int jj = 0; jj < n_j; jj += 4) {
#pragma unroll
        for (int u = 0; u < 4; u += 2) {
            const ulonglong2 xy = lds_u64x2(grp2 + 16u * (uint32_t)(jj + u));
            const unsigned long long zz = lds_u64(grp2 + 16u * (uint32_t)(jj + u) + 16u);
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                unsigned long long d2;
                if constexpr (kChord) {
                    const unsigned long long dx = fadd2(xy.x, pack2(nx[r], nx[r])), dy = fadd2(xy.y, pack2(ny[r], ny[r])),
                                             dz = fadd2(zz, pack2(nz[r], nz[r]));
                    d2 = ffma2(dx, dx, ffma2(dy, dy, ffma2(dz, dz, e2)));
                } else {
                    d2 = ffma2(pack2(nx[r], nx[r]), xy.x, ffma2(pack2(ny[r], ny[r]), xy.y, ffma2(pack2(nz[r], nz[r]), zz, e2)));
                }
                if (r & 1) asm("max.f32 %0, %0, %1, %2;" : "+f"(mx1) : "f"(lo32(d2)), "f"(hi32(d2)));
                else asm("max.f32 %0, %0, %1, %2;" : "+f"(mx0) : "f"(lo32(d2)), "f"(hi32(d2)));
            }
        }
    }
    return __all_sync(0xffffffffu, fmaxf(mx0, mx1) < -G);
}

// Edges m_a .. m_a + n_real - 1 (n_real <= K) against one span of staged j-points and this thread's kR i-points.
// A chunk fills rows m_a .. m_a + n_real - 1 (and m_a + n_real if it is the last of its window); the tallies above
// its last edge go to the next chunk through `carry`.  A chunk of fewer than K edges repeats its last edge: the
// repeated tallies are equal, the rows between them get nothing, and one compiled loop serves every window
// (the code of the rare shapes must not crowd the instruction cache of the common one).
template <int K, bool kWeighted, bool kChord>
__device__ __forceinline__ void window_chunk(const WinParams &p, const Tables tb, const Rows rows, const Span sp,
                                             const float (&nx)[kR], const float (&ny)[kR], const float (&nz)[kR],
                                             const float *wi_of, const int wi_stride, const int m_a, const int n_real, const bool first, const bool last,
                                             unsigned long long *stat, Carry *carry)
{
    // wi_of: the weights of this thread's i-points, wi_of[r * wi_stride]
    const int lane = threadIdx.x & 31;
    float e32, G;
    float dl[K];
    dl[0] = 0.f;
    if constexpr (kChord) {
        e32 = tb.sneg(m_a);
        G = K == 1 ? tb.gs1(m_a) : tb.gsk(m_a);
#pragma unroll
        for (int q = 1; q < K; ++q) {
            const int mq = m_a + (q < n_real ? q : n_real - 1);
            dl[q] = __fsub_rn(tb.sneg(mq), e32);
            G = fmaxf(G, tb.gsk(mq));
        }
    } else {
        const double e0 = tb.edge(m_a);
        e32 = edge32(e0);
        G = K == 1 ? kGuard1 : kGuardK;
#pragma unroll
        for (int q = 1; q < K; ++q) {
            const double eq = tb.edge(m_a + (q < n_real ? q : n_real - 1));
            dl[q] = eq <= -1.0 ? -8.0f : (float)(eq - e0);
        }
    }
    double t[K][kR];     // weighted: 2^-7 * sum of v_j over the pairs above edge q, per i-point
    uint32_t nb[K];      // unweighted: pairs not above edge q
    const uint32_t amb_steps = pair_loop<K, kWeighted, kChord>(sp.grp2 + 16u * (uint32_t)sp.jj0, sp.vgrp + 8u * (uint32_t)sp.jj0,
                                                               sp.jj1 - sp.jj0, nx, ny, nz, e32, dl, G, t, nb);

    if (amb_steps) {
        // exact corrections, applied to the (exact) accumulators before anything is read from them
        double dt[kChunk * kR];
        int dn[kChunk];
        fixup_chunk<kWeighted, kChord>(p, tb, sp, amb_steps, n_real, m_a, G, stat, dt, dn);
#pragma unroll
        for (int q = 0; q < K; ++q) {
            const int qq = q < n_real ? q : n_real - 1;  // a repeated edge gets the corrections of the edge it repeats
            if constexpr (kWeighted) {
#pragma unroll
                for (int r = 0; r < kR; ++r) t[q][r] += dt[qq * kR + r];
            } else {
                nb[q] += (uint32_t)dn[qq];
            }
        }
    }
    // ---- this thread's tallies -> row contributions -> the warp's rows
    const uint32_t n_all = (uint32_t)(sp.jj1 - sp.jj0) * kR;  // this thread's pairs
    auto unpack = [&](double tt, uint32_t &n) -> double {  // 2^-7 (n C + sum of w) -> sum of w, n += count
        double sw = tt * 128.0;
        if constexpr (kWeighted) {
            const double nn = floor(sw * rows.pack->inv_C);  // C is a power of two and the sum of w is below C: exact
            sw -= nn * rows.pack->C;
            n += (uint32_t)nn;
        }
        return sw;
    };
    uint32_t c_prev = 0;  // this thread's pairs above the previous edge (all its pairs before the first)
    double s_prev[kR];    // and, per i-point, the sum of their w_j
    if (first) {
        c_prev = n_all;
#pragma unroll
        for (int r = 0; r < kR; ++r) s_prev[r] = sp.wsum;
    } else {
        c_prev = carry->c;
#pragma unroll
        for (int r = 0; r < kR; ++r) s_prev[r] = carry->s[r];
    }
    __syncwarp();
    // The rows, one after the other in a rolled loop (this epilogue runs once per span of a rare shape: its code is kept
    // short for the instruction cache, its tallies go through a copy in local memory that the loop can index).
    double tl[K + 1][kR];
    uint32_t nbl[K + 1];
#pragma unroll
    for (int q = 0; q < K; ++q) {
        nbl[q] = nb[q];
#pragma unroll
        for (int r = 0; r < kR; ++r) tl[q][r] = t[q][r];
    }
    nbl[K] = n_all;  // nothing lies above the row after the last edge
#pragma unroll
    for (int r = 0; r < kR; ++r) tl[K][r] = 0.0;
    const int q_end = last ? K + 1 : K;
#pragma unroll 1
    for (int q = 0; q < q_end; ++q) {
        uint32_t c_q = 0;  // pairs above edge q
        double rw = 0.0;   // weight of this thread's pairs in row m_a + q
        if constexpr (kWeighted) {
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                const double sw = unpack(tl[q][r], c_q);
                rw = fma((double)wi_of[r * wi_stride], s_prev[r] - sw, rw);
                s_prev[r] = sw;
            }
        } else {
            c_q = n_all - nbl[q];
        }
        const uint32_t rc = c_prev - c_q;
        c_prev = c_q;
        if (rc == 0u) rw = 0.0;  // no pair of this thread in the row: not even a rounding residue
        const uint32_t rc_warp = __reduce_add_sync(0xffffffffu, rc);
        if constexpr (kWeighted) rw = warp_sum_f64(rw);
        if (lane == 0) rows.template add<kWeighted>(m_a + (q < n_real ? q : n_real), rc_warp, rw);
    }
    if (!last) {
        carry->c = c_prev;
#pragma unroll
        for (int r = 0; r < kR; ++r) carry->s[r] = s_prev[r];
    }
    __syncwarp();
}

// A window of two or more edges (rows r_lo .. r_hi): its edges kChunk at a time, every pass over the whole span.
// Not inlined: only the common case (one edge) lives in the kernel's own loop, so that the register
// allocation of that loop is not set by the rare variants.  It reloads the i-points.
template <bool kWeighted, bool kChord>
__device__ __noinline__ void window_multi(const WinParams &p, const Tables tb, const Rows rows, const Span sp, int r_lo, int r_hi,
                                          unsigned long long *stat)
{
    const int lane = threadIdx.x & 31;
    float nx[kR], ny[kR], nz[kR];
#pragma unroll
    for (int r = 0; r < kR; ++r) {
        const float4 v = sp.ipoint(r);
        nx[r] = v.x;
        ny[r] = v.y;
        nz[r] = v.z;
    }
    // the weight of i-point r: wi[r * 128] (float4 records, 32 apart)
    const float *wi = reinterpret_cast<const float *>(__cvta_shared_to_generic(sp.ipts)) + 4 * lane + 3;
    Carry carry;
    carry.c = 0u;
#pragma unroll
    for (int r = 0; r < kR; ++r) carry.s[r] = 0.0;
    int m = r_lo;  // edges below m are done
    while (m < r_hi) {
        const int left = r_hi - m;
        const int take = left < kChunk ? left : kChunk;
        window_chunk<kChunk, kWeighted, kChord>(p, tb, rows, sp, nx, ny, nz, wi, 128, m, take, m == r_lo, left <= kChunk, stat, &carry);
        m += take;
    }
}

// Pair by pair: ragged groups, the diagonal group of an auto-count and windows of many edges.  The fp32 squared
// chord length s of a pair picks a cell of the table (its float bits, shifted); the cell names the one edge that
// can matter inside it and the guard band around that edge (the error bound of chord_row).  A certified pair goes
// to its row at once; one within the guard band, or in a cell that holds several edges, gets its row from the
// search of chord_row and, where that leaves it open, from the fp64 definition.
template <bool kWeighted>
__device__ __noinline__ void general_span(const WinParams &p, const Tables tb, const Rows rows, const Span sp, const Mask mk,
                                          unsigned long long *stat)
{
    const int lane = threadIdx.x & 31;
    float4 pi[kR];
#pragma unroll
    for (int r = 0; r < kR; ++r) {
        pi[r] = sp.ipoint(r);  // negated in the stash
        pi[r].x = -pi[r].x;
        pi[r].y = -pi[r].y;
        pi[r].z = -pi[r].z;
    }
    const uint32_t cells = tb.cells();
    const CellKey ck(p.cell);
    uint32_t n_exact = 0;
    const int jj_end = sp.jj1 < mk.jn ? sp.jj1 : mk.jn;
    for (int jj = sp.jj0; jj < jj_end; ++jj) {
        const float4 pj = sp.point(jj);
#pragma unroll
        for (int r = 0; r < kR; ++r) {
            if (!mk.on(sp, r, jj)) continue;
            const float dx = __fsub_rn(pi[r].x, pj.x), dy = __fsub_rn(pi[r].y, pj.y), dz = __fsub_rn(pi[r].z, pj.z);
            const float s32 = fmaf(dx, dx, fmaf(dy, dy, __fmul_rn(dz, dz)));  // as chord_row computes it
            int row;
            if (!cell_row(cells, ck, s32, row)) {
                row = chord_row_ool(pi[r].x, pi[r].y, pi[r].z, pj.x, pj.y, pj.z, tb.sed_ptr(), tb.nbins, tb.margin());
                if (row < 0) {
                    row = exact_row(p.xyz_a, p.stride_a, p.perm_a[sp.i_first + r * 32 + lane], p.xyz_b, p.stride_b,
                                    p.perm_b[sp.j_first + jj], p.edges, p.nbins);
                    ++n_exact;
                }
            }
            rows.template add_atomic<kWeighted>(row, 1u, (double)pi[r].w * (double)pj.w);
        }
    }
    n_exact = __reduce_add_sync(0xffffffffu, n_exact);
    if (lane == 0 && n_exact) atomicAdd(&stat[kStatFp64], (unsigned long long)n_exact);
}

// The pairs of the j-points jj, jj + 1 that their cell did not certify (bit 2 r + h of `open`: i-point r, j-point jj + h):
// the search of chord_row, then the fp64 definition.  Called by the whole warp; rolled, out of line.
template <bool kWeighted>
__device__ __noinline__ void resolve_open(const WinParams &p, const Tables tb, const Rows rows, const Span sp, int jj, uint32_t open,
                                          unsigned long long *stat)
{
    const int lane = threadIdx.x & 31;
    uint32_t n_exact = 0;
#pragma unroll 1
    while (open) {
        const int b = __ffs((int)open) - 1;
        open &= open - 1u;
        const int r = b >> 1, h = b & 1;
        const float4 pi = sp.ipoint(r);  // negated in the stash
        const float4 pj = sp.point(jj + h);
        int rw = chord_row_ool(-pi.x, -pi.y, -pi.z, pj.x, pj.y, pj.z, tb.sed_ptr(), tb.nbins, tb.margin());
        if (rw < 0) {
            rw = exact_row(p.xyz_a, p.stride_a, p.perm_a[sp.i_first + r * 32 + lane], p.xyz_b, p.stride_b, p.perm_b[sp.j_first + jj + h],
                           p.edges, p.nbins);
            ++n_exact;
        }
        rows.template add_atomic<kWeighted>(rw, 1u, (double)pi.w * (double)pj.w);
    }
    n_exact = __reduce_add_sync(0xffffffffu, n_exact);
    if (lane == 0 && n_exact) atomicAdd(&stat[kStatFp64], (unsigned long long)n_exact);
}

// The same for a full span (nothing masked): two j-points at a time, their squared chord lengths by packed adds and
// FMAs (bit for bit the values chord_row computes), one 8-byte load per pair for its cell, one shared-memory
// reduction per pair for its row, and the search only for the pairs the cell does not certify.  Unweighted windows
// of more than kMaxPassEdges edges (the near field of a small-angle count) come here.
template <bool kWeighted>
__device__ __noinline__ void general_span_full(const WinParams &p, const Tables tb, const Rows rows, const Span sp,
                                               unsigned long long *stat)
{
    float nx[kR], ny[kR], nz[kR], wi[kR];
#pragma unroll
    for (int r = 0; r < kR; ++r) {
        const float4 v = sp.ipoint(r);  // negated in the stash
        nx[r] = v.x;
        ny[r] = v.y;
        nz[r] = v.z;
        wi[r] = v.w;
    }
    const uint32_t cells = tb.cells();
    const CellKey ck(p.cell);
    // (no branch around a pair's reduction: an uncertified pair adds to CtaHeader::trash, the last 16 bytes before the tables)
    const uint32_t cnt_a = smem_u32(rows.cnt), ws_a = kWeighted ? smem_u32(rows.ws) : 0u, trash = tb.base - 16u;
#pragma unroll 1
    for (int jj = sp.jj0; jj < sp.jj1; jj += 2) {
        const ulonglong2 xy = lds_u64x2(sp.grp2 + 16u * (uint32_t)jj);
        const ulonglong2 zw = lds_u64x2(sp.grp2 + 16u * (uint32_t)jj + 16u);  // {z0, z1}, {w0, w1}
        uint32_t open = 0u;
        // first all eight table loads, then the eight decisions and reductions: the loads and the reductions are
        // volatile and keep their order, and a load that waited behind the previous pair's reduction was what the loop
        // spent its time on
        unsigned long long s2[kR];
        float thr[kR][2];
        uint32_t word[kR][2];
#pragma unroll
        for (int r = 0; r < kR; ++r) {
            const unsigned long long dx = fadd2(xy.x, pack2(nx[r], nx[r])), dy = fadd2(xy.y, pack2(ny[r], ny[r])),
                                     dz = fadd2(zw.x, pack2(nz[r], nz[r]));
            unsigned long long zz2;
            asm("mul.rn.f32x2 %0, %1, %1;" : "=l"(zz2) : "l"(dz));
            s2[r] = ffma2(dx, dx, ffma2(dy, dy, zz2));
#pragma unroll
            for (int h = 0; h < 2; ++h) cell_load(cells, ck, h ? hi32(s2[r]) : lo32(s2[r]), thr[r][h], word[r][h]);
        }
#pragma unroll
        for (int r = 0; r < kR; ++r) {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                int row;
                const bool cert = cell_decide(h ? hi32(s2[r]) : lo32(s2[r]), thr[r][h], word[r][h], row);
                asm volatile("red.shared.add.u32 [%0], 1;" ::"r"(cert ? cnt_a + 4u * (uint32_t)row : trash) : "memory");
                if constexpr (kWeighted)
                    asm volatile("red.shared.add.f64 [%0], %1;" ::"r"(cert ? ws_a + 8u * (uint32_t)row : trash + 8u),
                                 "d"((double)wi[r] * (double)(h ? hi32(zw.y) : lo32(zw.y)))
                                 : "memory");
                open |= cert ? 0u : 1u << (2 * r + h);
            }
        }
        if (__any_sync(0xffffffffu, open != 0u)) resolve_open<kWeighted>(p, tb, rows, sp, jj, open, stat);
    }
}

// Fills the cell table of general_span from the edges as squared chord lengths (sed, ascending; -1 / +inf at the
// poles).  A cell [lo, hi) is taken with the guard bands at its two ends: every edge a value of the cell could fail to
// clear counts as inside it.  No edge inside: all of the cell is one row.  One: the edge and its guard band.  More:
// the cell is marked crowded (NaN threshold) and its pairs are searched.
__device__ __forceinline__ void fill_cells(uint32_t cells, const CellShape shape, const float *sed, int nbins, float margin, int tid,
                                           int n_threads)
{
    const int kShift = 23 - shape.bits;
    const uint32_t kKey0 = (uint32_t)(127 + shape.exp_lo) << shape.bits;
    auto guard_at = [&](float se) {  // chord_row's `cleared`, for an edge stored as se
        const float sm = se + margin;
        return 1.02f * (2.5e-7f * sqrtf(sm) + 4.0e-7f * sm + 1.0e-13f) + margin;
    };
    // a value s fails to clear edge k only if |s - se_k| <= guard_at(se_k); both ends of that band ascend with k
    auto band_hi = [&](int k) { return sed[k] < 0.f ? -1.0f : (sed[k] > 3.0e38f ? 3.4e38f : sed[k] + 1.05f * guard_at(sed[k])); };
    auto band_lo = [&](int k) { return sed[k] < 0.f ? -1.0f : (sed[k] > 3.0e38f ? 3.4e38f : sed[k] - 1.05f * guard_at(sed[k])); };
    for (int key = tid; key < shape.slots(); key += n_threads) {
        Cell c;
        if (key >= shape.count) {  // the slot of the values outside the table (and the padding after it)
            c.thr = __uint_as_float(0x7fc00000u);
            c.word = 0u;
            *reinterpret_cast<Cell *>(__cvta_shared_to_generic(cells + 8u * (uint32_t)key)) = c;
            continue;
        }
        const float lo = __uint_as_float(((uint32_t)key + kKey0) << kShift), hi = __uint_as_float(((uint32_t)key + kKey0 + 1u) << kShift);
        // below: the edges whose band ends before the cell (the pole edge e_0 = 1, stored as -1, always does: every pair is
        // at or beyond it); up: those whose band starts at or before its end (the pole edge e_n = -1, stored as +inf, never
        // does: no pair is beyond it).  Two binary searches over the nbins + 1 edges.
        int below = 0, up = 0;
        for (int a = 0, b = nbins + 1; a < b;) {
            const int m = (a + b) >> 1;
            if (band_hi(m) < lo) below = a = m + 1;
            else b = m;
        }
        for (int a = below, b = nbins + 1; a < b;) {
            const int m = (a + b) >> 1;
            if (band_lo(m) <= hi) a = m + 1;
            else b = m;
            up = a;
        }
        if (up < below) up = below;
        const int inside = up - below, first = below;
        c.word = (uint32_t)(below + 1);  // the row of s >= thr
        if (inside == 0) {
            c.thr = 3.0e38f;  // |s - thr| > 0 always, s >= thr never: all of the cell is row `below`
        } else if (inside == 1) {
            c.thr = sed[first];
            c.word |= (__float_as_uint(guard_at(sed[first])) + 0xffffu) & 0xffff0000u;  // rounded up to 8 mantissa bits
        } else {
            c.thr = __uint_as_float(0x7fc00000u);  // NaN: no pair of the cell is certified, the edges are searched
        }
        *reinterpret_cast<Cell *>(__cvta_shared_to_generic(cells + 8u * (uint32_t)key)) = c;
    }
}

// ---- the kernel ---------------------------------------------------------------------------------
// The warp-uniform state of a warp's stream.  It lives in shared memory (read a few times per j-group) so
// that it does not occupy registers of the pair loops.
struct WarpCtl {
    uint32_t q_tail, n_issued, n_done;  // units [n_done, q_tail) are queued, [n_done, n_issued) have their loads in flight;
                                        // unit number s lives in queue slot s % kQueue and stage s % kWStages
    uint32_t it, it_end;                // work items of the job still to be scanned
    int t, cx, cy, cz;                  // j-tiles of item `it` already scanned; that item {i-tile, first j-tile, j-tiles}
    int ig;                             // the job's i-group within its i-tiles
    int part;                           // the job takes the j-groups g of a tile with g % CtaHeader::split == part
    int no_more;                        // the global job counter has run out
    int sub;                            // the sub-group of the unit at the head of the queue that is being evaluated
    uint32_t since_flush;               // j-groups tallied in the warp's unflushed rows
    int tally_m;                        // the edge the threads' LaneTally belongs to, or -1
    uint32_t loaded_first;              // i_first of the i-points in WarpSm::ipts
    unsigned long long n_eval, n_win;   // pairs evaluated / of them by the single-edge loop
    unsigned long long n_chord;         // pairs classified on the fp32 chord length (chord-domain windows, pair-by-pair path)
};
static_assert(sizeof(WarpCtl) <= 96 && sizeof(WarpCtl) % 8 == 0, "per-warp header: 32 bytes of mbarriers, then WarpCtl");
constexpr int kWarpHeader = 128;

// Per-CTA header of the shared memory.
struct CtaHeader {
    unsigned long long stat[8];
    PackInfo pack;
    uint32_t n_items, chunk, n_jobs, split;
    uint32_t trash[4];  // where the pair-by-pair loop sends the reductions of the pairs it has not certified: a u32, then a double
};
static_assert(kNumStats <= 8 && sizeof(CtaHeader) % 16 == 0, "");

// A warp's shared memory, addressed from one 32-bit shared address:
// [mbarriers, WarpCtl | queue | lane tallies | the i-points {-x, -y, -z, w} | stages | rows].
template <bool kWeighted>
struct WarpSm {
    uint32_t base;
    int rows_n;
    static constexpr size_t kStage = wstage_bytes(kWeighted);
    __device__ __forceinline__ unsigned char *ptr(uint32_t off) const
    {
        return reinterpret_cast<unsigned char *>(__cvta_shared_to_generic(base + off));
    }
    __device__ __forceinline__ uint32_t full(int st) const { return base + 8u * (uint32_t)st; }
    __device__ __forceinline__ volatile WarpCtl *ctl() const { return reinterpret_cast<volatile WarpCtl *>(ptr(32)); }
    __device__ __forceinline__ Unit *queue() const { return reinterpret_cast<Unit *>(ptr(kWarpHeader)); }
    static constexpr uint32_t kFixed = kWarpHeader + (uint32_t)(sizeof(Unit) * kQueue) + 32u * (uint32_t)sizeof(LaneTally) + (uint32_t)(kGroup * sizeof(float4));
    __device__ __forceinline__ LaneTally *tally() const { return reinterpret_cast<LaneTally *>(ptr(kWarpHeader + (uint32_t)(sizeof(Unit) * kQueue))); }
    __device__ __forceinline__ float4 *ipts() const
    {
        return reinterpret_cast<float4 *>(ptr(kWarpHeader + (uint32_t)(sizeof(Unit) * kQueue) + 32u * (uint32_t)sizeof(LaneTally)));
    }
    __device__ __forceinline__ uint32_t stage(int st) const { return base + kFixed + (uint32_t)kStage * (uint32_t)st; }
    __device__ __forceinline__ uint32_t *cnt_own() const { return reinterpret_cast<uint32_t *>(ptr(kFixed + (uint32_t)(kStage * kWStages))); }
    __device__ __forceinline__ double *ws_own() const
    {
        return reinterpret_cast<double *>(reinterpret_cast<unsigned char *>(cnt_own()) + (((size_t)rows_n * sizeof(uint32_t) + 15) & ~size_t(15)));
    }
};

__device__ __forceinline__ void mbar_wait_s(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP_S:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE_S;\n"
        "bra WAIT_LOOP_S;\n"
        "WAIT_DONE_S:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}

extern __shared__ __align__(128) unsigned char smem[];

// The tables of the launch: right after the CtaHeader (pair_win_kernel); nothing of this needs a register.
__device__ __forceinline__ Tables tables_of(const WinParams &p)
{
    Tables tb;
    tb.base = smem_u32(smem) + (uint32_t)sizeof(CtaHeader);
    tb.nbins = p.nbins;
    tb.counters = p.counters;
    return tb;
}

// The rows a warp tallies into: its own, or the CTA's (many bins).
template <bool kWeighted>
__device__ __forceinline__ Rows rows_of(const WinParams &p, const WarpSm<kWeighted> w)
{
    CtaHeader *h = reinterpret_cast<CtaHeader *>(smem);
    Rows rows;
    rows.shared = p.shared_rows != 0;
    rows.pack = &h->pack;
    if (rows.shared) {
        // after the header, the edges and the chord tables (pair_win_kernel)
        size_t off = sizeof(CtaHeader) + sizeof(double) * (size_t)(p.nbins + 1) + sizeof(float) * 4 * (size_t)(p.nbins + 1);
        off = (off + 15) & ~size_t(15);
        off += sizeof(Cell) * (size_t)p.cell.slots();
        rows.cnt = reinterpret_cast<uint32_t *>(smem + off);
        off += sizeof(uint32_t) * (size_t)w.rows_n;
        off = (off + 15) & ~size_t(15);
        rows.ws = reinterpret_cast<double *>(smem + off);
    } else {
        rows.cnt = w.cnt_own();
        rows.ws = w.ws_own();
    }
    return rows;
}

// The kernel's own loop: the (sub-)window at the head of the warp's queue has at most one edge, WarpCtl::tally_m.
// Everything but the i-points is read from the warp's shared memory -- before the pair loop what the loop needs,
// after it what the tallies need (weight sum of the span, weights of the i-points, the lane's tallies of the two
// rows around the edge) -- so that the loop has the registers to itself and the i-points are live across no call.
template <bool kWeighted, bool kChord>
__device__ __forceinline__ void single_edge_span(const WinParams &p, const WarpSm<kWeighted> w)
{
    const int lane = threadIdx.x & 31;
    const Tables tb = tables_of(p);
    uint32_t grp2, vgrp;
    int n_j;
    float e32, G;
    bool no_edge;
    float nx[kR], ny[kR], nz[kR];  // the i-points, negated: loaded here so that they are live across no call
    {
        volatile WarpCtl *c = w.ctl();
        const uint32_t n_done = c->n_done;
        const Unit *u = &w.queue()[n_done % kQueue];
        const float4 *ip = w.ipts();  // (the kernel has seen to it that they are the unit's)
#pragma unroll
        for (int r = 0; r < kR; ++r) {
            const float4 v = ip[r * 32 + lane];
            nx[r] = v.x;
            ny[r] = v.y;
            nz[r] = v.z;
        }
        const int jj0 = u->nsub == 1 ? 0 : c->sub * kSub;
        n_j = u->nsub == 1 ? kGroup : kSub;
        grp2 = w.stage((int)(n_done % kWStages)) + 16u * (uint32_t)jj0;
        vgrp = w.stage((int)(n_done % kWStages)) + (uint32_t)kGroupBytes + 8u * (uint32_t)jj0;
        const int m_edge = c->tally_m;
        if constexpr (kChord) {
            e32 = tb.sneg(m_edge);
            G = tb.gs1(m_edge);
        } else {
            e32 = edge32(tb.edge(m_edge));
            G = kGuard1;
        }
        // a window with no edge inside, all of it in a row of the histogram: every pair is expected before the row's far edge
        const int s0 = u->nsub == 1 ? 0 : c->sub;
        no_edge = u->hi[s0] == u->lo[s0] && u->lo[s0] <= tb.nbins;
    }
    const float dl[1] = {0.f};
    double t[1][kR];
    uint32_t nb[1];
    uint32_t amb_steps = 0;
    bool verified = false;
    if constexpr (!kChord) verified = no_edge && verify_loop<false>(grp2, n_j, nx, ny, nz, e32, G);
    if (verified) {
        // every pair certified in row m_edge: nothing above the edge
        nb[0] = (uint32_t)n_j * kR;
#pragma unroll
        for (int r = 0; r < kR; ++r) t[0][r] = 0.0;
    } else {
        amb_steps = pair_loop<1, kWeighted, kChord>(grp2, vgrp, n_j, nx, ny, nz, e32, dl, G, t, nb);
    }

    volatile WarpCtl *c = w.ctl();
    const uint32_t n_done = c->n_done;
    const Unit *u = &w.queue()[n_done % kQueue];
    const int sub = u->nsub == 1 ? 0 : c->sub;
    CtaHeader *h = reinterpret_cast<CtaHeader *>(smem);
    if (amb_steps) {
        // exact corrections, applied to the (exact) accumulators before anything is read from them
        Span sp;
        sp.grp2 = w.stage((int)(n_done % kWStages));
        sp.vgrp = sp.grp2 + (uint32_t)kGroupBytes;
        sp.jj0 = u->nsub == 1 ? 0 : sub * kSub;
        sp.jj1 = sp.jj0 + n_j;
        sp.wsum = 0.0;
        sp.i_first = u->i_first;
        sp.j_first = u->j_first;
        sp.ipts = smem_u32(w.ipts());
        double dt[kChunk * kR];
        int dn[kChunk];
        fixup_chunk<kWeighted, kChord>(p, tb, sp, amb_steps, 1, c->tally_m, G, h->stat, dt, dn);
        if constexpr (kWeighted) {
#pragma unroll
            for (int r = 0; r < kR; ++r) t[0][r] += dt[r];
        } else {
            nb[0] += (uint32_t)dn[0];
        }
    }
    // ---- this thread's tallies of the two rows around the edge
    const uint32_t n_all = (uint32_t)n_j * kR;  // this thread's pairs
    uint32_t c_hi = kWeighted ? 0u : n_all - nb[0];
    double w_lo = 0.0, w_hi = 0.0;
    if constexpr (kWeighted) {
        const double wsum = u->wsum[sub], C = h->pack.C, inv_C = h->pack.inv_C;
        const float *wi = &w.ipts()[lane].w;
#pragma unroll
        for (int r = 0; r < kR; ++r) {
            // 2^-7 (n C + sum of w) -> n and the sum of w: C is a power of two and the sum of w is below C, so both are exact
            double sw = t[0][r] * 128.0;
            const double nn = floor(sw * inv_C);
            sw -= nn * C;
            c_hi += (uint32_t)nn;
            w_lo = fma((double)wi[r * 128], wsum - sw, w_lo);
            w_hi = fma((double)wi[r * 128], sw, w_hi);
        }
    }
    const uint32_t c_lo = n_all - c_hi;
    LaneTally *tally = w.tally() + lane;
    tally->c_lo += c_lo;
    tally->c_hi += c_hi;
    if constexpr (kWeighted) {
        if (c_lo != 0u) tally->w_lo += w_lo;  // no pair of this thread in the row: not even a rounding residue
        if (c_hi != 0u) tally->w_hi += w_hi;
    }
}

// The chord-domain form of the kernel's own loop, out of line: a call is either in the regime of one form or of the
// other (wide windows on the cosine, arc-minute windows on the chord), and the form it does not use should not
// sit in the instruction cache between the pieces of the one it does.
template <bool kWeighted>
__device__ __noinline__ void single_edge_span_chord(const WinParams &p, const WarpSm<kWeighted> w)
{
    single_edge_span<kWeighted, true>(p, w);
}

// The threads' tallies of the rows around edge WarpCtl::tally_m -> the warp's rows.  (Not inlined, like
// flush_rows: called when the edge changes, and the kernel's per-unit path should stay short.)
template <bool kWeighted>
__device__ __noinline__ void flush_tally(const WinParams &p, const WarpSm<kWeighted> w)
{
    const int lane = threadIdx.x & 31;
    volatile WarpCtl *c = w.ctl();
    const int tally_m = c->tally_m;
    if (tally_m < 0) return;
    const Rows rows = rows_of<kWeighted>(p, w);
    LaneTally *tl = w.tally() + lane;
    const LaneTally tally = *tl;
    *tl = LaneTally{0u, 0u, 0.0, 0.0};
    const uint32_t c_lo = __reduce_add_sync(0xffffffffu, tally.c_lo), c_hi = __reduce_add_sync(0xffffffffu, tally.c_hi);
    double w_lo = 0.0, w_hi = 0.0;
    if constexpr (kWeighted) {
        w_lo = warp_sum_f64(tally.w_lo);
        w_hi = warp_sum_f64(tally.w_hi);
    }
    if (lane == 0) {
        rows.template add<kWeighted>(tally_m, c_lo, w_lo);
        rows.template add<kWeighted>(tally_m + 1, c_hi, w_hi);
        c->tally_m = -1;
    }
    __syncwarp();
}

// This warp's rows -> global memory (u64 / f64 atomics); the rows restart from zero.
template <bool kWeighted>
__device__ __noinline__ void flush_rows(const WinParams &p, const WarpSm<kWeighted> w)
{
    const int lane = threadIdx.x & 31;
    flush_tally<kWeighted>(p, w);
    __syncwarp();
    const Rows rows = rows_of<kWeighted>(p, w);
    for (int row = lane; row < w.rows_n; row += 32) {
        // (shared rows: other warps add while this one takes the value and leaves zero)
        const uint32_t v = atomicExch(&rows.cnt[row], 0u);
        // read as signed: a correction (-1 now, its tally later) may be caught in between; the two's-complement
        // sum in global memory comes out the same
        if (row >= 1 && row <= p.nbins && v) atomicAdd(&p.counts[row - 1], (unsigned long long)(long long)(int32_t)v);
        if constexpr (kWeighted) {
            const double ws = __longlong_as_double((long long)atomicExch(reinterpret_cast<unsigned long long *>(&rows.ws[row]), 0ull));
            if (row >= 1 && row <= p.nbins && ws != 0.0) atomicAdd(&p.wsums[row - 1], ws);
        }
    }
    if (lane == 0) w.ctl()->since_flush = 0u;
    __syncwarp();
}

// The rows r_lo .. r_hi of the window of two caps, and whether it is classified on the chord length: r_lo | r_hi << 12 |
// chord << 24.  Out of line: refill calls it once per j-group and four times more per window of several edges, and its
// fp64 code should be resident once.
__device__ __noinline__ uint32_t bound_rows(const GroupCap ca, const GroupCap cj, const double slack, const double *edges_sm, const int nbins)
{
    int lo = 0, hi = nbins + 1;
    bool chord = false;
    double c_lo, c_hi;
    if (cap_window(ca, cj, slack, c_lo, c_hi)) {
        // rows of the two ends; the far end is a few rows on at most: walk there
        hi = lo = row_of_cos(c_hi, edges_sm, nbins);
        while (hi < nbins && c_lo <= edges_sm[hi]) ++hi;
        if (hi == nbins && c_lo < edges_sm[nbins]) ++hi;
        // (a window with no edge inside is tested against the far edge of its row: on the chord only if it comes close to it)
        chord = c_hi - c_lo < kChordWidth && c_lo > kChordCosMin && (hi > lo || (lo <= nbins && c_lo - edges_sm[lo] < 3.0e-6));
    }
    // The pair cosine is clamped to [-1, 1]: no pair lies before a pole edge e_0 = 1 or beyond e_n = -1, so
    // those two edges are in no window (and never tested in fp32: an unclamped c32 marginally outside, or
    // vectors a little longer than 1, would be misfiled).
    if (lo == 0 && edges_sm[0] >= 1.0) lo = 1;
    if (hi == nbins + 1 && edges_sm[nbins] <= -1.0) hi = nbins;
    if (hi < lo) hi = lo;
    return (uint32_t)lo | ((uint32_t)hi << 12) | (chord ? 1u << 24 : 0u);
}

// Keeps the warp's queue filled: takes the next job from the global counter when the current one has been scanned,
// and bounds the windows of the warp's i-group against the next (up to) kScan j-groups of its job -- two j-tiles,
// one lane per j-group, fp64 -- queueing the survivors: groups whose window lies wholly out of range are dropped
// (PAPER.md:126), a window of several edges is split by the sub-group caps of the j side.  Returns when kScan
// units are queued or no job is left.  Not inlined: its registers are its own.
template <bool kWeighted>
__device__ __noinline__ void refill(const WinParams &p, const WarpSm<kWeighted> w, const Tables tb)
{
    const int lane = threadIdx.x & 31;
    volatile WarpCtl *c = w.ctl();
    Unit *queue = w.queue();
    CtaHeader *h = reinterpret_cast<CtaHeader *>(smem);
    const Rows rows = rows_of<kWeighted>(p, w);
    const double slack = cap_slack(norm_eps(p.counters));
    const double *edges_sm = tb.edges_ptr();
    while (c->q_tail - c->n_done < (uint32_t)kScan) {
        if (c->it >= c->it_end) {
            // ---- the next job: {i-group of the tile, run of `chunk` work items}; 8 consecutive jobs share their items
            uint32_t job = 0;
            if (lane == 0) job = atomicAdd(reinterpret_cast<unsigned int *>(&p.counters[kCtrWorkHead]), 1u);  // (the low word: far fewer than 2^32 jobs)
            job = __shfl_sync(0xffffffffu, job, 0);
            if (job >= h->n_jobs) {
                if (lane == 0) c->no_more = 1;
                __syncwarp();
                return;
            }
            if (lane == 0) {
                const uint32_t it = job / (kGroupsPerTile * h->split) * h->chunk;
                const int3 cur = p.items[it];
                c->ig = (int)(job % kGroupsPerTile);
                c->part = (int)(job / kGroupsPerTile % h->split);
                c->it = it;
                c->it_end = it + h->chunk < h->n_items ? it + h->chunk : h->n_items;
                c->t = 0;
                c->cx = cur.x;
                c->cy = cur.y;
                c->cz = cur.z;
            }
            __syncwarp();
        }
        const int ig = c->ig;
        uint32_t it = c->it;
        const uint32_t it_end = c->it_end;
        int t = c->t, cx = c->cx, cy = c->cy, cz = c->cz;
        int ti0 = -1, tj0 = 0, ti1 = -1, tj1 = 0;
        if (it < it_end) {
            ti0 = cx;
            tj0 = cy + t;
            if (++t == cz) {
                t = 0;
                if (++it < it_end) {
                    const int3 nxt = p.items[it];
                    cx = nxt.x, cy = nxt.y, cz = nxt.z;
                }
            }
        }
        if (it < it_end) {
            ti1 = cx;
            tj1 = cy + t;
            if (++t == cz) {
                t = 0;
                if (++it < it_end) {
                    const int3 nxt = p.items[it];
                    cx = nxt.x, cy = nxt.y, cz = nxt.z;
                }
            }
        }
        const int ti = lane < kGroupsPerTile ? ti0 : ti1, tj = lane < kGroupsPerTile ? tj0 : tj1;
        const int g = lane & (kGroupsPerTile - 1);
        bool live = lane < kScan && ti >= 0 && (g & (int)(h->split - 1u)) == c->part;
        // first the window of the whole j-group (registers), then the queue slot, then -- straight into the slot -- the
        // windows of the sub-groups where the group's holds several edges (a rolled loop: this code should be short)
        uint32_t i0 = 0, j0 = 0, gj = 0, jgx = 0;
        int lo = 0, hi = 0;
        bool chord = false, masked = false, diag = false;
        double wsum_i = 0.0, wsum_j = 0.0;
        GroupCap ca;
        if (live) {
            const uint32_t igx = (uint32_t)ti * kGroupsPerTile + ig;
            jgx = (uint32_t)tj * kGroupsPerTile + g;
            i0 = igx * kGroup;
            j0 = jgx * kGroup;
            const uint32_t gi = i0 < p.n_a ? (p.n_a - i0 < (uint32_t)kGroup ? p.n_a - i0 : (uint32_t)kGroup) : 0u;
            gj = j0 < p.n_b ? (p.n_b - j0 < (uint32_t)kGroup ? p.n_b - j0 : (uint32_t)kGroup) : 0u;
            const bool diag_tile = p.is_auto && tj == ti;
            live = gi > 0 && gj > 0 && !(diag_tile && g < ig);
            if (live) {
                diag = diag_tile && g == ig;
                masked = gi < (uint32_t)kGroup || gj < (uint32_t)kGroup || diag;
                ca = p.gcaps_a[igx];
                const GroupCap cb = p.gcaps_b[jgx];
                wsum_i = ca.wsum;
                wsum_j = cb.wsum;
                const uint32_t r = bound_rows(ca, cb, slack, edges_sm, p.nbins);
                lo = (int)(r & 0xfffu);
                hi = (int)((r >> 12) & 0xfffu);
                chord = (r >> 24) != 0u;
                const bool out = hi == lo && (lo == 0 || lo > p.nbins);  // all closer than theta_min or all beyond theta_max
                if (p.prune && out) {
                    live = false;  // pruned at the level of groups, like whole tiles in the work list
                } else if (p.bulk && hi == lo && !out && !masked) {
                    // all pairs of two full groups in one bin: the bin gets the groups' pair count and the product of
                    // their weight sums, and nothing is evaluated (ACF_OPT_BULK)
                    const unsigned long long all = (unsigned long long)kGroup * kGroup;
                    rows.template add_atomic<kWeighted>(lo, (uint32_t)all, wsum_i * wsum_j);
                    atomicAdd(&h->stat[kStatBulk], all);
                    live = false;
                }
            }
        }
        const uint32_t alive = __ballot_sync(0xffffffffu, live);
        const uint32_t q_tail = c->q_tail;
        if (live) {
            Unit *q = &queue[(q_tail + __popc(alive & ((1u << lane) - 1u))) % kQueue];
            q->i_first = i0;
            q->j_first = j0;
            q->jn = (int32_t)gj;
            q->nsub = 1;
            q->masked = masked;
            q->diag = diag;
            q->chord = chord ? 1 : 0;
            q->lo[0] = (int16_t)lo;
            q->hi[0] = (int16_t)hi;
            q->wsum[0] = wsum_j;
            if (p.refine && !masked && hi - lo >= 2) {
                // several edges: the window of each sub-group of the j side is narrower
                uint32_t chords = 0;
                bool same = true;
#pragma unroll
                for (int s = 0; s < kSubsPerGroup; ++s) {
                    const GroupCap cs = p.scaps_b[(size_t)jgx * kSubsPerGroup + s];
                    const uint32_t r = bound_rows(ca, cs, slack, edges_sm, p.nbins);
                    int slo = (int)(r & 0xfffu), shi = (int)((r >> 12) & 0xfffu);
                    if (p.prune && shi == slo && (slo == 0 || slo > p.nbins)) slo = shi = -1;
                    q->lo[s] = (int16_t)slo;
                    q->hi[s] = (int16_t)shi;
                    q->wsum[s] = cs.wsum;
                    chords |= (r >> 24) << s;
                    same = same && slo >= 0 && slo == q->lo[0] && shi == q->hi[0];
                }
                same = same && (chords == 0u || chords == 15u);
                // the same window four times over: one span after all (one prologue, one epilogue)
                q->nsub = same ? 1 : kSubsPerGroup;
                q->chord = (uint8_t)(same ? (chords & 1u) : chords);
                if (same) q->wsum[0] = wsum_j;
            }
        }
        __syncwarp();
        if (lane == 0) {
            c->q_tail = q_tail + __popc(alive);
            c->it = it;
            c->t = t;
            c->cx = cx;
            c->cy = cy;
            c->cz = cz;
        }
        __syncwarp();
    }
}

template <bool kWeighted>
__global__ void __launch_bounds__(kThreads, 1) pair_win_kernel(const __grid_constant__ WinParams p)
{
    if (p.counters[kCtrBadInput] != 0) return;  // inputs failed validation
    if (kWeighted && p.pack_b->packed == 0) return;  // weights that do not pack: the table kernel does the call
    const int rows_n = p.nbins + 2;
    const int n_edges = p.nbins + 1;
    constexpr size_t kStage = wstage_bytes(kWeighted);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    // ---- shared memory: per CTA [CtaHeader | edges | chord tables | shared rows], then per warp (WarpSm)
    CtaHeader *h = reinterpret_cast<CtaHeader *>(smem);
    size_t off = sizeof(CtaHeader);
    double *edges_sm = reinterpret_cast<double *>(smem + off);
    off += sizeof(double) * (size_t)n_edges;
    float *sed_sm = reinterpret_cast<float *>(smem + off);
    float *sneg_sm = sed_sm + n_edges, *gs1_sm = sneg_sm + n_edges, *gsk_sm = gs1_sm + n_edges;
    off += sizeof(float) * 4 * (size_t)n_edges;
    off = (off + 15) & ~size_t(15);
    off += sizeof(Cell) * (size_t)p.cell.slots();  // the cell table (Tables::cells)
    if (p.shared_rows) {
        uint32_t *cnt_shared = reinterpret_cast<uint32_t *>(smem + off);
        off += sizeof(uint32_t) * (size_t)rows_n;
        off = (off + 15) & ~size_t(15);
        double *ws_shared = reinterpret_cast<double *>(smem + off);
        if constexpr (kWeighted) off += sizeof(double) * (size_t)rows_n;
        for (int i = tid; i < rows_n; i += blockDim.x) {
            cnt_shared[i] = 0;
            if constexpr (kWeighted) ws_shared[i] = 0.0;
        }
    }
    off = (off + 127) & ~size_t(127);
    size_t per_warp = WarpSm<kWeighted>::kFixed + kStage * kWStages;
    if (!p.shared_rows) per_warp += (((size_t)rows_n * sizeof(uint32_t) + 15) & ~size_t(15)) + (kWeighted ? (size_t)rows_n * sizeof(double) : 0);
    per_warp = (per_warp + 127) & ~size_t(127);
    WarpSm<kWeighted> w;
    w.base = smem_u32(smem + off + per_warp * (size_t)warp);
    w.rows_n = rows_n;

    const Tables tb = tables_of(p);
    {
        const float margin = tb.margin();
        for (int i = tid; i < n_edges; i += blockDim.x) {
            edges_sm[i] = p.edges[i];
            const float se = p.sedges[i];
            sed_sm[i] = se;
            sneg_sm[i] = -se;
            gs1_sm[i] = chord_guard(se, margin, false);
            gsk_sm[i] = chord_guard(se, margin, true);
        }
        fill_cells(tb.cells(), p.cell, p.sedges, p.nbins, margin, tid, blockDim.x);
    }
    if (!p.shared_rows)
        for (int i = lane; i < rows_n; i += 32) {
            w.cnt_own()[i] = 0;
            if constexpr (kWeighted) w.ws_own()[i] = 0.0;
        }
    if (lane == 0) {
        volatile WarpCtl *c = w.ctl();
        for (int s = 0; s < kWStages; ++s) mbar_init(reinterpret_cast<uint64_t *>(w.ptr(8u * (uint32_t)s)), 1);
        c->q_tail = c->n_issued = c->n_done = 0u;
        c->it = c->it_end = 0u;
        c->t = c->cx = c->cy = c->cz = c->ig = c->part = 0;
        c->no_more = 0;
        c->since_flush = 0u;
        c->tally_m = -1;
        c->loaded_first = 0xffffffffu;
        c->n_eval = c->n_win = c->n_chord = 0ull;
    }
    if (tid == 0) {
        for (int i = 0; i < 8; ++i) h->stat[i] = 0ull;
        h->pack = *p.pack_b;
        const uint32_t n_items = (uint32_t)(p.counters[kCtrWorkCount] > p.capacity ? p.capacity : p.counters[kCtrWorkCount]);
        uint32_t chunk = (uint32_t)((unsigned long long)n_items * kGroupsPerTile / (64ull * gridDim.x * kWarps));
        chunk = chunk < 1u ? 1u : (chunk > 4u ? 4u : chunk);
        // few items (small catalogues): a job takes only every split-th j-group of its items' tiles
        uint32_t split = 1u;
        while (split < (uint32_t)kGroupsPerTile && (unsigned long long)n_items * kGroupsPerTile * split < 2ull * gridDim.x * kWarps) split *= 2u;
        h->n_items = n_items;
        h->chunk = chunk;
        h->split = split;
        h->n_jobs = (n_items + chunk - 1u) / chunk * kGroupsPerTile * split;
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();

    w.tally()[lane] = LaneTally{0u, 0u, 0.0, 0.0};  // this thread's tallies of the rows around the edge WarpCtl::tally_m

    while (true) {
        volatile WarpCtl *c = w.ctl();
        if (!c->no_more && c->q_tail - c->n_done < (uint32_t)kScan) refill<kWeighted>(p, w, tables_of(p));
        // ---- issue: TMA loads of queued units into free stages
        const uint32_t n_done = c->n_done;
        {
            const uint32_t q_tail = c->q_tail;
            if (lane == 0) {
                uint32_t n_issued = c->n_issued;
                while (n_issued < q_tail && n_issued - n_done < (uint32_t)kWStages) {
                    const uint32_t j0 = w.queue()[n_issued % kQueue].j_first;
                    const int st = (int)(n_issued % kWStages);
                    const uint32_t dst = w.stage(st), bar = w.full(st);
                    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"((uint32_t)kStage) : "memory");
                    // the arrays are padded to whole tiles: always a full group
                    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                                 "l"(p.pts2_b + (size_t)j0 * 4), "r"((uint32_t)kGroupBytes), "r"(bar)
                                 : "memory");
                    if constexpr (kWeighted)
                        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                                         dst + (uint32_t)kGroupBytes),
                                     "l"(p.vj_b + (size_t)j0), "r"((uint32_t)kGroupVjBytes), "r"(bar)
                                     : "memory");
                    ++n_issued;
                }
                c->n_issued = n_issued;
            }
            __syncwarp();
            if (n_done == q_tail) {
                if (c->no_more) break;
                continue;
            }
        }
        // ---- evaluate the oldest unit
        const Unit *u = &w.queue()[n_done % kQueue];
        const int st = (int)(n_done % kWStages);
        mbar_wait_s(w.full(st), (n_done / kWStages) & 1u);
        Span sp;
        sp.grp2 = w.stage(st);
        sp.vgrp = sp.grp2 + (uint32_t)kGroupBytes;
        sp.i_first = u->i_first;
        sp.j_first = u->j_first;
        sp.ipts = smem_u32(w.ipts());
        if (c->loaded_first != sp.i_first) {
            // another i-group: its points, negated, into the warp's shared memory (the array is padded to a whole tile)
            float4 *ip = w.ipts();
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                const float4 v = p.pts_a[sp.i_first + r * 32 + lane];
                ip[r * 32 + lane] = make_float4(-v.x, -v.y, -v.z, v.w);
            }
            if (lane == 0) c->loaded_first = sp.i_first;
            __syncwarp();
        }
        // u32 rows, read as signed when flushed: flush before 2^30 pairs (shared rows take the pairs of all the CTA's warps)
        if (c->since_flush >= (1u << 30) / (uint32_t)(kGroup * kGroup) / (p.shared_rows ? (uint32_t)kWarps : 1u)) flush_rows<kWeighted>(p, w);
        const int nsub = u->nsub;
        const bool masked = u->masked != 0;
        uint32_t pairs = 0, pairs_win = 0, pairs_chord = 0;
        for (int s = 0; s < nsub; ++s) {
            const int r_lo = u->lo[s], r_hi = u->hi[s];
            if (r_lo < 0) continue;  // a sub-group whose window lies out of range
            sp.jj0 = nsub == 1 ? 0 : s * kSub;
            sp.jj1 = nsub == 1 ? kGroup : sp.jj0 + kSub;
            sp.wsum = u->wsum[s];
            const bool chord = (u->chord >> s) & 1;
            const int K = r_hi - r_lo;
            if (masked || (!kWeighted && K > kMaxPassEdges)) {
                Mask mk;
                mk.gi = p.n_a - sp.i_first < (uint32_t)kGroup ? p.n_a - sp.i_first : (uint32_t)kGroup;
                mk.jn = u->jn;
                mk.diag = u->diag != 0;
                if (masked) general_span<kWeighted>(p, tables_of(p), rows_of<kWeighted>(p, w), sp, mk, h->stat);
                else general_span_full<kWeighted>(p, tables_of(p), rows_of<kWeighted>(p, w), sp, h->stat);
                const uint32_t n = !masked ? (uint32_t)(sp.jj1 - sp.jj0) * kGroup : (mk.diag ? mk.gi * (mk.gi - 1) / 2 : mk.gi * (uint32_t)mk.jn);
                pairs += n;
                pairs_chord += n;
            } else if (K <= 1) {
                // a window inside one row is tested against the edge that bounds the row
                const int m_edge = K == 1 ? r_lo : (r_lo > p.nbins ? p.nbins : r_lo);
                if (m_edge != c->tally_m) {
                    flush_tally<kWeighted>(p, w);
                    if (lane == 0) c->tally_m = m_edge;
                }
                if (lane == 0) c->sub = s;
                __syncwarp();
                if (chord) single_edge_span_chord<kWeighted>(p, w);
                else single_edge_span<kWeighted, false>(p, w);
                pairs += (uint32_t)(sp.jj1 - sp.jj0) * kGroup;
                pairs_win += (uint32_t)(sp.jj1 - sp.jj0) * kGroup;
                if (chord) pairs_chord += (uint32_t)(sp.jj1 - sp.jj0) * kGroup;
            } else {
                if (chord) window_multi<kWeighted, true>(p, tables_of(p), rows_of<kWeighted>(p, w), sp, r_lo, r_hi, h->stat);
                else window_multi<kWeighted, false>(p, tables_of(p), rows_of<kWeighted>(p, w), sp, r_lo, r_hi, h->stat);
                pairs += (uint32_t)(sp.jj1 - sp.jj0) * kGroup;
                if (chord) pairs_chord += (uint32_t)(sp.jj1 - sp.jj0) * kGroup;
            }
            __syncwarp();
        }
        __syncwarp();  // every lane has read the stage (and the queue slot) before either is reused
        if (lane == 0) {
            c->n_eval += pairs;
            c->n_win += pairs_win;
            c->n_chord += pairs_chord;
            c->since_flush += 1u;
            c->n_done = n_done + 1u;
        }
        __syncwarp();
    }

    flush_rows<kWeighted>(p, w);
    if (lane == 0) {
        volatile WarpCtl *c = w.ctl();
        if (c->n_eval) atomicAdd(&h->stat[kStatEvaluated], c->n_eval);
        if (c->n_win) atomicAdd(&h->stat[kStatWindow], c->n_win);
        if (c->n_chord) atomicAdd(&h->stat[kStatChord], c->n_chord);
    }
    __syncthreads();
    if (tid == 0) {
        if (h->stat[kStatFp64]) atomicAdd(&p.counters[kCtrPairsFp64], h->stat[kStatFp64]);
        if (h->stat[kStatWindow]) atomicAdd(&p.counters[kCtrPairsWindow], h->stat[kStatWindow]);
        if (h->stat[kStatEvaluated]) atomicAdd(&p.counters[kCtrPairsEvaluated], h->stat[kStatEvaluated]);
        if (h->stat[kStatChord]) atomicAdd(&p.counters[kCtrPairsChord], h->stat[kStatChord]);
        if (h->stat[kStatBulk]) atomicAdd(&p.counters[kCtrPairsBulk], h->stat[kStatBulk]);
    }
}

}  // namespace

// Launches the window kernel on the work items of the context's work list.
// The shape of the cell table for a call's edges (see CellShape): the table starts two octaves below the octave of the
// first edge that is not a pole (closer pairs, a factor 2 to 2.8 below theta_min, are searched); a cell is 0.69 / 2^bits
// of its s wide, and the narrowest bin should be at least two cells wide.
static CellShape cell_shape(const double *h_edges, int nbins, bool weighted)
{
    double s_first = 4.0, rel_min = 1.0;
    double prev = -1.0;
    for (int k = 0; k <= nbins; ++k) {
        const double sk = 2.0 * (1.0 - h_edges[k]);  // ascending
        if (sk > 0.0 && sk < s_first) s_first = sk;
        if (prev > 0.0 && sk > prev) rel_min = std::min(rel_min, (sk - prev) / sk);
        prev = sk;
    }
    CellShape c;
    int e = 0;
    std::frexp(s_first, &e);  // s_first = f 2^e, f in [0.5, 1): the octave of s_first starts at 2^(e - 1)
    c.exp_lo = std::max(kCellExpMin, std::min(1, e - 3));
    c.bits = weighted ? 4 : 6;
    if (!weighted)
        while (c.bits < 10 && 0.69 / (double)(1 << c.bits) > 0.5 * rel_min && sizeof(Cell) * ((size_t)(2 - c.exp_lo) << (c.bits + 1)) <= kCellBudget) ++c.bits;
    c.count = (2 - c.exp_lo) << c.bits;
    return c;
}

int launch_pair_win(acf_ctx *ctx, const Prepared &a, const Prepared &b, int is_auto, const double *h_edges, int nbins, uint32_t capacity,
                    unsigned long long *d_counts, double *d_wsums)
{
    const bool weighted = d_wsums != nullptr;
    CellShape cell = cell_shape(h_edges, nbins, weighted);
    const int rows_n = nbins + 2, n_edges = nbins + 1;
    auto smem_for = [&](bool shared_rows) {
        size_t m = sizeof(CtaHeader) + sizeof(double) * (size_t)n_edges + sizeof(float) * 4 * (size_t)n_edges;
        m = (m + 15) & ~size_t(15);
        m += sizeof(Cell) * (size_t)cell.slots();
        if (shared_rows) {
            m += sizeof(uint32_t) * (size_t)rows_n;
            m = (m + 15) & ~size_t(15);
            if (weighted) m += sizeof(double) * (size_t)rows_n;
        }
        m = (m + 127) & ~size_t(127);
        size_t per_warp = kWarpHeader + sizeof(Unit) * kQueue + 32 * sizeof(LaneTally) + kGroup * sizeof(float4) + wstage_bytes(weighted) * kWStages;
        if (!shared_rows) per_warp += (((size_t)rows_n * sizeof(uint32_t) + 15) & ~size_t(15)) + (weighted ? (size_t)rows_n * sizeof(double) : 0);
        per_warp = (per_warp + 127) & ~size_t(127);
        return m + per_warp * kWarps + 128;  // (+128: the dynamic segment need not start on a 128-byte boundary)
    };
    const size_t budget = (size_t)ctx->max_smem_optin;
    // what gives way when the shared memory is short: first the cell table's resolution, then the rows per warp (one
    // set per CTA instead, every update atomic), then the resolution again
    auto shrink_cells = [&](bool shared_rows) {
        while (smem_for(shared_rows) > budget && cell.bits > (weighted ? 4 : 6)) {
            --cell.bits;
            cell.count = (2 - cell.exp_lo) << cell.bits;
        }
    };
    shrink_cells(false);
    const bool shared_rows = smem_for(false) > budget;
    if (shared_rows) {
        cell = cell_shape(h_edges, nbins, weighted);
        shrink_cells(true);
    }
    if (smem_for(shared_rows) > budget) return fail(ctx, ACF_EINVAL, "too many bins for the window kernel (%d)", nbins);
    const size_t smem = smem_for(shared_rows);

    WinParams p{};
    p.pts_a = a.pts;
    p.pts2_b = b.pts2;
    p.vj_b = b.vj;
    p.pack_b = b.pack;
    p.perm_a = a.perm;
    p.perm_b = b.perm;
    p.gcaps_a = a.gcaps;
    p.gcaps_b = b.gcaps;
    p.scaps_b = b.scaps;
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
    p.shared_rows = shared_rows ? 1 : 0;
    p.prune = ctx->opt_prune;
    p.bulk = ctx->opt_bulk;
    p.refine = 1;
    p.cell = cell;

    const int grid = ctx->num_sms;  // one CTA of 16 warps per SM: 128 registers a thread
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
