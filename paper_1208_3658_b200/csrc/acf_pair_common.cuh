// acf_pair_common.cuh -- device helpers shared by the two pair kernels (acf_pair.cu: single-edge
// windows + cell-table path; acf_pair_win.cu: windows of any number of edges).
#pragma once

#include <cuda_runtime.h>

#include <cstdint>

#include "acf_device.cuh"
#include "acf_internal.h"

namespace acf {

constexpr int kMaxStages = 8;      // j-tile buffers of the producer/consumer ring (at least 2)
constexpr int kSmemHeader = 512;   // mbarriers + stage descriptors
// one staged j-tile: the paired fp32 records, then (weighted) the fp64 window-path weights
constexpr size_t kTileBytes = (size_t)kTile * sizeof(float4);
constexpr size_t kVjBytes = (size_t)kTile * sizeof(double);
__host__ __device__ constexpr size_t stage_bytes(bool weighted) { return kTileBytes + (weighted ? kVjBytes : 0); }

struct StageMeta {
    int ti, tj, jn, pad;
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// non-blocking: has the phase with this parity completed?
__device__ __forceinline__ bool mbar_test(uint64_t *bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
// TMA 1-D bulk copy global -> shared, completion signalled on an mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void bulk_load(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

__device__ __forceinline__ unsigned long long pack2(float lo, float hi)
{
    return ((unsigned long long)__float_as_uint(hi) << 32) | __float_as_uint(lo);
}
// two fp32 FMAs in one instruction (SASS FFMA2): each half is the IEEE fma of its operands
__device__ __forceinline__ unsigned long long ffma2(unsigned long long a, unsigned long long b, unsigned long long c)
{
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
// point jj of a staged tile in the paired layout
__device__ __forceinline__ float4 tile_point(const float *__restrict__ tile2, int jj)
{
    const float *pp = tile2 + (size_t)(jj >> 1) * 8 + (jj & 1);
    return make_float4(pp[0], pp[2], pp[4], pp[6]);
}

// Exact histogram row of a pair: the definition of include/acf.h on the caller's doubles.
static __device__ __noinline__ int exact_row(const double *__restrict__ xyz_a, size_t stride_a, size_t gi,
                                      const double *__restrict__ xyz_b, size_t stride_b, size_t gj,
                                      const double *__restrict__ edges, int nbins)
{
    const double c = pair_cos_fp64(xyz_a[gi], xyz_a[stride_a + gi], xyz_a[2 * stride_a + gi], xyz_b[gj],
                                   xyz_b[stride_b + gj], xyz_b[2 * stride_b + gj]);
    const int k = bin_of_fp64(c, edges, nbins);
    if (k >= 0) return k + 1;
    return c > edges[0] ? 0 : nbins + 1;
}

// Histogram row of a cosine (the definition of include/acf.h): 0 if c > e[0]; nbins + 1 if c < e[nbins];
// else 1 + its bin.  Equals #{m <= nbins - 1 : c <= e[m]} + [c < e[nbins]], non-increasing in c.
__device__ __forceinline__ int row_of_cos(double c, const double *__restrict__ e, int nbins)
{
    int lo = 0, hi = nbins;  // c <= e[m] for m < lo; c > e[m] for m >= hi
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (c <= e[mid]) lo = mid + 1; else hi = mid;
    }
    return lo + ((lo == nbins && c < e[nbins]) ? 1 : 0);
}


// ---- chord tier ---------------------------------------------------------------------------------------
// Below a few arc minutes 1 - cos(theta) is smaller than the fp32 error of the cosine (3e-7), so the
// cosine test leaves every such pair open.  The squared chord length s = |u_i - u_j|^2 does not cancel:
// c = (|u_i|^2 + |u_j|^2 - s) / 2, and in fp32 from the fp32 coordinates
//   |s32 - s| <= 2.4e-7 sqrt(s) + 3.1e-7 s + 6e-14
// (coordinates rounded to 2^-24 relative: an error vector of at most 1.19e-7 + 2^-24 sqrt(s); three
// roundings of the sum of squares).  With eps = max |u|^2 - 1 over the validated points and the 4e-16
// of the fp64 chain, c64 <= e_k holds iff s >= s_k + eta, s_k = 2 (1 - e_k), |eta| <= 2 eps + 8e-16.
// sed[m] = fp32(s_m) ascending (a pole edge e_0 = 1 is stored as -1: always passed; e_n = -1 as +inf:
// never passed).  Returns the histogram row (0 .. nbins + 1) if s32 clears both neighbouring edges by
// the bound (with the rounding of sed and of this arithmetic folded in), else -1: the fp64 definition
// decides.  (xi, yi, zi) and (xj, yj, zj) are the fp32 coordinates the kernels hold.
__device__ __forceinline__ int chord_row(float xi, float yi, float zi, float xj, float yj, float zj,
                                         const float *__restrict__ sed, int nbins, float margin)
{
    const float dx = __fsub_rn(xi, xj), dy = __fsub_rn(yi, yj), dz = __fsub_rn(zi, zj);
    const float s = fmaf(dx, dx, fmaf(dy, dy, __fmul_rn(dz, dz)));
    int lo = 0, hi = nbins + 1;  // s >= sed[m] for m < lo; s < sed[m] for m >= hi
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (s >= sed[mid]) lo = mid + 1; else hi = mid;
    }
    auto cleared = [&](float se, float gap) {
        const float sm = se + margin;  // G is taken at the far end of the uncertainty of the edge
        return gap > 1.02f * (2.5e-7f * sqrtf(sm) + 4.0e-7f * sm + 1.0e-13f) + margin;
    };
    if (lo >= 1) {
        const float se = sed[lo - 1];
        if (se >= 0.f && !cleared(se, s - se)) return -1;
    }
    if (lo <= nbins) {
        const float se = sed[lo];
        if (se < 3.0e38f && !cleared(se, se - s)) return -1;
    }
    return lo;
}
// margin of chord_row from the validation's largest | |u|^2 - 1 |
__device__ __forceinline__ float chord_margin(const unsigned long long *counters)
{
    const double eps = __longlong_as_double((long long)counters[kCtrNormDev]);
    // 8e-16 for the fp64 chain, 7e-16 for the rounding of the two |u|^2 the validation computed, and slack
    return (float)(2.02 * eps + 3.0e-15) * 1.0001f;
}

// Largest | |u|^2 - 1 | over the validated points of the call (validate_kernel), as a double.
__device__ __forceinline__ double norm_eps(const unsigned long long *counters)
{
    return __longlong_as_double((long long)counters[kCtrNormDev]);
}
// What the cap bounds are widened by.  The caps bound the DIRECTIONS of the points (gather_caps_kernel divides
// by the norms); the pair cosine of include/acf.h is the dot product of the vectors as given, i.e. the cosine of
// the angle times |u_i| |u_j|, and | |u_i| |u_j| - 1 | <= eps (1 + eps) for | |u|^2 - 1 | <= eps.  1e-9 covers the
// rounding of the few fp64 operations of the bound itself (~1e-15).
__device__ __forceinline__ double cap_slack(double eps) { return 1.001 * eps + 1e-9; }

// fp32 stand-in of an edge in the cosine tests d = e - c.  The pair cosine is clamped to [-1, 1], so nothing lies
// beyond a pole edge: it is never tested in fp32 (an unclamped c32 marginally outside, or vectors a little longer
// than 1, would be misfiled); +-4 decides every pair the clamped way and keeps |d| far above any guard band.
__device__ __forceinline__ float edge32(double e) { return e >= 1.0 ? 4.0f : (e <= -1.0 ? -4.0f : (float)e); }

// All pairs between points of caps a and b have c_lo <= c <= c_hi for the pair cosine c of include/acf.h
// (theta = angle between the centres, rho = sum of the radii: cos(theta -+ rho) = cos(theta) cos(rho) +-
// sin(theta) sin(rho), clamped at the poles, widened by `slack` = cap_slack(eps)).  Returns false when the caps
// give no bound.
__device__ __forceinline__ bool cap_window(const GroupCap &a, const GroupCap &b, double slack, double &c_lo, double &c_hi)
{
    c_lo = -1.0;
    c_hi = 1.0;
    if (a.cos_r > 1.5 || b.cos_r > 1.5) return false;  // an empty group
    if (a.cos_r + b.cos_r <= 0.0) return false;         // radii sum to pi or more: no bound
    const double d = fmin(1.0, fmax(-1.0, a.cx * b.cx + a.cy * b.cy + a.cz * b.cz));
    const double C = a.cos_r * b.cos_r - a.sin_r * b.sin_r;  // cos(rho)
    const double S = a.sin_r * b.cos_r + a.cos_r * b.sin_r;  // sin(rho) >= 0
    const double sd = sqrt(fmax(0.0, 1.0 - d * d));
    c_hi = d >= C ? 1.0 : d * C + sd * S;
    c_lo = d <= -C ? -1.0 : d * C - sd * S;
    c_hi = fmin(1.0, c_hi + slack);
    c_lo = fmax(-1.0, c_lo - slack);
    return true;
}

}  // namespace acf
