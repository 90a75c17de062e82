// acf_device.cuh -- device helpers shared by the kernels of libacf.
#pragma once

#include <cuda_runtime.h>

#include <cstdint>

namespace acf {

// The pair cosine of include/acf.h: c = fma(xi, xj, fma(yi, yj, zi*zj)), IEEE round-to-nearest,
// clamped to [-1, 1] (the C term of Appendix A is the dot product of the two unit
// vectors).  Intrinsics pin the operation order whatever -fmad says.
__device__ __forceinline__ double pair_cos_fp64(double xi, double yi, double zi, double xj, double yj, double zj)
{
    double c = __fma_rn(xi, xj, __fma_rn(yi, yj, __dmul_rn(zi, zj)));
    c = c > 1.0 ? 1.0 : c;
    c = c < -1.0 ? -1.0 : c;
    return c;
}

// Bin of c under descending cosine edges e[0..nbins]: -1 if c > e[0] or c < e[nbins] (PAPER.md:103,
// 126: out-of-range pairs are not histogrammed); else k = #{ m in [1, nbins-1] : c <= e[m] }, i.e.
// e[k+1] < c <= e[k] with the last bin closed at e[nbins].  {m : c <= e[m]} is a prefix because e is
// descending, so a binary search for its length gives the same k as the count.
__device__ __forceinline__ int bin_of_fp64(double c, const double *e, int nbins)
{
    if (c > e[0] || c < e[nbins]) return -1;
    int lo = 0, hi = nbins - 1;  // invariant: c <= e[m] for all m in [1, lo]; c > e[m] for m in (hi, nbins-1]
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (c <= e[mid]) lo = mid; else hi = mid - 1;
    }
    return lo;
}

__device__ __forceinline__ unsigned long long warp_sum_u64(unsigned long long v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

}  // namespace acf
