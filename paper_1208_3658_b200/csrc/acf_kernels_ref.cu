// acf_kernels_ref.cu -- the fp64 reference kernel: every pair evaluated exactly as include/acf.h
// defines it (PAPER.md:215 C term as a dot product; PAPER.md:70 pair sets; PAPER.md:103, 126
// range).  It is the arbiter the fast path defers to for pairs near a bin edge, and it is
// selectable on its own with ACF_OPT_KERNEL = ACF_KERNEL_FP64.  Also: input validation.
#include "acf_device.cuh"
#include "acf_internal.h"

namespace acf {

namespace {

constexpr int kRefThreads = 128;   // rows per CTA (one per thread)
constexpr int kRefTileJ = 256;     // columns staged in shared memory at a time

// grid.x: row blocks; grid.y: column chunks (keeps small row ranges parallel)
__global__ void __launch_bounds__(kRefThreads)
pair_count_fp64_kernel(const double *__restrict__ a, const float *__restrict__ wa, size_t n_a, size_t i_begin,
                       size_t i_end, const double *__restrict__ b, const float *__restrict__ wb, size_t n_b,
                       const double *__restrict__ edges, int nbins, int is_auto,
                       unsigned long long *__restrict__ counts, double *__restrict__ wsums,
                       unsigned long long *__restrict__ counters)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *s_edges = reinterpret_cast<double *>(smem_raw);                  // nbins + 1
    double *s_x = s_edges + (nbins + 1);                                     // kRefTileJ each
    double *s_y = s_x + kRefTileJ;
    double *s_z = s_y + kRefTileJ;
    double *s_w = s_z + kRefTileJ;
    double *s_wsum = s_w + kRefTileJ;                                        // nbins
    unsigned int *s_cnt = reinterpret_cast<unsigned int *>(s_wsum + nbins);  // nbins

    const bool weighted = wsums != nullptr;
    for (int k = threadIdx.x; k <= nbins; k += blockDim.x) s_edges[k] = edges[k];
    for (int k = threadIdx.x; k < nbins; k += blockDim.x) {
        s_cnt[k] = 0;
        s_wsum[k] = 0.0;
    }

    const size_t i = i_begin + (size_t)blockIdx.x * kRefThreads + threadIdx.x;
    const bool row_ok = i < i_end;
    double xi = 0, yi = 0, zi = 0, wi = 0;
    if (row_ok) {
        xi = a[i];
        yi = a[n_a + i];
        zi = a[2 * n_a + i];
        if (weighted) wi = (double)wa[i];
    }
    // this CTA's column chunk
    const size_t chunk = (n_b + gridDim.y - 1) / gridDim.y;
    size_t j_lo = (size_t)blockIdx.y * chunk;
    size_t j_hi = j_lo + chunk < n_b ? j_lo + chunk : n_b;
    if (is_auto) {
        // nothing below the first row of this block can pair with it
        size_t first_row = i_begin + (size_t)blockIdx.x * kRefThreads;
        if (j_lo < first_row + 1) j_lo = first_row + 1 < j_hi ? first_row + 1 : j_hi;
    }
    unsigned long long evaluated = 0;
    __syncthreads();

    for (size_t j0 = j_lo; j0 < j_hi; j0 += kRefTileJ) {
        const int jn = (int)((j_hi - j0) < (size_t)kRefTileJ ? (j_hi - j0) : (size_t)kRefTileJ);
        for (int t = threadIdx.x; t < jn; t += blockDim.x) {
            s_x[t] = b[j0 + t];
            s_y[t] = b[n_b + j0 + t];
            s_z[t] = b[2 * n_b + j0 + t];
            s_w[t] = weighted ? (double)wb[j0 + t] : 0.0;
        }
        __syncthreads();
        if (row_ok) {
            for (int t = 0; t < jn; ++t) {
                const size_t j = j0 + t;
                if (is_auto && j <= i) continue;
                const double c = pair_cos_fp64(xi, yi, zi, s_x[t], s_y[t], s_z[t]);
                const int k = bin_of_fp64(c, s_edges, nbins);
                ++evaluated;
                if (k >= 0) {
                    atomicAdd(&s_cnt[k], 1u);
                    if (weighted) atomicAdd(&s_wsum[k], wi * s_w[t]);
                }
            }
        }
        __syncthreads();
    }
    for (int k = threadIdx.x; k < nbins; k += blockDim.x) {
        if (s_cnt[k]) atomicAdd(&counts[k], (unsigned long long)s_cnt[k]);
        if (weighted && s_wsum[k] != 0.0) atomicAdd(&wsums[k], s_wsum[k]);
    }
    if (counters) {
        evaluated = warp_sum_u64(evaluated);
        if ((threadIdx.x & 31) == 0 && evaluated) {
            atomicAdd(&counters[kCtrPairsEvaluated], evaluated);
            atomicAdd(&counters[kCtrPairsFp64], evaluated);
        }
    }
}

__global__ void validate_kernel(const double *__restrict__ xyz, size_t stride, size_t off, size_t cnt, const float *__restrict__ w,
                                PackInfo *__restrict__ pack)
{
    unsigned int bad = 0;
    double dev = 0.0;  // largest |r^2 - 1| seen: the chord tier and the cap bounds of the pair kernels need it (acf_pair_common.cuh)
    for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < cnt; k += (size_t)gridDim.x * blockDim.x) {
        const size_t i = off + k;
        const double x = xyz[i], y = xyz[stride + i], z = xyz[2 * stride + i];
        const double r2 = x * x + y * y + z * z;
        bool ok = isfinite(x) && isfinite(y) && isfinite(z) && fabs(r2 - 1.0) <= 1e-6;
        if (ok) dev = fmax(dev, fabs(r2 - 1.0));
        if (w) {
            const float wi = w[i];
            ok = ok && isfinite(wi) && wi >= 0.0f;
        }
        bad += ok ? 0u : 1u;
    }
    bad = __reduce_add_sync(0xffffffffu, bad);
    if ((threadIdx.x & 31) == 0 && bad) atomicAdd(&pack->bad, (int)(bad > 0x3fffffffu ? 0x3fffffffu : bad));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dev = fmax(dev, __shfl_xor_sync(0xffffffffu, dev, o));
    // non-negative doubles order like their bit patterns
    if ((threadIdx.x & 31) == 0 && dev > 0.0)
        atomicMax(reinterpret_cast<unsigned long long *>(&pack->eps), (unsigned long long)__double_as_longlong(dev));
}

}  // namespace

cudaError_t launch_validate(acf_ctx *ctx, const double *d_xyz, size_t stride, size_t off, size_t cnt, const float *d_w, PackInfo *pack)
{
    if (cnt == 0) return cudaSuccess;
    int blocks = (int)((cnt + 255) / 256);
    if (blocks > ctx->num_sms * 8) blocks = ctx->num_sms * 8;
    validate_kernel<<<blocks, 256, 0, ctx->stream>>>(d_xyz, stride, off, cnt, d_w, pack);
    ctx->last.kernel_launches++;
    return cudaGetLastError();
}

cudaError_t launch_pair_count_fp64(acf_ctx *ctx, const double *d_a, const float *d_wa, size_t n_a,
                                   size_t i_begin, size_t i_end, const double *d_b, const float *d_wb,
                                   size_t n_b, const double *d_edges, int nbins, int is_auto,
                                   unsigned long long *d_counts, double *d_wsums)
{
    if (i_end <= i_begin || n_b == 0) return cudaSuccess;
    const size_t rows = i_end - i_begin;
    const unsigned row_blocks = (unsigned)((rows + kRefThreads - 1) / kRefThreads);
    // enough CTAs to fill the chip ~4x over, column chunks of at least one tile
    unsigned col_chunks = 1;
    const unsigned want = (unsigned)ctx->num_sms * 8;
    if (row_blocks < want) {
        col_chunks = (want + row_blocks - 1) / row_blocks;
        const unsigned max_chunks = (unsigned)((n_b + kRefTileJ - 1) / kRefTileJ);
        if (col_chunks > max_chunks) col_chunks = max_chunks;
        if (col_chunks > 65535u) col_chunks = 65535u;
        if (col_chunks < 1) col_chunks = 1;
    }
    const size_t smem = sizeof(double) * (size_t)(nbins + 1 + 4 * kRefTileJ + nbins) + sizeof(unsigned int) * (size_t)nbins;
    dim3 grid(row_blocks, col_chunks);
    pair_count_fp64_kernel<<<grid, kRefThreads, smem, ctx->stream>>>(
        d_a, d_wa, n_a, i_begin, i_end, d_b, d_wb, n_b, d_edges, nbins, is_auto, d_counts, d_wsums,
        ctx->opt_stats ? ctx->d_counters : nullptr);
    ctx->last.kernel_launches++;
    return cudaGetLastError();
}

}  // namespace acf
