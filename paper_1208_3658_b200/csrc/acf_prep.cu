// acf_prep.cu -- O(N) preparation of a catalogue for the pair kernel:
//   1. spatial key of every point (cube face of the unit vector + Hilbert index on the face),
//   2. LSD radix sort of (key, index) -- own kernels, 4 passes of 8 bits,
//   3. gather into sorted fp32 float4 {x, y, z, w} + bounding caps in fp64, per tile of kTile points
//      and per group of kGroup points,
//   4. the work list: (i-tile, run of j-tiles) items that may hold an in-range pair
//      (calculations that fall outside the bin range need not be made;
//       the pair matrix is walked sub-matrix by sub-matrix).
// Pair counts do not depend on the order of the points, so sorting changes nothing in the
// result; it makes tiles compact on the sky, which is what lets whole tile pairs be skipped.
#include "acf_device.cuh"
#include "acf_internal.h"

namespace acf {

namespace {

// ------------------------------------------------------------------ keys
// Hilbert index of (x, y) on a 2^14 x 2^14 grid (the classic xy -> d walk, one quadrant per level).
__device__ __forceinline__ uint32_t hilbert14(uint32_t x, uint32_t y)
{
    constexpr uint32_t n = 1u << 14;
    uint32_t d = 0;
#pragma unroll
    for (uint32_t s = n >> 1; s > 0; s >>= 1) {
        const uint32_t rx = (x & s) ? 1u : 0u, ry = (y & s) ? 1u : 0u;
        d += s * s * ((3u * rx) ^ ry);
        if (ry == 0) {
            if (rx == 1) {
                x = n - 1 - x;
                y = n - 1 - y;
            }
            const uint32_t t = x;
            x = y;
            y = t;
        }
    }
    return d;
}

// Key = cube face (3 bits) | Hilbert index of the equal-angle face coordinates (28 bits).  Points
// that are consecutive in key order are neighbours on the sky, so a run of sorted points has a small
// bounding cap (about 1.5x the ideal radius), which is what tile pruning and the per-window
// threshold selection of the pair kernel live on.  Any key gives correct counts.
__global__ void key_kernel(const double *__restrict__ xyz, size_t stride, size_t off, uint32_t n,
                           uint32_t *__restrict__ keys, uint32_t *__restrict__ idx)
{
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const size_t g = off + i;
        const float v[3] = {(float)xyz[g], (float)xyz[stride + g], (float)xyz[2 * stride + g]};
        int f = 0;
        if (fabsf(v[1]) > fabsf(v[f])) f = 1;
        if (fabsf(v[2]) > fabsf(v[f])) f = 2;
        const float major = v[f], inv = 1.0f / fmaxf(fabsf(major), 1e-30f);
        const float a1 = v[(f + 1) % 3] * inv, a2 = v[(f + 2) % 3] * inv;  // in [-1, 1]
        const float u = atanf(a1) * 1.2732395447351628f, w = atanf(a2) * 1.2732395447351628f;  // * 4/pi
        const uint32_t qx = (uint32_t)fminf(fmaxf((u + 1.0f) * 8192.0f, 0.0f), 16383.0f);
        const uint32_t qy = (uint32_t)fminf(fmaxf((w + 1.0f) * 8192.0f, 0.0f), 16383.0f);
        const uint32_t face = 2u * (uint32_t)f + (major < 0.0f ? 1u : 0u);
        keys[i] = (face << 28) | hilbert14(qx, qy);
        idx[i] = i;
    }
}

// ------------------------------------------------------------------ radix sort (stable, LSD)
constexpr int kSortThreads = 256;
constexpr int kSortWarps = kSortThreads / 32;
// Elements per lane: 16 (4096 per CTA), or 64 for catalogues of more than 2 M points, so that the one-CTA scan of the
// 256 x nblocks digit counts stays short (8 M points: 125 k counters instead of 500 k, 0.46 ms per pass before).
__host__ __device__ constexpr int sort_per_lane(uint32_t n) { return n > (2u << 20) ? 64 : 16; }
__host__ __device__ constexpr uint32_t sort_block_chunk(int per_lane) { return (uint32_t)(kSortWarps * 32 * per_lane); }

// counts[d * nblocks + b] = number of keys of CTA b whose digit is d
__global__ void __launch_bounds__(kSortThreads)
radix_count_kernel(const uint32_t *__restrict__ keys, uint32_t n, int shift, uint32_t *__restrict__ counts, uint32_t nblocks, int per_lane)
{
    __shared__ uint32_t hist[256];
    hist[threadIdx.x] = 0;
    __syncthreads();
    const uint32_t chunk = sort_block_chunk(per_lane), base = blockIdx.x * chunk;
    for (uint32_t t = threadIdx.x; t < chunk; t += kSortThreads) {
        const uint32_t i = base + t;
        if (i < n) atomicAdd(&hist[(keys[i] >> shift) & 255u], 1u);
    }
    __syncthreads();
    counts[threadIdx.x * nblocks + blockIdx.x] = hist[threadIdx.x];
}

// in-place exclusive scan of `len` counters by one CTA of 1024 threads
__global__ void __launch_bounds__(1024) scan_kernel(uint32_t *__restrict__ data, uint32_t len)
{
    __shared__ uint32_t partial[1024];
    const uint32_t per = (len + 1023u) / 1024u;
    const uint32_t lo = threadIdx.x * per, hi = lo + per < len ? lo + per : len;
    uint32_t sum = 0;
    for (uint32_t i = lo; i < hi; ++i) sum += data[i];
    partial[threadIdx.x] = sum;
    __syncthreads();
    // Hillis-Steele over the 1024 partial sums
    for (int o = 1; o < 1024; o <<= 1) {
        uint32_t v = threadIdx.x >= o ? partial[threadIdx.x - o] : 0u;
        __syncthreads();
        partial[threadIdx.x] += v;
        __syncthreads();
    }
    uint32_t run = threadIdx.x ? partial[threadIdx.x - 1] : 0u;
    for (uint32_t i = lo; i < hi; ++i) {
        const uint32_t v = data[i];
        data[i] = run;
        run += v;
    }
}

// Stable scatter.  Each warp owns a contiguous run of the CTA's chunk and walks it 32 keys at a
// time; __match_any_sync ranks equal digits inside a round by lane order.
__global__ void __launch_bounds__(kSortThreads)
radix_scatter_kernel(const uint32_t *__restrict__ keys_in, const uint32_t *__restrict__ idx_in,
                     uint32_t *__restrict__ keys_out, uint32_t *__restrict__ idx_out, uint32_t n, int shift,
                     const uint32_t *__restrict__ offsets, uint32_t nblocks, int per_lane)
{
    __shared__ uint32_t whist[kSortWarps][256];  // per-warp digit counts, then running output positions
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int t = threadIdx.x; t < kSortWarps * 256; t += kSortThreads) (&whist[0][0])[t] = 0;
    __syncthreads();
    const uint32_t wbase = blockIdx.x * sort_block_chunk(per_lane) + (uint32_t)(warp * 32 * per_lane);
    for (int r = 0; r < per_lane; ++r) {
        const uint32_t i = wbase + r * 32 + lane;
        if (i < n) atomicAdd(&whist[warp][(keys_in[i] >> shift) & 255u], 1u);
    }
    __syncthreads();
    {   // digit d = threadIdx.x: global offset of this CTA's digit-d run, then split over warps in order
        uint32_t run = offsets[threadIdx.x * nblocks + blockIdx.x];
        for (int w = 0; w < kSortWarps; ++w) {
            const uint32_t c = whist[w][threadIdx.x];
            whist[w][threadIdx.x] = run;
            run += c;
        }
    }
    __syncthreads();
    const uint32_t lt_mask = (1u << lane) - 1u;
    for (int r = 0; r < per_lane; ++r) {
        const uint32_t i = wbase + r * 32 + lane;
        const bool ok = i < n;
        const uint32_t key = ok ? keys_in[i] : 0u;
        const uint32_t digit = ok ? ((key >> shift) & 255u) : (256u + lane);  // invalid lanes match nobody
        const uint32_t peers = __match_any_sync(0xffffffffu, digit);
        uint32_t pos = 0;
        if (ok) pos = whist[warp][digit] + __popc(peers & lt_mask);
        __syncwarp();
        if (ok && (peers & lt_mask) == 0) whist[warp][digit] += __popc(peers);  // first peer advances the cursor
        __syncwarp();
        if (ok) {
            keys_out[pos] = key;
            idx_out[pos] = idx_in[i];
        }
    }
}

// ------------------------------------------------------------------ weight range
// range[0] = max of the weights' float bits, range[1] = max of ~bits over the non-zero weights (so that
// both start from a zeroed buffer).  Weights are non-negative and finite (validate_kernel), so the
// bit patterns order like the values.
__global__ void __launch_bounds__(256) wrange_kernel(const float *__restrict__ w, size_t off, uint32_t n, uint32_t *__restrict__ range)
{
    uint32_t mx = 0u, inv_mn = 0u;
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const uint32_t bits = __float_as_uint(w[off + i]) & 0x7fffffffu;
        if (bits) {
            mx = max(mx, bits);
            inv_mn = max(inv_mn, ~bits);
        }
    }
    mx = __reduce_max_sync(0xffffffffu, mx);
    inv_mn = __reduce_max_sync(0xffffffffu, inv_mn);
    if ((threadIdx.x & 31) == 0 && mx) {
        atomicMax(&range[0], mx);
        atomicMax(&range[1], inv_mn);
    }
}

// ------------------------------------------------------------------ gather + caps
// One CTA per tile of kTile sorted points, one warp per group of kGroup points: writes the fp32 float4
// records, the tile's bounding cap {unit centre, cos(radius)} and the kGroupsPerTile group caps, all
// computed in fp64 from the fp64 vectors.
__global__ void __launch_bounds__(256)
gather_caps_kernel(const double *__restrict__ xyz, size_t stride, size_t off, const float *__restrict__ w,
                   const uint32_t *__restrict__ idx, uint32_t n, float4 *__restrict__ pts,
                   uint32_t *__restrict__ perm, double4 *__restrict__ caps, GroupCap *__restrict__ gcaps,
                   GroupCap *__restrict__ scaps, float *__restrict__ pts2, double *__restrict__ vj, const uint32_t *__restrict__ range,
                   PackInfo *__restrict__ pack)
{
    static_assert(kGroupsPerTile == 8 && kGroup == 128, "one warp of 256 threads per group");
    __shared__ double red[3][8];
    __shared__ double centre[3];
    constexpr int kPer = kGroup / 32;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t base = blockIdx.x * kTile + warp * kGroup;
    double px[kPer], py[kPer], pz[kPer];  // the points' directions (the vectors divided by their norms)
    float wr[kPer];
    double sx = 0, sy = 0, sz = 0, sw = 0;
    static_assert(kPer == kSubsPerGroup && kSub == 32, "register slot r of a warp is sub-group r of its group");
    // window-path weights (PackInfo): C = 2^(exponent(w_max) + 9) > 256 w_max, a power of two
    const uint32_t mx_bits = w ? range[0] : 0x3f800000u, mn_bits = w ? ~range[1] : 0x3f800000u;
    const int ex_max = (int)(mx_bits >> 23), ex_min = (int)(mn_bits >> 23);
    const bool packed = mx_bits != 0u && ex_min >= 1 && ex_max - ex_min <= 13;
    const double packC = __hiloint2double((ex_max - 127 + 9 + 1023) << 20, 0);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        pack->C = packC;  // (bad and eps are the validation's)
        pack->inv_C = __hiloint2double((127 - 9 - ex_max + 1023) << 20, 0);
        pack->packed = packed ? 1 : 0;
    }
#pragma unroll
    for (int r = 0; r < kPer; ++r) {
        const uint32_t s = base + r * 32 + lane;
        float *p2 = pts2 + (size_t)(s >> 1) * 8 + (s & 1u);
        if (s < n) {
            const uint32_t local = idx[s];
            const size_t g = off + local;
            px[r] = xyz[g];
            py[r] = xyz[stride + g];
            pz[r] = xyz[2 * stride + g];
            const float wi = w ? w[g] : 1.0f;
            wr[r] = wi;
            pts[s] = make_float4((float)px[r], (float)py[r], (float)pz[r], wi);
            p2[0] = (float)px[r];
            p2[2] = (float)py[r];
            p2[4] = (float)pz[r];
            p2[6] = wi;
            vj[s] = packed ? packC + (double)wi : (double)wi;
            perm[s] = (uint32_t)g;  // index into the caller's catalogue
            // the caps bound directions: norms may be off 1 by the 1e-6 the validation accepts (cap_slack)
            const double inv = 1.0 / sqrt(fmax(1e-300, px[r] * px[r] + py[r] * py[r] + pz[r] * pz[r]));
            px[r] *= inv;
            py[r] *= inv;
            pz[r] *= inv;
            sx += px[r];
            sy += py[r];
            sz += pz[r];
            sw += (double)wi;
        } else {
            px[r] = py[r] = pz[r] = 0.0;
            wr[r] = 0.f;
            pts[s] = make_float4(0.f, 0.f, 0.f, 0.f);  // padding up to the tile boundary, never paired
            p2[0] = p2[2] = p2[4] = p2[6] = 0.f;
            vj[s] = 0.0;
        }
    }
    // ---- sub-group caps: register slot r of the warp holds sub-group r (kSub consecutive sorted points)
#pragma unroll
    for (int r = 0; r < kPer; ++r) {
        const bool have = base + r * 32 + lane < n;
        double ux = have ? px[r] : 0.0, uy = have ? py[r] : 0.0, uz = have ? pz[r] : 0.0;
        double uw = have ? (double)wr[r] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            ux += __shfl_xor_sync(0xffffffffu, ux, o);
            uy += __shfl_xor_sync(0xffffffffu, uy, o);
            uz += __shfl_xor_sync(0xffffffffu, uz, o);
            uw += __shfl_xor_sync(0xffffffffu, uw, o);
        }
        double cx = 0.0, cy = 0.0, cz = 1.0;
        const double nrm = sqrt(ux * ux + uy * uy + uz * uz);
        if (nrm > 1e-9) {
            cx = ux / nrm;
            cy = uy / nrm;
            cz = uz / nrm;
        }
        double mind = have ? cx * px[r] + cy * py[r] + cz * pz[r] : 2.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) mind = fmin(mind, __shfl_xor_sync(0xffffffffu, mind, o));
        if (lane == 0) {
            GroupCap sc;
            sc.cx = cx;
            sc.cy = cy;
            sc.cz = cz;
            if (base + r * 32 < n) {
                sc.cos_r = fmax(-1.0, fmin(1.0, mind) - 1e-9);
                sc.sin_r = sqrt(fmax(0.0, 1.0 - sc.cos_r * sc.cos_r));
            } else {
                sc.cos_r = 2.0;  // no points
                sc.sin_r = 0.0;
            }
            sc.wsum = uw;
            scaps[((size_t)blockIdx.x * kGroupsPerTile + warp) * kSubsPerGroup + r] = sc;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        sx += __shfl_xor_sync(0xffffffffu, sx, o);
        sy += __shfl_xor_sync(0xffffffffu, sy, o);
        sz += __shfl_xor_sync(0xffffffffu, sz, o);
        sw += __shfl_xor_sync(0xffffffffu, sw, o);
    }
    // ---- group cap (this warp's points)
    {
        double cx = 0.0, cy = 0.0, cz = 1.0;  // any centre is valid; the radius makes it a bound
        const double nrm = sqrt(sx * sx + sy * sy + sz * sz);
        if (nrm > 1e-9) {
            cx = sx / nrm;
            cy = sy / nrm;
            cz = sz / nrm;
        }
        double mind = 2.0;
#pragma unroll
        for (int r = 0; r < kPer; ++r)
            if (base + r * 32 + lane < n) mind = fmin(mind, cx * px[r] + cy * py[r] + cz * pz[r]);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) mind = fmin(mind, __shfl_xor_sync(0xffffffffu, mind, o));
        if (lane == 0) {
            GroupCap gc;
            gc.cx = cx;
            gc.cy = cy;
            gc.cz = cz;
            if (base < n) {
                // cos of the bounding radius, pushed outwards by far more than the rounding of the dots
                gc.cos_r = fmax(-1.0, fmin(1.0, mind) - 1e-9);
                gc.sin_r = sqrt(fmax(0.0, 1.0 - gc.cos_r * gc.cos_r));
            } else {
                gc.cos_r = 2.0;  // no points
                gc.sin_r = 0.0;
            }
            gc.wsum = sw;
            gcaps[(size_t)blockIdx.x * kGroupsPerTile + warp] = gc;
        }
    }
    // ---- tile cap
    if (lane == 0) {
        red[0][warp] = sx;
        red[1][warp] = sy;
        red[2][warp] = sz;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double cx = 0, cy = 0, cz = 0;
        for (int k = 0; k < 8; ++k) {
            cx += red[0][k];
            cy += red[1][k];
            cz += red[2][k];
        }
        const double nrm = sqrt(cx * cx + cy * cy + cz * cz);
        if (nrm > 1e-9) {
            centre[0] = cx / nrm;
            centre[1] = cy / nrm;
            centre[2] = cz / nrm;
        } else {  // points spread over the whole sphere: any centre, the radius will say pi
            centre[0] = 0.0;
            centre[1] = 0.0;
            centre[2] = 1.0;
        }
    }
    __syncthreads();
    const double cx = centre[0], cy = centre[1], cz = centre[2];
    double mind = 2.0;
#pragma unroll
    for (int r = 0; r < kPer; ++r) {
        const uint32_t s = base + r * 32 + lane;
        if (s < n) mind = fmin(mind, cx * px[r] + cy * py[r] + cz * pz[r]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mind = fmin(mind, __shfl_xor_sync(0xffffffffu, mind, o));
    __syncthreads();
    if (lane == 0) red[0][warp] = mind;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < 8; ++k) mind = fmin(mind, red[0][k]);
        caps[blockIdx.x] = make_double4(cx, cy, cz, fmax(-1.0, fmin(1.0, mind) - 1e-9));
    }
}

// ------------------------------------------------------------------ work list
// Whether no pair between two caps can be in range, without trigonometry: with R = rho_a + rho_b (both radii at most
// 90 degrees, else nothing is decided) and d the cosine between the centres,
//   all pairs beyond theta_max  <=>  theta_ab - R > theta_max  <=>  d < cos(theta_max + R)   (theta_max + R < 180 deg)
//   all pairs closer than theta_min  <=>  theta_ab + R < theta_min  <=>  d > cos(theta_min - R)   (R < theta_min)
// taken with a margin on the cosine: 3e-7 for the padding of the radii (1e-7 rad) and the rounding of these few
// operations, plus `slack` (the caps bound directions; the pair cosine carries the norms: cap_slack).  sa = sin rho_a.
struct RangeTest {
    double c_max, s_max, c_min, s_min;  // cos and sin of theta_max (the last edge) and of theta_min (the first)
    double margin;
    __device__ __forceinline__ bool out_of_range(const double4 a, double sa, const double4 b) const
    {
        if (a.w < 0.0 || b.w < 0.0) return false;
        const double d = a.x * b.x + a.y * b.y + a.z * b.z;
        const double sb = sqrt(fmax(0.0, 1.0 - b.w * b.w));
        const double cR = a.w * b.w - sa * sb, sR = sa * b.w + a.w * sb;  // R in [0, 180 deg]
        if (cR > -c_max && d < c_max * cR - s_max * sR - margin) return true;  // beyond theta_max
        if (cR > c_min && d > c_min * cR + s_min * sR + margin) return true;   // closer than theta_min
        return false;
    }
};

// One CTA per i-tile.  Tests every candidate j-tile cap, then one thread walks the survivor bitmap
// and appends items {ti, first j-tile, number of j-tiles <= kItemTiles}.
__global__ void __launch_bounds__(256)
worklist_kernel(const double4 *__restrict__ caps_a, int ti_begin, int ti_end, const double4 *__restrict__ caps_b,
                int n_tiles_b, int is_auto, int prune, int max_len, int ti_stride, double e_first, double e_last,
                int3 *__restrict__ items, uint32_t capacity, unsigned long long *__restrict__ counters)
{
    extern __shared__ uint32_t keep[];  // bitmap over j tiles
    const int ti = ti_begin + blockIdx.x * ti_stride;
    if (ti >= ti_end) return;
    const int words = (n_tiles_b + 31) / 32;
    const int tj_first = is_auto ? ti : 0;
    const double4 ca = caps_a[ti];
    const double slack = 1.001 * __longlong_as_double((long long)counters[kCtrNormDev]);
    RangeTest rt;
    rt.c_max = e_last;
    rt.s_max = sqrt(fmax(0.0, 1.0 - e_last * e_last));
    rt.c_min = e_first;
    rt.s_min = sqrt(fmax(0.0, 1.0 - e_first * e_first));
    rt.margin = slack + 3e-7;
    const double sa = sqrt(fmax(0.0, 1.0 - ca.w * ca.w));
    uint32_t pruned = 0;
    for (int wbase = 0; wbase < words; wbase += blockDim.x / 32) {
        const int word = wbase + (threadIdx.x >> 5);
        const int tj = word * 32 + (threadIdx.x & 31);
        bool k = false;
        if (word < words && tj < n_tiles_b && tj >= tj_first) {
            k = true;
            if (prune && rt.out_of_range(ca, sa, caps_b[tj])) k = false;
            pruned += k ? 0u : 1u;
        }
        const uint32_t bits = __ballot_sync(0xffffffffu, k);
        if ((threadIdx.x & 31) == 0 && word < words) keep[word] = bits;
    }
    // (one atomic per CTA and counter: thousands of CTAs add to the same two words)
    __shared__ uint32_t pruned_cta;
    if (threadIdx.x == 0) pruned_cta = 0u;
    __syncthreads();
    pruned = __reduce_add_sync(0xffffffffu, pruned);
    if ((threadIdx.x & 31) == 0 && pruned) atomicAdd(&pruned_cta, pruned);
    __syncthreads();
    if (threadIdx.x == 0) {
        if (pruned_cta) atomicAdd(&counters[kCtrTilePairsPruned], (unsigned long long)pruned_cta);
        atomicAdd(&counters[kCtrTilePairsTotal], (unsigned long long)(n_tiles_b - tj_first));
        int tj = tj_first;
        while (tj < n_tiles_b) {
            // skip to the next surviving tile
            uint32_t wv = keep[tj >> 5] >> (tj & 31);
            if (wv == 0) {
                tj = ((tj >> 5) + 1) << 5;
                continue;
            }
            tj += __ffs(wv) - 1;
            if (tj >= n_tiles_b) break;
            int len = 1;
            // the diagonal tile of an auto count is always an item of its own (it runs the i<j variant)
            const bool diag = is_auto && tj == ti;
            while (!diag && len < max_len && tj + len < n_tiles_b && ((keep[(tj + len) >> 5] >> ((tj + len) & 31)) & 1u)) ++len;
            const unsigned long long slot = atomicAdd(&counters[kCtrWorkCount], 1ull);
            if (slot < capacity) items[slot] = make_int3(ti, tj, len);
            tj += len;
        }
    }
}

}  // namespace

// ------------------------------------------------------------------ host side
int prepare_catalogue(acf_ctx *ctx, CatBuffers &buf, const double *xyz, size_t stride, size_t off, size_t cnt,
                      const float *w, Prepared *out)
{
    cudaStream_t st = ctx->stream;
    const uint32_t n = (uint32_t)cnt;
    const int n_tiles = (int)((cnt + kTile - 1) / kTile);
    out->xyz = xyz;
    out->w = w;
    out->stride = stride;
    out->n = cnt;
    out->n_tiles = n_tiles;
    // one slab per catalogue: [PackInfo + weight range (64 B) | pts | pts2 | vj | perm | caps | gcaps | scaps]
    const size_t padded = (size_t)n_tiles * kTile;
    auto up = [](size_t v) { return (v + 255) & ~size_t(255); };
    const size_t o_pts = 256, o_pts2 = o_pts + up(sizeof(float4) * padded), o_vj = o_pts2 + up(sizeof(float4) * padded),
                 o_perm = o_vj + up(sizeof(double) * padded), o_caps = o_perm + up(sizeof(uint32_t) * padded),
                 o_gcaps = o_caps + up(sizeof(double4) * (size_t)n_tiles),
                 o_scaps = o_gcaps + up(sizeof(GroupCap) * (size_t)n_tiles * kGroupsPerTile),
                 total = o_scaps + up(sizeof(GroupCap) * (size_t)n_tiles * kGroupsPerTile * kSubsPerGroup);
    ACF_CUDA_TRY(ctx, buf.slab.reserve(total));
    char *base = buf.slab.as<char>();
    out->pack = reinterpret_cast<PackInfo *>(base);
    ACF_CUDA_TRY(ctx, cudaMemsetAsync(out->pack, 0, 64, st));
    if (cnt == 0) return ACF_OK;
    ACF_CUDA_TRY(ctx, launch_validate(ctx, xyz, stride, off, cnt, w, out->pack));
    ACF_CUDA_TRY(ctx, ctx->s_keys.reserve(sizeof(uint32_t) * 4 * (size_t)n));  // keys x2, idx x2
    const int per_lane = sort_per_lane(n);
    const uint32_t nblocks = (n + sort_block_chunk(per_lane) - 1) / sort_block_chunk(per_lane);
    ACF_CUDA_TRY(ctx, ctx->s_misc.reserve(sizeof(uint32_t) * 256 * (size_t)nblocks));
    out->pts = reinterpret_cast<float4 *>(base + o_pts);
    out->pts2 = reinterpret_cast<float *>(base + o_pts2);
    out->vj = reinterpret_cast<double *>(base + o_vj);
    out->perm = reinterpret_cast<uint32_t *>(base + o_perm);
    out->caps = reinterpret_cast<double4 *>(base + o_caps);
    out->gcaps = reinterpret_cast<GroupCap *>(base + o_gcaps);
    out->scaps = reinterpret_cast<GroupCap *>(base + o_scaps);
    uint32_t *range = reinterpret_cast<uint32_t *>(base + 48);
    uint32_t *k0 = ctx->s_keys.as<uint32_t>(), *k1 = k0 + n, *i0 = k1 + n, *i1 = i0 + n;
    uint32_t *counts = ctx->s_misc.as<uint32_t>();

    int blocks = (int)((n + 255) / 256);
    if (blocks > ctx->num_sms * 16) blocks = ctx->num_sms * 16;
    key_kernel<<<blocks, 256, 0, st>>>(xyz, stride, off, n, k0, i0);
    ctx->last.kernel_launches++;
    for (int pass = 0; pass < 4; ++pass) {
        const int shift = 8 * pass;
        radix_count_kernel<<<nblocks, kSortThreads, 0, st>>>(k0, n, shift, counts, nblocks, per_lane);
        scan_kernel<<<1, 1024, 0, st>>>(counts, 256u * nblocks);
        radix_scatter_kernel<<<nblocks, kSortThreads, 0, st>>>(k0, i0, k1, i1, n, shift, counts, nblocks, per_lane);
        ctx->last.kernel_launches += 3;
        uint32_t *t = k0; k0 = k1; k1 = t;
        t = i0; i0 = i1; i1 = t;
    }
    if (w) {
        wrange_kernel<<<blocks, 256, 0, st>>>(w, off, n, range);
        ctx->last.kernel_launches++;
    }
    gather_caps_kernel<<<n_tiles, 256, 0, st>>>(xyz, stride, off, w, i0, n, out->pts, out->perm, out->caps, out->gcaps, out->scaps, out->pts2,
                                               out->vj, range, out->pack);
    ctx->last.kernel_launches++;
    ACF_CUDA_TRY(ctx, cudaGetLastError());
    return ACF_OK;
}

int build_worklist(acf_ctx *ctx, const Prepared &a, int ti_begin, int ti_end, int ti_stride, const Prepared &b, int is_auto,
                   double e_first, double e_last, int3 *items, uint32_t capacity)
{
    const int n_ti = (ti_end - ti_begin + ti_stride - 1) / ti_stride;
    if (n_ti <= 0 || b.n_tiles == 0) return ACF_OK;
    const size_t smem = sizeof(uint32_t) * (size_t)((b.n_tiles + 31) / 32);
    // items of up to kItemTiles j-tiles; shorter ones when the whole call is only a few tile pairs (small catalogues)
    long long max_len = (long long)n_ti * b.n_tiles / ((long long)ctx->num_sms * 64);
    max_len = max_len < 1 ? 1 : (max_len > kItemTiles ? kItemTiles : max_len);
    if (smem > 48 * 1024) return fail(ctx, ACF_EINVAL, "catalogue too large for the work-list kernel (%d tiles)", b.n_tiles);
    worklist_kernel<<<n_ti, 256, smem, ctx->stream>>>(a.caps, ti_begin, ti_end, b.caps, b.n_tiles, is_auto, ctx->opt_prune, (int)max_len, ti_stride,
                                                     e_first, e_last, items, capacity, ctx->d_counters);
    ctx->last.kernel_launches++;
    ACF_CUDA_TRY(ctx, cudaGetLastError());
    return ACF_OK;
}

}  // namespace acf
