// acf_static.cu -- acf_pair_count_static: a pair count that allocates nothing (include/acf.h).
//
// Some callers cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that
// forbid it.  Every other entry point of the library works on a context whose scratch buffers grow on demand.
// This one needs no context: its kernel is a variant of the fp64 reference kernel (acf_kernels_ref.cu: every pair
// evaluated as include/acf.h defines it) whose scratch memory -- the device copy of the edges,
// a status word and one partial histogram per CTA -- lives in a file-scope __device__ array of fixed size.  The
// array is part of the library's device image: every GPU that loads the library holds its 4.2 MB until the process
// exits.  All calls share it, so calls that overlap on one GPU (two streams, two threads) race; calls on one
// stream are ordered and safe.
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "acf.h"
#include "acf_device.cuh"

namespace {

constexpr int kThreads = 128;  // rows per CTA (one per thread)
constexpr int kTileJ = 256;    // columns staged in shared memory at a time
constexpr int kMaxCtas = ACF_STATIC_MAX_POINTS / kThreads;
static_assert(ACF_STATIC_MAX_POINTS % kThreads == 0, "");

// [edges: nbins + 1 doubles | status: u32 number of invalid points | partial histograms: u32[n_ctas][nbins]]
constexpr size_t kEdgesBytes = ((sizeof(double) * (ACF_MAX_BINS + 1) + 255) / 256) * 256;
constexpr size_t kStatusBytes = 256;
constexpr size_t kPartialBytes = sizeof(unsigned int) * (size_t)kMaxCtas * ACF_MAX_BINS;
constexpr size_t kScratchBytes = kEdgesBytes + kStatusBytes + kPartialBytes;

// In host code this name is a host-side stand-in, not a device address: the address a kernel may use comes
// from cudaGetSymbolAddress (scratch_of below).
static __device__ __align__(256) unsigned char g_static_scratch[kScratchBytes];

__device__ __forceinline__ bool point_ok(double x, double y, double z)
{
    return isfinite(x) && isfinite(y) && isfinite(z) && fabs(x * x + y * y + z * z - 1.0) <= 1e-6;
}

// grid.x: row blocks of kThreads rows; grid.y: column chunks.  Every CTA writes all nbins words of its own
// partial histogram (nothing there has to start at zero); the status word is cleared by the host before the launch.
__global__ void __launch_bounds__(kThreads)
pair_count_static_kernel(const double *__restrict__ a, size_t n_a, const double *__restrict__ b, size_t n_b, int nbins,
                         int is_auto, unsigned char *__restrict__ scratch)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *s_edges = reinterpret_cast<double *>(smem_raw);  // nbins + 1
    double *s_x = s_edges + (nbins + 1);                     // kTileJ each
    double *s_y = s_x + kTileJ;
    double *s_z = s_y + kTileJ;
    unsigned int *s_cnt = reinterpret_cast<unsigned int *>(s_z + kTileJ);  // nbins

    const double *edges = reinterpret_cast<const double *>(scratch);
    unsigned int *status = reinterpret_cast<unsigned int *>(scratch + kEdgesBytes);
    unsigned int *partial = reinterpret_cast<unsigned int *>(scratch + kEdgesBytes + kStatusBytes) +
                            ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * (size_t)nbins;

    for (int k = threadIdx.x; k <= nbins; k += blockDim.x) s_edges[k] = edges[k];
    for (int k = threadIdx.x; k < nbins; k += blockDim.x) s_cnt[k] = 0;

    const size_t i = (size_t)blockIdx.x * kThreads + threadIdx.x;
    const bool row_ok = i < n_a;
    double xi = 0, yi = 0, zi = 0;
    unsigned int bad = 0;
    if (row_ok) {
        xi = a[i];
        yi = a[n_a + i];
        zi = a[2 * n_a + i];
        if (blockIdx.y == 0 && !point_ok(xi, yi, zi)) ++bad;  // every row is checked by the first column chunk
    }
    const size_t chunk = (n_b + gridDim.y - 1) / gridDim.y;
    size_t j_lo = (size_t)blockIdx.y * chunk;
    j_lo = j_lo < n_b ? j_lo : n_b;
    const size_t j_hi = j_lo + chunk < n_b ? j_lo + chunk : n_b;
    if (is_auto) {
        // no column at or before the first row of this block pairs with it
        const size_t first = (size_t)blockIdx.x * kThreads + 1;
        if (j_lo < first) j_lo = first < j_hi ? first : j_hi;
    }
    __syncthreads();

    for (size_t j0 = j_lo; j0 < j_hi; j0 += kTileJ) {
        const int jn = (int)((j_hi - j0) < (size_t)kTileJ ? (j_hi - j0) : (size_t)kTileJ);
        for (int t = threadIdx.x; t < jn; t += blockDim.x) {
            const double x = b[j0 + t], y = b[n_b + j0 + t], z = b[2 * n_b + j0 + t];
            s_x[t] = x;
            s_y[t] = y;
            s_z[t] = z;
            if (blockIdx.x == 0 && !is_auto && !point_ok(x, y, z)) ++bad;  // every column, by the first row block
        }
        __syncthreads();
        if (row_ok) {
            for (int t = 0; t < jn; ++t) {
                if (is_auto && j0 + t <= i) continue;  // unordered pairs i < j
                const double c = acf::pair_cos_fp64(xi, yi, zi, s_x[t], s_y[t], s_z[t]);
                const int k = acf::bin_of_fp64(c, s_edges, nbins);
                if (k >= 0) atomicAdd(&s_cnt[k], 1u);
            }
        }
        __syncthreads();
    }
    for (int k = threadIdx.x; k < nbins; k += blockDim.x) partial[k] = s_cnt[k];
    bad = __reduce_add_sync(0xffffffffu, bad);
    if ((threadIdx.x & 31) == 0 && bad) atomicAdd(status, bad);
}

// counts[k] = sum of the CTAs' partial histograms; *bad_out = the status word.
__global__ void __launch_bounds__(256)
reduce_static_kernel(const unsigned char *__restrict__ scratch, int nbins, int n_ctas, unsigned long long *__restrict__ counts,
                     unsigned int *__restrict__ bad_out)
{
    const unsigned int *status = reinterpret_cast<const unsigned int *>(scratch + kEdgesBytes);
    const unsigned int *partial = reinterpret_cast<const unsigned int *>(scratch + kEdgesBytes + kStatusBytes);
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < nbins) {
        unsigned long long sum = 0;
        for (int c = 0; c < n_ctas; ++c) sum += partial[(size_t)c * nbins + k];
        counts[k] = sum;
    }
    if (k == 0 && bad_out) *bad_out = status[0];
}

// ---- host side ------------------------------------------------------------------------------------
constexpr int kMaxDevices = 64;
std::mutex g_mu;
unsigned char *g_scratch_ptr[kMaxDevices];  // the array's device address, per device (zero: not asked yet)

int fail(char *err, size_t err_len, int code, const char *fmt, ...)
{
    if (err && err_len) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(err, err_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

// The device address of g_static_scratch on `device`, which must be the current device: asked once per device.
// (The first call on a device also makes the runtime load the library's device image there: set-up, not to be captured.)
cudaError_t scratch_of(int device, unsigned char **out)
{
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_ptr[device]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return e;
        g_scratch_ptr[device] = static_cast<unsigned char *>(p);
    }
    *out = g_scratch_ptr[device];
    return cudaSuccess;
}

// puts the caller's device back when the call returns
struct DeviceGuard {
    int prev = -1;
    ~DeviceGuard()
    {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

}  // namespace

extern "C" int acf_pair_count_static(int device, const double *d_a, size_t n_a, const double *d_b, size_t n_b,
                                     const double *cos_edges, int nbins, int is_auto, uint64_t *d_counts, uint32_t *d_bad,
                                     void *cuda_stream, char *err, size_t err_len)
{
    if (err && err_len) err[0] = 0;
    if (!cos_edges) return fail(err, err_len, ACF_EINVAL, "cos_edges is NULL");
    if (nbins < 1 || nbins > ACF_MAX_BINS) return fail(err, err_len, ACF_EINVAL, "nbins = %d: must be in [1, %d]", nbins, ACF_MAX_BINS);
    for (int m = 0; m <= nbins; ++m) {
        if (!(cos_edges[m] >= -1.0 && cos_edges[m] <= 1.0)) return fail(err, err_len, ACF_EINVAL, "cos_edges must lie within [-1, 1]");
        if (m && !(cos_edges[m] < cos_edges[m - 1])) return fail(err, err_len, ACF_EINVAL, "cos_edges must be strictly descending");
    }
    if (!d_counts) return fail(err, err_len, ACF_EINVAL, "d_counts is NULL");
    if ((n_a && !d_a) || (n_b && !d_b)) return fail(err, err_len, ACF_EINVAL, "catalogue pointer is NULL");
    is_auto = is_auto != 0;
    if (is_auto && (d_a != d_b || n_a != n_b)) return fail(err, err_len, ACF_EINVAL, "is_auto needs d_b == d_a and n_b == n_a");
    if (n_a > ACF_STATIC_MAX_POINTS || n_b > ACF_STATIC_MAX_POINTS)
        return fail(err, err_len, ACF_EINVAL,
                    "acf_pair_count_static takes at most ACF_STATIC_MAX_POINTS = %d points per catalogue (its scratch memory is a fixed "
                    "array; got n_a = %zu, n_b = %zu): use acf_pair_count",
                    ACF_STATIC_MAX_POINTS, n_a, n_b);
    if (device < 0 || device >= kMaxDevices) return fail(err, err_len, ACF_EINVAL, "device index %d out of range", device);

    DeviceGuard guard;
    cudaError_t e = cudaGetDevice(&guard.prev);
    if (e == cudaSuccess) e = cudaSetDevice(device);
    if (e != cudaSuccess) return fail(err, err_len, ACF_ECUDA, "cudaSetDevice(%d): %s", device, cudaGetErrorString(e));
    unsigned char *scratch = nullptr;
    e = scratch_of(device, &scratch);
    if (e != cudaSuccess) return fail(err, err_len, ACF_ECUDA, "cudaGetSymbolAddress: %s", cudaGetErrorString(e));
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);

    // the status word starts at zero; the edges go into the array (a copy, not an allocation)
    e = cudaMemsetAsync(scratch + kEdgesBytes, 0, kStatusBytes, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(scratch, cos_edges, sizeof(double) * (size_t)(nbins + 1), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return fail(err, err_len, ACF_ECUDA, "staging the edges: %s", cudaGetErrorString(e));

    int n_ctas = 0;
    if (n_a > 0 && n_b > 0 && !(is_auto && n_a < 2)) {
        const unsigned gx = (unsigned)((n_a + kThreads - 1) / kThreads);  // <= kMaxCtas
        unsigned gy = (unsigned)kMaxCtas / gx;
        const unsigned cols = (unsigned)((n_b + kTileJ - 1) / kTileJ);
        gy = gy < 1u ? 1u : (gy > cols ? cols : gy);
        n_ctas = (int)(gx * gy);
        const size_t smem = sizeof(double) * (size_t)(nbins + 1) + sizeof(double) * 3 * kTileJ + sizeof(unsigned int) * (size_t)nbins;
        pair_count_static_kernel<<<dim3(gx, gy), kThreads, smem, st>>>(d_a, n_a, d_b, n_b, nbins, is_auto, scratch);
    }
    reduce_static_kernel<<<(nbins + 255) / 256, 256, 0, st>>>(scratch, nbins, n_ctas, reinterpret_cast<unsigned long long *>(d_counts), d_bad);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(err, err_len, ACF_ECUDA, "kernel launch: %s", cudaGetErrorString(e));
    return ACF_OK;
}
