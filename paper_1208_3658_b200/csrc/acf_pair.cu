// acf_pair.cu -- fast path (placeholder while the fp32-certify kernel is being written):
// routes to the fp64 reference kernel.
#include "acf_internal.h"

namespace acf {
int run_pair_count_fast(acf_ctx *ctx, const double *d_a, const float *d_wa, size_t n_a, size_t i_begin,
                        size_t i_end, const double *d_b, const float *d_wb, size_t n_b, const double *,
                        int nbins, int is_auto, unsigned long long *d_counts, double *d_wsums)
{
    ACF_CUDA_TRY(ctx, launch_pair_count_fp64(ctx, d_a, d_wa, n_a, i_begin, i_end, d_b, d_wb, n_b,
                                             ctx->s_edges.as<double>(), nbins, is_auto, d_counts, d_wsums));
    return ACF_OK;
}
}  // namespace acf
