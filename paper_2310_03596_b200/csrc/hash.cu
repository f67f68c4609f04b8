// Stage 1: bucket hash (step a PAPER.md:19; readings S1-S3).
// Pure streaming kernel: 16 B read + 4 B written per particle, HBM-bound.
#include "sph_internal.cuh"

namespace sphb {

__global__ void __launch_bounds__(256) hash_kernel(int64_t n, const float4 *__restrict__ posm,
                                                   uint32_t *__restrict__ hash, Grid g)
{
    // two particles per thread, both loads issued before use
    int64_t i0 = ((int64_t)blockIdx.x * blockDim.x) * 2 + threadIdx.x;
    int64_t i1 = i0 + blockDim.x;
    float4 p0, p1;
    if (i0 < n) p0 = __ldcs(posm + i0);
    if (i1 < n) p1 = __ldcs(posm + i1);
    if (i0 < n) {
        hash[i0] = bucket_hash(p0, g);
    }
    if (i1 < n) {
        hash[i1] = bucket_hash(p1, g);
    }
}

int launch_hash(sph_ctx *c, int64_t n, const float *posm, uint32_t *hash)
{
    if (n == 0) return SPH_OK;
    int blocks = div_up(n, 512);
    hash_kernel<<<blocks, 256, 0, c->stream>>>(n, reinterpret_cast<const float4 *>(posm), hash,
                                               c->grid);
    SPH_CHECK_LAUNCH(c);
    return SPH_OK;
}

}  // namespace sphb
