// Stage 4a, reference-shaped kernel: one thread per particle walking the 27-bucket stencil
// straight out of global memory ("restricted to its bucket and to the surrounding
// buckets"; steps e/f PAPER.md:24-25; equations DESIGN.md O6-O8).
//
// This is the simple first CUDA path and the fallback for tiles that do not fit the shared-
// memory kernel in interact_tiled.cu.  x-fastest hashing makes the three buckets (cx-1, cx,
// cx+1) of a stencil row contiguous, so the 27 buckets are 9 contiguous runs.
#include "sph_internal.cuh"
#include "interact_math.cuh"

namespace sphb {

__global__ void __launch_bounds__(128)
interact_direct_kernel(int64_t n, InteractIn in, const uint32_t *__restrict__ sorted_hash,
                       const uint32_t *__restrict__ cs, const uint32_t *__restrict__ ce, Grid g,
                       Consts k, InteractOut out, unsigned long long *pair_count, int mode)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long my_pairs = 0;
    if (i < n) {
        const uint32_t h = sorted_hash[i];
        const int cx = h % g.nx, cy = (h / g.nx) % g.ny, cz = h / (g.nx * g.ny);
        my_pairs = direct_particle(i, cx, cy, cz, in, cs, ce, g, k, out, mode);
    }
    if (pair_count) {
        // warp, then one atomic per warp
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) my_pairs += __shfl_xor_sync(0xffffffffu, my_pairs, o);
        if ((threadIdx.x & 31) == 0 && my_pairs) atomicAdd(pair_count, my_pairs);
    }
}

int launch_interact_direct(sph_ctx *c, int64_t n, const InteractIn &in, const uint32_t *sorted_hash,
                           const uint32_t *cs, const uint32_t *ce, const InteractOut &out,
                           unsigned long long *pair_count, int mode)
{
    Consts kc = c->consts;
    if (in.h) kc.cF = kc.cF_varh;   // per-particle smoothing lengths: h_ij^-5 is applied per pair
    interact_direct_kernel<<<div_up(n, 128), 128, 0, c->stream>>>(n, in, sorted_hash, cs, ce, c->grid,
                                                                  kc, out, pair_count, mode);
    SPH_CHECK_LAUNCH(c);
    return SPH_OK;
}

}  // namespace sphb
