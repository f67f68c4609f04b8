// Stage 4a dispatcher: picks the shared-memory tiled kernel, or the direct global-memory kernel
// when forced (SPH_FLAG_INTERACT_DIRECT).  pair_count accumulates (callers zero it).
#include "sph_internal.cuh"
#include "interact_math.cuh"

namespace sphb {

int launch_interact(sph_ctx *c, int64_t n, const sph_state *sorted, const uint32_t *sorted_hash,
                    const uint32_t *cs, const uint32_t *ce, float *drho, float *acc,
                    float *const dsig[6], unsigned long long *pair_count)
{
    if (n == 0) return SPH_OK;
    InteractIn in;
    InteractOut out;
    in.posm = reinterpret_cast<const float4 *>(sorted->posm);
    in.velr = reinterpret_cast<const float4 *>(sorted->velr);
    out.drho = drho;
    out.acc = reinterpret_cast<float4 *>(acc);
    for (int i = 0; i < 6; ++i) { in.sig[i] = sorted->sig[i]; out.dsig[i] = dsig[i]; }
    if (c->params.flags & SPH_FLAG_INTERACT_DIRECT)
        return launch_interact_direct(c, n, in, sorted_hash, cs, ce, out, pair_count);
    return launch_interact_tiled(c, n, in, sorted_hash, cs, ce, out, pair_count);
}

}  // namespace sphb
