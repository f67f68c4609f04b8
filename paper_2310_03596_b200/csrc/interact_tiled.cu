#include "sph_internal.cuh"
#include "interact_math.cuh"
namespace sphb {
int launch_interact_tiled(sph_ctx *c, int64_t n, const InteractIn &in, const uint32_t *sorted_hash,
                          const uint32_t *cs, const uint32_t *ce, const InteractOut &out,
                          unsigned long long *pair_count)
{
    return launch_interact_direct(c, n, in, sorted_hash, cs, ce, out, pair_count);
}
}  // namespace sphb
