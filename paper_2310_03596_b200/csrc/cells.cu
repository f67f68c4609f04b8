// Stage 2c: cell start/end tables (BASELINE.json north_star; reading S7).
// cell_start[c] = #{k : sorted_hash[k] < c},  cell_end[c] = #{k : sorted_hash[k] <= c}.
// One thread per sorted particle marks the run boundaries; runs of EMPTY buckets between two
// occupied ones (long in config 3's clipped geometry) are filled by the whole warp, not by one
// thread.  Traffic: 4 B read per particle + 8 B written per bucket.
#include "sph_internal.cuh"

namespace sphb {

__global__ void __launch_bounds__(256)
cell_ranges_kernel(int64_t n, const uint32_t *__restrict__ sorted_hash, uint32_t *__restrict__ cs,
                   uint32_t *__restrict__ ce, uint32_t n_cells)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    // boundary between sorted positions k-1 and k (k == n closes the table)
    int64_t lo = 0, hi = -1;  // empty-bucket range [lo, hi] to fill with value k
    uint32_t fill = 0;
    if (k <= n) {
        const int64_t hp = (k == 0) ? -1 : (int64_t)sorted_hash[k - 1];
        const int64_t hc = (k == n) ? (int64_t)n_cells : (int64_t)sorted_hash[k];
        if (hc != hp) {
            if (k < n) cs[hc] = (uint32_t)k;
            if (k > 0) ce[hp] = (uint32_t)k;
            lo = hp + 1;
            hi = hc - 1;
            fill = (uint32_t)k;
        }
    }
    // short gaps inline, long gaps cooperatively
    const int64_t gap = hi - lo + 1;
    if (gap > 0 && gap <= 4) {
        for (int64_t c = lo; c <= hi; ++c) { cs[c] = fill; ce[c] = fill; }
    }
    uint32_t pending = __ballot_sync(0xffffffffu, gap > 4);
    while (pending) {
        const int src = __ffs(pending) - 1;
        pending &= pending - 1;
        const int64_t l = __shfl_sync(0xffffffffu, lo, src);
        const int64_t h = __shfl_sync(0xffffffffu, hi, src);
        const uint32_t f = __shfl_sync(0xffffffffu, fill, src);
        for (int64_t c = l + lane; c <= h; c += 32) { cs[c] = f; ce[c] = f; }
    }
}

int launch_cell_ranges(sph_ctx *c, int64_t n, const uint32_t *sorted_hash, uint32_t *cs, uint32_t *ce)
{
    // n + 1 boundaries (k = 0 .. n); with n == 0 the single boundary fills every bucket with 0
    const int blocks = div_up(n + 1, 256);
    cell_ranges_kernel<<<blocks, 256, 0, c->stream>>>(n, sorted_hash, cs, ce, c->grid.n_cells);
    SPH_CHECK_LAUNCH(c);
    return SPH_OK;
}

}  // namespace sphb
