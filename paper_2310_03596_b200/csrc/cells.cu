// Stage 2c: cell start/end tables (BASELINE.json north_star; reading S7).
// cell_start[c] = #{k : sorted_hash[k] < c},  cell_end[c] = #{k : sorted_hash[k] <= c}.
// One thread per 8 sorted particles (two 128-bit loads) marks the run boundaries; runs of EMPTY buckets between two
// occupied ones (long in config 3's clipped geometry) are filled by the whole warp, not by one
// thread.  Traffic: 4 B read per particle + 8 B written per bucket.
#include "sph_internal.cuh"

namespace sphb {

constexpr int kCellItems = 8;  // sorted positions per thread (two 128-bit loads in flight)

// boundary between sorted positions k-1 (hash hp) and k (hash hc): closes bucket hp, opens hc;
// the empty buckets in between get start == end == k.  Returns the gap range for the caller.
__device__ __forceinline__ void mark_boundary(int64_t k, int64_t n, int64_t hp, int64_t hc,
                                              uint32_t *__restrict__ cs, uint32_t *__restrict__ ce,
                                              int64_t &lo, int64_t &hi, uint32_t &fill)
{
    if (hc == hp) return;
    if (k < n) cs[hc] = (uint32_t)k;
    if (k > 0) ce[hp] = (uint32_t)k;
    const int64_t l = hp + 1, h = hc - 1;
    if (h - l + 1 > 4) {        // at most one long gap is kept per thread; earlier ones are
        if (hi >= lo)           // written inline (rare: two long gaps inside 8 positions)
            for (int64_t c = lo; c <= hi; ++c) { cs[c] = fill; ce[c] = fill; }
        lo = l; hi = h; fill = (uint32_t)k;
    } else {
        for (int64_t c = l; c <= h; ++c) { cs[c] = (uint32_t)k; ce[c] = (uint32_t)k; }
    }
}

__global__ void __launch_bounds__(256)
cell_ranges_kernel(int64_t n, const uint32_t *__restrict__ sorted_hash, uint32_t *__restrict__ cs,
                   uint32_t *__restrict__ ce, uint32_t n_cells)
{
    // thread t owns the boundaries k = 8t .. 8t+7 (k == n closes the table)
    const int64_t k0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * kCellItems;
    const int lane = threadIdx.x & 31;
    int64_t hcur[kCellItems];
    if (k0 + kCellItems <= n && (reinterpret_cast<uintptr_t>(sorted_hash) & 15) == 0) {
#pragma unroll
        for (int q = 0; q < kCellItems / 4; ++q) {
            const uint4 v = __ldcs(reinterpret_cast<const uint4 *>(sorted_hash + k0) + q);
            hcur[4 * q] = v.x; hcur[4 * q + 1] = v.y; hcur[4 * q + 2] = v.z; hcur[4 * q + 3] = v.w;
        }
    } else {
#pragma unroll
        for (int j = 0; j < kCellItems; ++j)
            hcur[j] = (k0 + j < n) ? (int64_t)sorted_hash[k0 + j] : (int64_t)n_cells;
    }
    // hash of position k0 - 1: the previous lane's last one, lane 0 reads it
    int64_t hprev = __shfl_up_sync(0xffffffffu, hcur[kCellItems - 1], 1);
    if (lane == 0) hprev = (k0 == 0) ? -1 : ((k0 - 1 < n) ? (int64_t)sorted_hash[k0 - 1] : (int64_t)n_cells);
    int64_t lo = 0, hi = -1;  // long empty-bucket range [lo, hi] to fill with `fill`
    uint32_t fill = 0;
#pragma unroll
    for (int j = 0; j < kCellItems; ++j) {
        if (k0 + j <= n) mark_boundary(k0 + j, n, hprev, hcur[j], cs, ce, lo, hi, fill);
        hprev = hcur[j];
    }
    // long gaps (config 3's clipped geometry has runs of thousands) are filled by the whole warp
    uint32_t pending = __ballot_sync(0xffffffffu, hi >= lo);
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
    const int blocks = div_up(div_up(n + 1, kCellItems), 256);
    cell_ranges_kernel<<<blocks, 256, 0, c->stream>>>(n, sorted_hash, cs, ce, c->grid.n_cells);
    SPH_CHECK_LAUNCH(c);
    return SPH_OK;
}

}  // namespace sphb
