// Stage 2c: cell start/end tables (BASELINE.json north_star; reading S7).
// cell_start[c] = #{k : sorted_hash[k] < c},  cell_end[c] = #{k : sorted_hash[k] <= c}.
// One thread per 8 sorted particles (two 128-bit loads) marks the run boundaries; runs of EMPTY buckets between two
// occupied ones (long in config 3's clipped geometry) are filled by the whole warp, not by one
// thread.  Traffic: 4 B read per particle + 8 B written per bucket.
#include "sph_internal.cuh"

namespace sphb {

constexpr int kCellItems = 8;  // sorted positions per thread (two 128-bit loads in flight)

// boundary between sorted positions k-1 (hash hp) and k (hash hc): closes bucket hp, opens hc;
// the empty buckets in between get start == end == k.  Everything is 32-bit: n < 2^30 and
// n_cells < 2^32 - 1 (sph_create), the bucket before position 0 is passed as hp1 = hp + 1 = 0 and
// the one behind position n - 1 as hc = n_cells.  A long gap is handed back to the caller.
__device__ __forceinline__ void mark_boundary(uint32_t k, uint32_t n, uint32_t hp1, uint32_t hc,
                                              uint32_t *__restrict__ cs, uint32_t *__restrict__ ce,
                                              uint32_t &lo, uint32_t &cnt, uint32_t &fill)
{
    if (hc + 1u == hp1) return;                 // same bucket as the previous position
    if (k < n) cs[hc] = k;
    if (k > 0) ce[hp1 - 1u] = k;
    const uint32_t gap = hc - hp1;              // empty buckets hp1 .. hc - 1
    if (gap > 4u) {             // at most one long gap is kept per thread; earlier ones are
        for (uint32_t c = 0; c < cnt; ++c) { cs[lo + c] = fill; ce[lo + c] = fill; }   // written inline (rare)
        lo = hp1; cnt = gap; fill = k;
    } else {
        for (uint32_t c = hp1; c < hc; ++c) { cs[c] = k; ce[c] = k; }
    }
}

__global__ void __launch_bounds__(256)
cell_ranges_kernel(int64_t n64, const uint32_t *__restrict__ sorted_hash, uint32_t *__restrict__ cs,
                   uint32_t *__restrict__ ce, uint32_t n_cells)
{
    // thread t owns the boundaries k = 8t .. 8t+7 (k == n closes the table)
    const uint32_t n = (uint32_t)n64;
    // (k0 <= n + 8 * 256 < 2^31: no wrap; threads behind the last boundary mark nothing but stay
    //  in the warp collectives)
    const uint32_t k0 = (uint32_t)(((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * kCellItems);
    const int lane = threadIdx.x & 31;
    uint32_t hcur[kCellItems];
    if (k0 + kCellItems <= n && (reinterpret_cast<uintptr_t>(sorted_hash) & 15) == 0) {
#pragma unroll
        for (int q = 0; q < kCellItems / 4; ++q) {
            const uint4 v = __ldcs(reinterpret_cast<const uint4 *>(sorted_hash + k0) + q);
            hcur[4 * q] = v.x; hcur[4 * q + 1] = v.y; hcur[4 * q + 2] = v.z; hcur[4 * q + 3] = v.w;
        }
    } else {
#pragma unroll
        for (int j = 0; j < kCellItems; ++j)
            hcur[j] = (k0 + j < n) ? sorted_hash[k0 + j] : n_cells;
    }
    // hash of position k0 - 1 (+ 1): the previous lane's last one, lane 0 reads it
    uint32_t hp1 = __shfl_up_sync(0xffffffffu, hcur[kCellItems - 1], 1) + 1u;
    if (lane == 0) hp1 = (k0 == 0) ? 0u : ((k0 - 1 < n) ? sorted_hash[k0 - 1] + 1u : n_cells + 1u);
    uint32_t lo = 0, cnt = 0;   // long empty-bucket range [lo, lo + cnt) to fill with `fill`
    uint32_t fill = 0;
#pragma unroll
    for (int j = 0; j < kCellItems; ++j) {
        if (k0 + j <= n) mark_boundary(k0 + j, n, hp1, hcur[j], cs, ce, lo, cnt, fill);
        hp1 = hcur[j] + 1u;
    }
    // long gaps (config 3's clipped geometry has runs of thousands) are filled by the whole warp
    uint32_t pending = __ballot_sync(0xffffffffu, cnt > 0);
    while (pending) {
        const int src = __ffs(pending) - 1;
        pending &= pending - 1;
        const uint32_t l = __shfl_sync(0xffffffffu, lo, src);
        const uint32_t m = __shfl_sync(0xffffffffu, cnt, src);
        const uint32_t f = __shfl_sync(0xffffffffu, fill, src);
        for (uint32_t c = lane; c < m; c += 32) { cs[l + c] = f; ce[l + c] = f; }
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
