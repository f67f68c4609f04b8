// Stage 2a: hand-written onesweep LSD radix sort on (hash, id)  (reading S5).
//
// One histogram kernel reads the keys once and builds the digit histograms of every pass.
// Each pass is then ONE kernel: a tile of 4096 keys is ranked with warp-level match/popc
// (stable), the tile's per-digit counts are chained to the previous tiles with decoupled
// look-back (single 32-bit status word = 2 flag bits + 30-bit count, so no fence is needed), and
// keys/values are staged through shared memory so each digit's run leaves as one contiguous
// write.  Tiles take their index from an atomic ticket, which guarantees forward progress of the
// look-back chain.  Values of the first pass are the implicit ids 0..n-1 (never read), and only
// the live key bits ceil(log2(cells)) are sorted.  Stability + ascending ids on input give the
// lexicographic (hash, id) order.
#include "sph_internal.cuh"

namespace sphb {

// --------------------------------------------------------------------------- histograms
__global__ void __launch_bounds__(256) radix_hist_kernel(int64_t n, const uint32_t *__restrict__ keys,
                                                         uint32_t *__restrict__ hist, int n_passes)
{
    __shared__ uint32_t s_hist[kMaxPasses][kRadix];
    for (int i = threadIdx.x; i < kMaxPasses * kRadix; i += blockDim.x) (&s_hist[0][0])[i] = 0;
    __syncthreads();
    const int64_t stride = (int64_t)gridDim.x * blockDim.x * 4;
    // block-uniform trip count, so every warp-collective below runs with a full mask
    for (int64_t tb = (int64_t)blockIdx.x * blockDim.x * 4; tb < n; tb += stride) {
        const int64_t base = tb + (int64_t)threadIdx.x * 4;
        uint32_t k[4] = {0, 0, 0, 0};
        int cnt = 0;
        if (base + 4 <= n) {
            uint4 v = __ldcs(reinterpret_cast<const uint4 *>(keys + base));
            k[0] = v.x; k[1] = v.y; k[2] = v.z; k[3] = v.w;
            cnt = 4;
        } else if (base < n) {
            cnt = (int)(n - base);
            for (int j = 0; j < cnt; ++j) k[j] = keys[base + j];
        }
        for (int p = 0; p < n_passes; ++p) {
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                // warp-aggregate equal digits (spatially coherent ids share their high digits)
                const bool valid = j < cnt;
                const uint32_t d = valid ? ((k[j] >> (p * kRadixBits)) & (kRadix - 1)) : 0x1000u;
                const uint32_t peers = __match_any_sync(0xffffffffu, d);
                if (valid && (peers & lanemask_lt()) == 0) atomicAdd(&s_hist[p][d], __popc(peers));
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n_passes * kRadix; i += blockDim.x) {
        uint32_t v = (&s_hist[0][0])[i];
        if (v) atomicAdd(hist + i, v);
    }
}

// exclusive scan of each pass's 256-bin histogram, in place; one block per pass
__global__ void __launch_bounds__(kRadix) radix_hist_scan_kernel(uint32_t *hist)
{
    __shared__ uint32_t s_warp[kRadix / 32];
    uint32_t *h = hist + blockIdx.x * kRadix;
    const int t = threadIdx.x, lane = t & 31, w = t >> 5;
    const uint32_t v = h[t];
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t x = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += x;
    }
    if (lane == 31) s_warp[w] = inc;
    __syncthreads();
    uint32_t add = 0;
    for (int i = 0; i < w; ++i) add += s_warp[i];
    h[t] = inc - v + add;
}

// --------------------------------------------------------------------------- onesweep pass
template <bool FIRST>
__global__ void __launch_bounds__(kSortThreads)
onesweep_kernel(int64_t n, const uint32_t *__restrict__ keys_in, const uint32_t *__restrict__ vals_in,
                uint32_t *__restrict__ keys_out, uint32_t *__restrict__ vals_out,
                const uint32_t *__restrict__ hist_excl, uint32_t *status, uint32_t *ticket, int shift)
{
    constexpr int kWarps = kSortThreads / 32;
    __shared__ uint32_t s_warp_hist[kWarps][kRadix];
    __shared__ uint32_t s_keys[kSortTile];
    __shared__ uint32_t s_vals[kSortTile];
    __shared__ uint32_t s_digit_base[kRadix];
    __shared__ uint32_t s_gbase[kRadix];
    __shared__ uint32_t s_scan[kWarps];
    __shared__ uint32_t s_tile;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
#pragma unroll
    for (int i = tid; i < kWarps * kRadix; i += kSortThreads) (&s_warp_hist[0][0])[i] = 0;
    __syncthreads();
    const uint32_t tile = s_tile;
    const int64_t tile_base = (int64_t)tile * kSortTile;
    const int tile_valid = (int)min((int64_t)kSortTile, n - tile_base);
    const int64_t chunk = tile_base + warp * (32 * kSortItems) + lane;

    // ---- load (warp-striped: item r of lane l = chunk[r*32 + l]) ----
    uint32_t key[kSortItems], val[kSortItems];
#pragma unroll
    for (int r = 0; r < kSortItems; ++r) {
        const int64_t idx = chunk + r * 32;
        key[r] = idx < n ? __ldcs(keys_in + idx) : 0xFFFFFFFFu;
    }
    if (!FIRST) {
#pragma unroll
        for (int r = 0; r < kSortItems; ++r) {
            const int64_t idx = chunk + r * 32;
            val[r] = idx < n ? __ldcs(vals_in + idx) : 0u;
        }
    } else {
#pragma unroll
        for (int r = 0; r < kSortItems; ++r) val[r] = (uint32_t)(chunk + r * 32);
    }

    // ---- stable rank inside the warp ----
    uint32_t rank[kSortItems];
    const uint32_t lt = lanemask_lt();
#pragma unroll
    for (int r = 0; r < kSortItems; ++r) {
        const uint32_t d = (key[r] >> shift) & (kRadix - 1);
        const uint32_t peers = __match_any_sync(0xffffffffu, d);
        const uint32_t before = __popc(peers & lt);
        uint32_t basev = 0;
        if (before == 0) {
            basev = s_warp_hist[warp][d];
            s_warp_hist[warp][d] = basev + __popc(peers);
        }
        __syncwarp();
        basev = __shfl_sync(0xffffffffu, basev, __ffs(peers) - 1);
        rank[r] = basev + before;
    }
    __syncthreads();

    // ---- per-digit work: thread d owns digit d ----
    {
        const int d = tid;
        uint32_t run = 0;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) {
            const uint32_t c = s_warp_hist[w][d];
            s_warp_hist[w][d] = run;
            run += c;
        }
        // padding keys (0xFFFFFFFF) sit at the very end of digit 255
        const uint32_t valid_total = (d == kRadix - 1) ? run - (uint32_t)(kSortTile - tile_valid) : run;
        uint32_t *my_status = status + (size_t)tile * kRadix + d;
        st_volatile_u32(my_status, (tile == 0 ? kFlagPrefix : kFlagAgg) | valid_total);

        // block exclusive scan of `run` over digits -> position of the digit's run in the tile
        uint32_t inc = run;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t x = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += x;
        }
        if (lane == 31) s_scan[warp] = inc;
        __syncthreads();
        uint32_t add = 0;
#pragma unroll
        for (int i = 0; i < kWarps; ++i) add += (i < warp) ? s_scan[i] : 0u;
        const uint32_t dbase = inc - run + add;
        s_digit_base[d] = dbase;

        // decoupled look-back over the previous tiles
        uint32_t excl = 0;
        if (tile > 0) {
            int64_t t = (int64_t)tile - 1;
            while (true) {
                const uint32_t s = ld_volatile_u32(status + (size_t)t * kRadix + d);
                const uint32_t f = s & kFlagMask;
                if (f == 0) continue;  // not published yet
                excl += s & kValueMask;
                if (f == kFlagPrefix) break;
                --t;
            }
            st_volatile_u32(my_status, kFlagPrefix | (excl + valid_total));
        }
        s_gbase[d] = hist_excl[d] + excl - dbase;
    }
    __syncthreads();

    // ---- scatter into the tile-local sorted order ----
#pragma unroll
    for (int r = 0; r < kSortItems; ++r) {
        const uint32_t d = (key[r] >> shift) & (kRadix - 1);
        const uint32_t pos = s_digit_base[d] + s_warp_hist[warp][d] + rank[r];
        s_keys[pos] = key[r];
        s_vals[pos] = val[r];
    }
    __syncthreads();

    // ---- each digit run leaves as one contiguous stretch ----
#pragma unroll
    for (int k = 0; k < kSortItems; ++k) {
        const int p = tid + k * kSortThreads;
        if (p < tile_valid) {
            const uint32_t kk = s_keys[p];
            const uint32_t d = (kk >> shift) & (kRadix - 1);
            const uint32_t dst = s_gbase[d] + (uint32_t)p;
            keys_out[dst] = kk;
            vals_out[dst] = s_vals[p];
        }
    }
}

__global__ void __launch_bounds__(256) iota_copy_kernel(int64_t n, const uint32_t *__restrict__ hash,
                                                        uint32_t *__restrict__ sorted_hash,
                                                        uint32_t *__restrict__ perm)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { sorted_hash[i] = hash[i]; perm[i] = (uint32_t)i; }
}

int launch_sort(sph_ctx *c, int64_t n, const uint32_t *hash, uint32_t *sorted_hash, uint32_t *perm)
{
    if (n == 0) return SPH_OK;
    const int P = c->n_passes;
    if (P == 0) {  // a single bucket: the order is the id order
        iota_copy_kernel<<<div_up(n, 256), 256, 0, c->stream>>>(n, hash, sorted_hash, perm);
        SPH_CHECK_LAUNCH(c);
        return SPH_OK;
    }
    const int64_t tiles = (n + kSortTile - 1) / kSortTile;
    SPH_CUDA_TRY(c, cudaMemsetAsync(c->hist, 0, sizeof(uint32_t) * kMaxPasses * kRadix, c->stream));
    SPH_CUDA_TRY(c, cudaMemsetAsync(c->tile_counter, 0, sizeof(uint32_t) * (kMaxPasses + 2), c->stream));
    SPH_CUDA_TRY(c, cudaMemsetAsync(c->tile_status, 0, sizeof(uint32_t) * (size_t)P * tiles * kRadix,
                                    c->stream));
    int hb = (int)min((int64_t)c->num_sms * 8, (n + 1023) / 1024);
    if (hb < 1) hb = 1;
    radix_hist_kernel<<<hb, 256, 0, c->stream>>>(n, hash, c->hist, P);
    SPH_CHECK_LAUNCH(c);
    radix_hist_scan_kernel<<<P, kRadix, 0, c->stream>>>(c->hist);
    SPH_CHECK_LAUNCH(c);

    // the last pass must land in (sorted_hash, perm): alternate backwards from there
    const uint32_t *kin = hash, *vin = nullptr;
    for (int p = 0; p < P; ++p) {
        const bool to_user = ((P - 1 - p) % 2) == 0;
        uint32_t *kout = to_user ? sorted_hash : c->alt_keys;
        uint32_t *vout = to_user ? perm : c->alt_vals;
        uint32_t *status = c->tile_status + (size_t)p * tiles * kRadix;
        if (p == 0)
            onesweep_kernel<true><<<(unsigned)tiles, kSortThreads, 0, c->stream>>>(
                n, kin, vin, kout, vout, c->hist + p * kRadix, status, c->tile_counter + p,
                p * kRadixBits);
        else
            onesweep_kernel<false><<<(unsigned)tiles, kSortThreads, 0, c->stream>>>(
                n, kin, vin, kout, vout, c->hist + p * kRadix, status, c->tile_counter + p,
                p * kRadixBits);
        SPH_CHECK_LAUNCH(c);
        kin = kout;
        vin = vout;
    }
    return SPH_OK;
}

// --------------------------------------------------------------------------- generic scan
// Single-pass exclusive prefix sum of uint32 with decoupled look-back (used for the compaction
// offsets of the boundary-particle list).  Totals must stay below 2^30.
__global__ void __launch_bounds__(kScanThreads)
scan_exclusive_kernel(int64_t n, const uint32_t *__restrict__ in, uint32_t *__restrict__ out,
                      uint32_t *status, uint32_t *ticket, uint32_t *total_out)
{
    __shared__ uint32_t s_warp[kScanThreads / 32];
    __shared__ uint32_t s_tile, s_excl;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    const int64_t base = (int64_t)tile * kScanTile + (int64_t)tid * kScanItems;
    uint32_t v[kScanItems];
    uint32_t sum = 0;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        v[i] = (base + i < n) ? in[base + i] : 0u;
        sum += v[i];
    }
    uint32_t inc = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t x = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += x;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    uint32_t add = 0, tile_total = 0;
#pragma unroll
    for (int i = 0; i < kScanThreads / 32; ++i) {
        const uint32_t w = s_warp[i];
        add += (i < warp) ? w : 0u;
        tile_total += w;
    }
    if (tid == 0) {
        st_volatile_u32(status + tile, (tile == 0 ? kFlagPrefix : kFlagAgg) | tile_total);
        uint32_t excl = 0;
        if (tile > 0) {
            int64_t t = (int64_t)tile - 1;
            while (true) {
                const uint32_t s = ld_volatile_u32(status + t);
                const uint32_t f = s & kFlagMask;
                if (f == 0) continue;
                excl += s & kValueMask;
                if (f == kFlagPrefix) break;
                --t;
            }
            st_volatile_u32(status + tile, kFlagPrefix | (excl + tile_total));
        }
        s_excl = excl;
        if ((int64_t)(tile + 1) * kScanTile >= n && total_out) *total_out = excl + tile_total;
    }
    __syncthreads();
    uint32_t run = s_excl + add + (inc - sum);
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        if (base + i < n) out[base + i] = run;
        run += v[i];
    }
}

int launch_scan_exclusive(sph_ctx *c, int64_t n, const uint32_t *in, uint32_t *out, uint32_t *total)
{
    if (n == 0) {
        if (total) SPH_CUDA_TRY(c, cudaMemsetAsync(total, 0, sizeof(uint32_t), c->stream));
        return SPH_OK;
    }
    const int64_t tiles = (n + kScanTile - 1) / kScanTile;
    uint32_t *ticket = c->tile_counter + kMaxPasses;
    SPH_CUDA_TRY(c, cudaMemsetAsync(ticket, 0, sizeof(uint32_t), c->stream));
    SPH_CUDA_TRY(c, cudaMemsetAsync(c->scan_status, 0, sizeof(uint32_t) * tiles, c->stream));
    scan_exclusive_kernel<<<(unsigned)tiles, kScanThreads, 0, c->stream>>>(n, in, out, c->scan_status,
                                                                          ticket, total);
    SPH_CHECK_LAUNCH(c);
    return SPH_OK;
}

}  // namespace sphb
