// Stage 2a: hand-written onesweep LSD radix sort on (hash, id)  (reading S5).
//
// One histogram kernel reads the keys once and builds the digit histograms of every pass (inside
// sph_step the bucket-hash pass counts them instead, hash_hist_kernel below, and launch_sort skips
// it).  Each pass is then ONE kernel: a tile of 6144 keys is ranked with warp-level match/popc
// (stable), the tile's per-digit counts are chained to the previous tiles with decoupled
// look-back (single 32-bit status word = 2 flag bits + 30-bit count, so no fence is needed), and
// keys/values are staged through shared memory so each digit's run leaves as one contiguous
// write.  Tiles take their index from an atomic ticket, which guarantees forward progress of the
// look-back chain; every tile also prefetches the keys / values of the tile one wave of resident
// CTAs ahead into the L2 (the passes are bound by the bytes a tile has in flight, not by DRAM
// bandwidth).  Values of the first pass are the implicit ids 0..n-1 (never read), and only
// the live key bits ceil(log2(cells)) are sorted.  Stability + ascending ids on input give the
// lexicographic (hash, id) order.
#include "sph_internal.cuh"

namespace sphb {

// --------------------------------------------------------------------------- histograms
// Digit counts of one 128-bit load (4 consecutive keys of one thread) for pass P.  Spatially
// coherent ids share their high digits: one atomic for the whole warp when all 128 keys agree,
// one per thread when its 4 keys agree, 4 otherwise.
template <int P>
__device__ __forceinline__ void hist_add4(uint32_t (*s_hist)[kRadix], const uint4 &v, int lane)
{
    const uint32_t d0 = (v.x >> (P * kRadixBits)) & (kRadix - 1), d1 = (v.y >> (P * kRadixBits)) & (kRadix - 1);
    const uint32_t d2 = (v.z >> (P * kRadixBits)) & (kRadix - 1), d3 = (v.w >> (P * kRadixBits)) & (kRadix - 1);
    if (P == 0) {  // the lowest digit changes every few keys
        // plain increments: with the digit runs aggregated per thread (1-4 predicated atomics of
        // 1..4) the kernel executed 20 % more instructions and took 82 instead of 72 us at 64 M
        atomicAdd(&s_hist[P][d0], 1u); atomicAdd(&s_hist[P][d1], 1u);
        atomicAdd(&s_hist[P][d2], 1u); atomicAdd(&s_hist[P][d3], 1u);
        return;
    }
    const bool same = (d0 == d1) & (d2 == d3) & (d0 == d2);
    int all_lanes = 0;
    __match_all_sync(0xffffffffu, same ? d0 : (0x100u + (uint32_t)lane), &all_lanes);
    if (all_lanes) {
        if (lane == 0) atomicAdd(&s_hist[P][d0], 128u);
    } else if (same) {
        atomicAdd(&s_hist[P][d0], 4u);
    } else {
        atomicAdd(&s_hist[P][d0], 1u); atomicAdd(&s_hist[P][d1], 1u);
        atomicAdd(&s_hist[P][d2], 1u); atomicAdd(&s_hist[P][d3], 1u);
    }
}


// Passes 1 .. NP-1 of one 128-bit load: spatially coherent ids share ALL their upper digits, so
// one match over the key bits above the lowest digit decides for every upper pass at once (one
// atomic per pass for the whole warp); anything else falls back to the per-pass aggregation.
template <int NP>
__device__ __forceinline__ void hist_upper(uint32_t (*s_hist)[kRadix], const uint4 &v, int lane)
{
    const uint32_t u = v.x >> kRadixBits;
    const bool same = (((v.x ^ v.y) | (v.x ^ v.z) | (v.x ^ v.w)) >> kRadixBits) == 0u;
    int all_lanes = 0;
    __match_all_sync(0xffffffffu, same ? u : (0xFF000000u + (uint32_t)lane), &all_lanes);
    if (all_lanes) {
        if (lane == 0) {
            atomicAdd(&s_hist[1][u & (kRadix - 1)], 128u);
            if (NP > 2) atomicAdd(&s_hist[2][(u >> kRadixBits) & (kRadix - 1)], 128u);
            if (NP > 3) atomicAdd(&s_hist[3][(u >> (2 * kRadixBits)) & (kRadix - 1)], 128u);
        }
    } else {
        hist_add4<1>(s_hist, v, lane);
        if (NP > 2) hist_add4<2>(s_hist, v, lane);
        if (NP > 3) hist_add4<3>(s_hist, v, lane);
    }
}

template <int NP>
__global__ void __launch_bounds__(256) radix_hist_kernel(int64_t n, const uint32_t *__restrict__ keys,
                                                         uint32_t *__restrict__ hist, uint32_t *__restrict__ status,
                                                         int64_t n_status, uint32_t *__restrict__ tickets, int n_tickets)
{
    __shared__ uint32_t s_hist[kMaxPasses][kRadix];
    // the look-back status words and tile tickets of the passes are cleared here (this kernel only
    // reads otherwise, the stores ride along): two memset launches less per sort
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_status; i += (int64_t)gridDim.x * blockDim.x)
        status[i] = 0u;
    if (blockIdx.x == 0 && threadIdx.x < n_tickets) tickets[threadIdx.x] = 0u;
    for (int i = threadIdx.x; i < kMaxPasses * kRadix; i += blockDim.x) (&s_hist[0][0])[i] = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31;
    // keys are only 4-byte aligned by contract (include/sph.h): a scalar head of up to 3 keys
    // brings the 128-bit loads onto a 16-byte boundary
    int64_t head = (int64_t)((16 - (reinterpret_cast<uintptr_t>(keys) & 15)) & 15) >> 2;
    if (head > n) head = n;
    if (blockIdx.x == 0 && threadIdx.x == 32)
        for (int64_t i = 0; i < head; ++i)
            for (int p = 0; p < NP; ++p) atomicAdd(&s_hist[p][(keys[i] >> (p * kRadixBits)) & (kRadix - 1)], 1u);
    keys += head;
    n -= head;
    const int64_t n4 = n >> 2;                       // whole 128-bit groups
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint4 *k4 = reinterpret_cast<const uint4 *>(keys);
    // main part: iterations in which every thread of the grid has data -- four loads in flight,
    // no bounds checks, no votes
    const int64_t full = n4 / (4 * stride);
    for (int64_t it = 0; it < full; ++it, g += 4 * stride) {
        const uint4 a = __ldcs(k4 + g), b = __ldcs(k4 + g + stride);
        const uint4 c = __ldcs(k4 + g + 2 * stride), d = __ldcs(k4 + g + 3 * stride);
        hist_add4<0>(s_hist, a, lane);
        if (NP > 1) hist_upper<NP>(s_hist, a, lane);
        hist_add4<0>(s_hist, b, lane);
        if (NP > 1) hist_upper<NP>(s_hist, b, lane);
        hist_add4<0>(s_hist, c, lane);
        if (NP > 1) hist_upper<NP>(s_hist, c, lane);
        hist_add4<0>(s_hist, d, lane);
        if (NP > 1) hist_upper<NP>(s_hist, d, lane);
    }
    // rest: block-uniform trip count (the warp-collective needs full warps), two loads in flight
    const int64_t rest = n4 - full * 4 * stride;
    const int64_t iters = (rest + 2 * stride - 1) / (2 * stride);
    for (int64_t it = 0; it < iters; ++it, g += 2 * stride) {
        const bool ok0 = g < n4, ok1 = g + stride < n4;
        uint4 a = make_uint4(0, 0, 0, 0), b = a;
        if (ok0) a = __ldcs(k4 + g);
        if (ok1) b = __ldcs(k4 + g + stride);
        // a lane without data joins the collectives with a value that never matches
        if (__all_sync(0xffffffffu, ok0)) {
            hist_add4<0>(s_hist, a, lane);
            if (NP > 1) hist_upper<NP>(s_hist, a, lane);
        } else if (ok0) {
            const uint32_t kk[4] = {a.x, a.y, a.z, a.w};
            for (int p = 0; p < NP; ++p)
                for (int j = 0; j < 4; ++j) atomicAdd(&s_hist[p][(kk[j] >> (p * kRadixBits)) & (kRadix - 1)], 1u);
        }
        if (__all_sync(0xffffffffu, ok1)) {
            hist_add4<0>(s_hist, b, lane);
            if (NP > 1) hist_upper<NP>(s_hist, b, lane);
        } else if (ok1) {
            const uint32_t kk[4] = {b.x, b.y, b.z, b.w};
            for (int p = 0; p < NP; ++p)
                for (int j = 0; j < 4; ++j) atomicAdd(&s_hist[p][(kk[j] >> (p * kRadixBits)) & (kRadix - 1)], 1u);
        }
    }
    // the ragged tail (n % 4 keys) goes to one thread
    if (blockIdx.x == 0 && threadIdx.x == 0)
        for (int64_t i = n4 << 2; i < n; ++i)
            for (int p = 0; p < NP; ++p) atomicAdd(&s_hist[p][(keys[i] >> (p * kRadixBits)) & (kRadix - 1)], 1u);
    __syncthreads();
    for (int i = threadIdx.x; i < NP * kRadix; i += blockDim.x) {
        uint32_t v = (&s_hist[0][0])[i];
        if (v) atomicAdd(hist + i, v);
    }
}

// Stage 1 + the histogram of stage 2 in ONE pass over the positions (inside sph_step): the bucket
// hash of PAPER.md:13 / :19 (readings S1-S3, the pinned fp32 sequence of bucket_hash) is written and
// counted while it is still in registers, so the sort reads its keys once less (4 of its 52 bytes
// per particle and a 60 us kernel at 64 M particles).  A warp takes 128 consecutive ids per
// iteration (four coalesced 16-byte loads per lane); the digit counts follow the histogram kernel
// above: plain increments for the lowest digit, one match for all upper digits.
template <int NP>
__global__ void __launch_bounds__(256) hash_hist_kernel(int64_t n, const float4 *__restrict__ posm,
                                                        uint32_t *__restrict__ hash, Grid g,
                                                        uint32_t *__restrict__ hist, uint32_t *__restrict__ status,
                                                        int64_t n_status, uint32_t *__restrict__ tickets, int n_tickets)
{
    __shared__ uint32_t s_hist[kMaxPasses][kRadix];
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_status; i += (int64_t)gridDim.x * blockDim.x)
        status[i] = 0u;
    if (blockIdx.x == 0 && threadIdx.x < n_tickets) tickets[threadIdx.x] = 0u;
    for (int i = threadIdx.x; i < kMaxPasses * kRadix; i += blockDim.x) (&s_hist[0][0])[i] = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t chunk = 256 * 4;                       // particles per block and iteration
    for (int64_t base = (int64_t)blockIdx.x * chunk; base < n; base += (int64_t)gridDim.x * chunk) {
        const int64_t i0 = base + warp * 128 + lane;
        {   // the warp's 16 lines of the next iteration go to the L2 while this one is processed
            const int64_t nb = base + (int64_t)gridDim.x * chunk + warp * 128 + lane * 8;
            if (lane < 16 && nb < n) asm volatile("prefetch.global.L2 [%0];" ::"l"(posm + nb));
        }
        if (base + chunk <= n) {                          // block-uniform: every lane has four particles
            const float4 p0 = __ldcs(posm + i0), p1 = __ldcs(posm + i0 + 32);
            const float4 p2 = __ldcs(posm + i0 + 64), p3 = __ldcs(posm + i0 + 96);
            uint4 v;
            v.x = bucket_hash(p0, g); v.y = bucket_hash(p1, g); v.z = bucket_hash(p2, g); v.w = bucket_hash(p3, g);
            hash[i0] = v.x; hash[i0 + 32] = v.y; hash[i0 + 64] = v.z; hash[i0 + 96] = v.w;
            hist_add4<0>(s_hist, v, lane);
            if (NP > 1) hist_upper<NP>(s_hist, v, lane);
        } else {
            for (int j = 0; j < 4; ++j) {
                const int64_t i = i0 + 32 * j;
                if (i < n) {
                    const uint32_t k = bucket_hash(__ldcs(posm + i), g);
                    hash[i] = k;
                    for (int p = 0; p < NP; ++p) atomicAdd(&s_hist[p][(k >> (p * kRadixBits)) & (kRadix - 1)], 1u);
                }
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < NP * kRadix; i += blockDim.x) {
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
constexpr int kSortWarps = kSortThreads / 32;
struct SortSmem {
    uint16_t warp_hist[kSortWarps][kRadix];   // per-warp digit counts -> exclusive over the warps (<= 8192)
    uint32_t keys[kSortTile];
    uint32_t vals[kSortTile];
    uint32_t digit_base[kRadix];              // start of the digit's run inside the tile
    uint32_t gbase[kRadix];                   // global position of that run minus digit_base
    uint32_t scan[kRadix / 32];
    uint32_t tile;
};

template <bool FIRST>
__global__ void __launch_bounds__(kSortThreads, 3)
onesweep_kernel(int64_t n, const uint32_t *__restrict__ keys_in, const uint32_t *__restrict__ vals_in,
                uint32_t *__restrict__ keys_out, uint32_t *__restrict__ vals_out,
                const uint32_t *__restrict__ hist_excl, uint32_t *status, uint32_t *ticket, int shift,
                uint32_t *__restrict__ inv_out /* optional: inv_out[value] = destination */, int pf_tiles)
{
    extern __shared__ __align__(16) unsigned char sort_smem_raw[];
    SortSmem &sm = *reinterpret_cast<SortSmem *>(sort_smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) sm.tile = atomicAdd(ticket, 1u);
#pragma unroll
    for (int i = tid; i < kSortWarps * kRadix / 2; i += kSortThreads)
        reinterpret_cast<uint32_t *>(&sm.warp_hist[0][0])[i] = 0;
    __syncthreads();
    const uint32_t tile = sm.tile;
    const int64_t tile_base = (int64_t)tile * kSortTile;
    const int tile_valid = (int)min((int64_t)kSortTile, n - tile_base);
    const int64_t chunk = tile_base + warp * (32 * kSortItems) + lane;
    // L2 prefetch of the tile this CTA slot will see next (tickets are taken in launch order, so
    // that is ~one wave of resident CTAs ahead): the passes are bound by the few bytes a tile has
    // in flight, not by DRAM bandwidth -- the next tile's key and value loads then hit the L2
    {
        constexpr int kLines = kSortTile * 4 / 128;               // 128-byte lines of a tile's keys
        const int64_t pf = tile_base + (int64_t)pf_tiles * kSortTile;
        if (tid < kLines && pf + (int64_t)tid * 32 < n) {
            asm volatile("prefetch.global.L2 [%0];" ::"l"(keys_in + pf + (int64_t)tid * 32));
            if (!FIRST) asm volatile("prefetch.global.L2 [%0];" ::"l"(vals_in + pf + (int64_t)tid * 32));
        }
    }

    // ---- load (warp-striped: item r of lane l = chunk[r*32 + l]) ----
    // (values are fetched later, straight into the staging buffer: 16 fewer live registers, which
    //  is what lets three 512-thread CTAs share an SM)
    uint32_t key[kSortItems];
#pragma unroll
    for (int r = 0; r < kSortItems; ++r) {
        const int64_t idx = chunk + r * 32;
        key[r] = idx < n ? __ldcs(keys_in + idx) : 0xFFFFFFFFu;
    }

    // ---- stable rank inside the warp ----
    uint32_t rank2[kSortItems / 2];   // two 16-bit ranks per register (rank < 512)
    const uint32_t lt = lanemask_lt();
#pragma unroll
    for (int r = 0; r < kSortItems; ++r) {
        const uint32_t d = (key[r] >> shift) & (kRadix - 1);
        // MATCH.ANY costs 8 cycles per DISTINCT value and scheduler (measured: 96 cycles at 12
        // values, 256 at 32).  The lowest digit of spatially coherent ids changes every few keys,
        // so the first pass would pay ~12 values per round -- but there the digits of a stripe
        // are almost always non-decreasing over the lanes, and then equal digits are adjacent:
        // the peer group is the run between two "head" lanes (two ballots, no match).
        uint32_t peers;
        if (FIRST) {
            const uint32_t dp = __shfl_up_sync(0xffffffffu, d, 1);
            const uint32_t heads = __ballot_sync(0xffffffffu, lane == 0 || d != dp);
            if (__ballot_sync(0xffffffffu, lane != 0 && d < dp) == 0u) {
                const uint32_t le = lt | (1u << lane);                          // lanes <= lane
                const uint32_t start = 31u - (uint32_t)__clz(heads & le);       // head of my run (bit 0 is set)
                const uint32_t above = heads & ~le;                            // heads at lanes > lane
                const uint32_t end_mask = above ? ((above & (0u - above)) - 1u) : 0xffffffffu;
                peers = end_mask & ~((1u << start) - 1u);
            } else {
                peers = __match_any_sync(0xffffffffu, d);
            }
        } else {
            peers = __match_any_sync(0xffffffffu, d);
        }
        const uint32_t before = __popc(peers & lt);
        uint32_t basev = 0;
        // the histogram is private to the warp: the lowest peer books the whole group with a plain
        // read-modify-write (shared-memory atomics with a return value measured slower)
        if (before == 0) {
            basev = sm.warp_hist[warp][d];
            sm.warp_hist[warp][d] = (uint16_t)(basev + (uint32_t)__popc(peers));
        }
        __syncwarp();
        basev = __shfl_sync(0xffffffffu, basev, __ffs(peers) - 1);
        if (r & 1) rank2[r >> 1] |= (basev + before) << 16; else rank2[r >> 1] = basev + before;
    }
    __syncthreads();

    // ---- per-digit work: thread d < 256 owns digit d ----
    const int d = tid;
    uint32_t my_total = 0, run = 0, inc = 0;
    if (d < kRadix) {
#pragma unroll
        for (int w = 0; w < kSortWarps; ++w) {
            const uint32_t c = sm.warp_hist[w][d];
            sm.warp_hist[w][d] = (uint16_t)run;
            run += c;
        }
        // padding keys (0xFFFFFFFF) sit at the very end of digit 255
        my_total = (d == kRadix - 1) ? run - (uint32_t)(kSortTile - tile_valid) : run;
        st_volatile_u32(status + (size_t)tile * kRadix + d, (tile == 0 ? kFlagPrefix : kFlagAgg) | my_total);
        // block exclusive scan of `run` over digits -> position of the digit's run in the tile
        inc = run;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t x = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += x;
        }
        if (lane == 31) sm.scan[warp] = inc;
    }
    __syncthreads();
    if (d < kRadix) {
        uint32_t add = 0;
#pragma unroll
        for (int i = 0; i < kRadix / 32; ++i) add += (i < warp) ? sm.scan[i] : 0u;
        sm.digit_base[d] = inc - run + add;
    }
    __syncthreads();

    // ---- scatter into the tile-local sorted order (needs no global offset yet: the look-back
    //      comes after it, which gives the preceding tiles time to publish their prefixes) ----
#pragma unroll
    for (int r = 0; r < kSortItems; ++r) {
        const uint32_t dg = (key[r] >> shift) & (kRadix - 1);
        const uint32_t pos = sm.digit_base[dg] + sm.warp_hist[warp][dg] + ((rank2[r >> 1] >> ((r & 1) * 16)) & 0xFFFFu);
        sm.keys[pos] = key[r];
        const int64_t idx = chunk + r * 32;
        sm.vals[pos] = FIRST ? (uint32_t)idx : (idx < n ? __ldcs(vals_in + idx) : 0u);
    }

    // ---- decoupled look-back over the previous tiles ----
    if (d < kRadix) {
        uint32_t excl = 0;
        if (tile > 0) {
            // kLook status words are requested at once (independent loads), then consumed in
            // order: a thread-serial walk would cost one L2 round trip per preceding tile
            constexpr int kLook = 4;   // measured at 64 M keys: 1 -> 1.08 ms, 2 -> 0.99, 4 -> 0.966, 8 -> 0.974, 16 -> 1.02; with the L2 prefetch: 2 -> 0.905, 4 -> 0.882, 8 -> 0.890; batches that grow to 16 after a fully consumed batch: 0.937 (the walk mostly polls ONE unpublished word: 10.4 round trips per tile and warp)
            int64_t t = (int64_t)tile - 1;
            bool done = false;
            while (!done) {
                uint32_t sw[kLook];
#pragma unroll
                for (int j = 0; j < kLook; ++j)
                    sw[j] = (t - j >= 0) ? ld_volatile_u32(status + (size_t)(t - j) * kRadix + d) : kFlagPrefix;
                int used = 0;
#pragma unroll
                for (int j = 0; j < kLook; ++j) {
                    const uint32_t f = sw[j] & kFlagMask;
                    if (!done && used == j && f != 0) {
                        excl += sw[j] & kValueMask;
                        used = j + 1;
                        if (f == kFlagPrefix) done = true;
                    }
                }
                t -= used;  // an unpublished word stops the batch; it is polled again
            }
            st_volatile_u32(status + (size_t)tile * kRadix + d, kFlagPrefix | (excl + my_total));
        }
        sm.gbase[d] = hist_excl[d] + excl - sm.digit_base[d];
    }
    __syncthreads();

    // ---- each digit run leaves as one contiguous stretch ----
#pragma unroll
    for (int k = 0; k < kSortItems; ++k) {
        const int p = tid + k * kSortThreads;
        if (p < tile_valid) {
            const uint32_t kk = sm.keys[p];
            const uint32_t dg = (kk >> shift) & (kRadix - 1);
            const uint32_t dst = sm.gbase[dg] + (uint32_t)p;
            const uint32_t vv = sm.vals[p];
            keys_out[dst] = kk;
            vals_out[dst] = vv;
            if (inv_out) inv_out[vv] = dst;
        }
    }
}

// (moved up: used by the sort and by the partition)
// the opt-in to > 48 KB of dynamic shared memory is per device: once per ctx (a ctx is bound to
// the device that was current at sph_create)
static int sort_smem_opt_in(sph_ctx *c)
{
    if (c->attr_sort) return SPH_OK;
    SPH_CUDA_TRY(c, cudaFuncSetAttribute(onesweep_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)sizeof(SortSmem)));
    SPH_CUDA_TRY(c, cudaFuncSetAttribute(onesweep_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)sizeof(SortSmem)));
    c->attr_sort = true;
    return SPH_OK;
}

__global__ void __launch_bounds__(256) iota_copy_kernel(int64_t n, const uint32_t *__restrict__ hash,
                                                        uint32_t *__restrict__ sorted_hash,
                                                        uint32_t *__restrict__ perm)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { sorted_hash[i] = hash[i]; perm[i] = (uint32_t)i; }
}

int launch_hash_hist(sph_ctx *c, int64_t n, const float *posm, uint32_t *hash)
{
    c->hist_for = nullptr;
    const int P = c->n_passes;
    if (n == 0 || P == 0) return launch_hash(c, n, posm, hash);
    const int64_t tiles = (n + kSortTile - 1) / kSortTile;
    const int64_t n_status = (int64_t)P * tiles * kRadix;
    SPH_CUDA_TRY(c, cudaMemsetAsync(c->hist, 0, sizeof(uint32_t) * kMaxPasses * kRadix, c->stream));
    int hb = (int)min((int64_t)c->num_sms * 8, (n + 1023) / 1024);
    if (hb < 1) hb = 1;
    const float4 *p4 = reinterpret_cast<const float4 *>(posm);
    switch (P) {
    case 1: hash_hist_kernel<1><<<hb, 256, 0, c->stream>>>(n, p4, hash, c->grid, c->hist, c->tile_status, n_status, c->tile_counter, kMaxPasses); break;
    case 2: hash_hist_kernel<2><<<hb, 256, 0, c->stream>>>(n, p4, hash, c->grid, c->hist, c->tile_status, n_status, c->tile_counter, kMaxPasses); break;
    case 3: hash_hist_kernel<3><<<hb, 256, 0, c->stream>>>(n, p4, hash, c->grid, c->hist, c->tile_status, n_status, c->tile_counter, kMaxPasses); break;
    default: hash_hist_kernel<4><<<hb, 256, 0, c->stream>>>(n, p4, hash, c->grid, c->hist, c->tile_status, n_status, c->tile_counter, kMaxPasses); break;
    }
    SPH_CHECK_LAUNCH(c);
    radix_hist_scan_kernel<<<P, kRadix, 0, c->stream>>>(c->hist);
    SPH_CHECK_LAUNCH(c);
    c->hist_for = hash;
    return SPH_OK;
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
    const bool have_hist = c->hist_for == hash;   // sph_step: counted by the fused hash kernel
    c->hist_for = nullptr;
    if (!have_hist) {
    SPH_CUDA_TRY(c, cudaMemsetAsync(c->hist, 0, sizeof(uint32_t) * kMaxPasses * kRadix, c->stream));
    const int64_t n_status = (int64_t)P * tiles * kRadix;
    int hb = (int)min((int64_t)c->num_sms * 8, (n + 1023) / 1024);
    if (hb < 1) hb = 1;
    switch (P) {
    case 1: radix_hist_kernel<1><<<hb, 256, 0, c->stream>>>(n, hash, c->hist, c->tile_status, n_status, c->tile_counter, kMaxPasses); break;
    case 2: radix_hist_kernel<2><<<hb, 256, 0, c->stream>>>(n, hash, c->hist, c->tile_status, n_status, c->tile_counter, kMaxPasses); break;
    case 3: radix_hist_kernel<3><<<hb, 256, 0, c->stream>>>(n, hash, c->hist, c->tile_status, n_status, c->tile_counter, kMaxPasses); break;
    default: radix_hist_kernel<4><<<hb, 256, 0, c->stream>>>(n, hash, c->hist, c->tile_status, n_status, c->tile_counter, kMaxPasses); break;
    }
    SPH_CHECK_LAUNCH(c);
    radix_hist_scan_kernel<<<P, kRadix, 0, c->stream>>>(c->hist);
    SPH_CHECK_LAUNCH(c);
    }

    {
        int rc = sort_smem_opt_in(c);
        if (rc != SPH_OK) return rc;
    }
    // the last pass must land in (sorted_hash, perm): alternate backwards from there
    const int pf_tiles = c->num_sms * 3;   // one wave of resident CTAs ahead (measured at 64 M keys: 0 -> 0.911 ms, 1 wave 0.894, 2 waves 0.946, 4 waves 1.005; without the prefetch 0.966)
    const uint32_t *kin = hash, *vin = nullptr;
    for (int p = 0; p < P; ++p) {
        const bool to_user = ((P - 1 - p) % 2) == 0;
        uint32_t *kout = to_user ? sorted_hash : c->alt_keys;
        uint32_t *vout = to_user ? perm : c->alt_vals;
        uint32_t *status = c->tile_status + (size_t)p * tiles * kRadix;
        if (p == 0)
            onesweep_kernel<true><<<(unsigned)tiles, kSortThreads, sizeof(SortSmem), c->stream>>>(
                n, kin, vin, kout, vout, c->hist + p * kRadix, status, c->tile_counter + p,
                p * kRadixBits, nullptr, pf_tiles);
        else
            onesweep_kernel<false><<<(unsigned)tiles, kSortThreads, sizeof(SortSmem), c->stream>>>(
                n, kin, vin, kout, vout, c->hist + p * kRadix, status, c->tile_counter + p,
                p * kRadixBits, nullptr, pf_tiles);
        SPH_CHECK_LAUNCH(c);
        kin = kout;
        vin = vout;
    }
    return SPH_OK;
}

// --------------------------------------------------------------------------- stable partition
// NEXT-1 (per-owner send buffers): cut the boundary list into one segment per owner.  A stable
// partition on a label < 256 is exactly ONE onesweep pass (digit = the label) with the list
// entries as values; the exclusive digit histogram is the table of segment offsets.
__global__ void __launch_bounds__(256)
gather_label_kernel(int64_t m, const uint32_t *__restrict__ ids, const int32_t *__restrict__ label,
                    uint32_t *__restrict__ key)
{
    // four independent id -> label chains per thread (a single dependent chain per thread left the
    // kernel latency-bound: 294 us at 64 M entries with 15 % of the issue slots used)
    const int64_t k0 = ((int64_t)blockIdx.x * blockDim.x) * 4 + threadIdx.x;
    uint32_t id[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) { const int64_t k = k0 + j * 256; id[j] = k < m ? __ldcs(ids + k) : 0u; }
    uint32_t lb[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) { const int64_t k = k0 + j * 256; lb[j] = k < m ? (uint32_t)__ldg(label + id[j]) : 0u; }
#pragma unroll
    for (int j = 0; j < 4; ++j) { const int64_t k = k0 + j * 256; if (k < m) key[k] = lb[j] & (kRadix - 1); }
}

__global__ void segment_offsets_kernel(const uint32_t *__restrict__ hist_excl, int n_labels, uint32_t m,
                                       uint32_t *__restrict__ offsets)
{
    const int g = threadIdx.x;
    if (g < n_labels) offsets[g] = hist_excl[g];
    if (g == n_labels) offsets[g] = m;
}

// Stable partition of the implicit indices 0..m-1 by the keys in c->alt_keys (< 256): offsets
// [n_labels + 1] = segment starts, *order = the indices in partition order (ctx scratch), dest
// (optional) = destination of every index (the inverse map).
int launch_partition_keys(sph_ctx *c, int64_t m, int n_labels, uint32_t *offsets, uint32_t *dest, uint32_t **order)
{
    uint32_t *key = c->alt_keys, *key_out = c->alt_vals, *val_out = c->s_comm_hash;  // scratch (stream-ordered)
    c->hist_for = nullptr;   // the histogram scratch is reused below
    if (order) *order = val_out;
    if (m == 0) {
        SPH_CUDA_TRY(c, cudaMemsetAsync(offsets, 0, sizeof(uint32_t) * (n_labels + 1), c->stream));
        return SPH_OK;
    }
    const int64_t tiles = (m + kSortTile - 1) / kSortTile;
    SPH_CUDA_TRY(c, cudaMemsetAsync(c->hist, 0, sizeof(uint32_t) * kRadix, c->stream));
    int hb = (int)min((int64_t)c->num_sms * 8, (m + 1023) / 1024);
    if (hb < 1) hb = 1;
    radix_hist_kernel<1><<<hb, 256, 0, c->stream>>>(m, key, c->hist, c->tile_status, tiles * kRadix, c->tile_counter, 1);
    SPH_CHECK_LAUNCH(c);
    radix_hist_scan_kernel<<<1, kRadix, 0, c->stream>>>(c->hist);
    SPH_CHECK_LAUNCH(c);
    segment_offsets_kernel<<<1, 512, 0, c->stream>>>(c->hist, n_labels, (uint32_t)m, offsets);
    SPH_CHECK_LAUNCH(c);
    {
        int rc = sort_smem_opt_in(c);
        if (rc != SPH_OK) return rc;
    }
    // values = the implicit indices 0..m-1 (FIRST), so inv_out[k] is index k's destination
    onesweep_kernel<true><<<(unsigned)tiles, kSortThreads, sizeof(SortSmem), c->stream>>>(
        m, key, nullptr, key_out, val_out, c->hist, c->tile_status, c->tile_counter, 0, dest, c->num_sms * 3);
    SPH_CHECK_LAUNCH(c);
    return SPH_OK;
}

int launch_partition_by_label(sph_ctx *c, int64_t m, const uint32_t *ids, const int32_t *label, int n_labels,
                              uint32_t *offsets, uint32_t *dest)
{
    // dest[k] = position of list entry k in the label-segmented order (a SCATTER map: the caller
    // then reads the list and the records in list order, which is sector-friendly, and writes
    // n_labels sequential streams -- the gather form re-read every sector once per label)
    if (m > 0) {
        gather_label_kernel<<<div_up(m, 1024), 256, 0, c->stream>>>(m, ids, label, c->alt_keys);
        SPH_CHECK_LAUNCH(c);
    }
    return launch_partition_keys(c, m, n_labels, offsets, dest, nullptr);
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
    static_assert(kScanItems % 4 == 0, "128-bit loads and stores");
    const bool vec = base + kScanItems <= n &&
                     ((reinterpret_cast<uintptr_t>(in) | reinterpret_cast<uintptr_t>(out)) & 15) == 0;
    if (vec) {
#pragma unroll
        for (int q = 0; q < kScanItems / 4; ++q) {
            const uint4 x = __ldcs(reinterpret_cast<const uint4 *>(in + base) + q);
            v[4 * q] = x.x; v[4 * q + 1] = x.y; v[4 * q + 2] = x.z; v[4 * q + 3] = x.w;
        }
#pragma unroll
        for (int i = 0; i < kScanItems; ++i) sum += v[i];
    } else {
#pragma unroll
        for (int i = 0; i < kScanItems; ++i) {
            v[i] = (base + i < n) ? in[base + i] : 0u;
            sum += v[i];
        }
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
    if (warp == 0) {
        // warp-parallel decoupled look-back: lane l inspects tile t0 - l; the window moves back by
        // 32 tiles until it holds an inclusive prefix with every tile after it published
        if (lane == 0) st_volatile_u32(status + tile, (tile == 0 ? kFlagPrefix : kFlagAgg) | tile_total);
        uint32_t excl = 0;
        if (tile > 0) {
            int64_t t0 = (int64_t)tile - 1;
            while (true) {
                const int64_t t = t0 - lane;
                const uint32_t s = t >= 0 ? ld_volatile_u32(status + t) : kFlagPrefix;  // nothing before tile 0
                const uint32_t f = s & kFlagMask;
                const uint32_t pref = __ballot_sync(0xffffffffu, f == kFlagPrefix);
                const uint32_t unpub = __ballot_sync(0xffffffffu, f == 0);
                const int fp = pref ? __ffs(pref) - 1 : 31;          // last lane that counts
                const uint32_t need = 0xffffffffu >> (31 - fp);      // lanes 0 .. fp
                if (unpub & need) continue;                          // not all published yet
                excl += __reduce_add_sync(0xffffffffu, lane <= fp ? (s & kValueMask) : 0u);
                if (pref) break;
                t0 -= 32;
            }
            if (lane == 0) st_volatile_u32(status + tile, kFlagPrefix | (excl + tile_total));
        }
        if (lane == 0) {
            s_excl = excl;
            if ((int64_t)(tile + 1) * kScanTile >= n && total_out) *total_out = excl + tile_total;
        }
    }
    __syncthreads();
    uint32_t run = s_excl + add + (inc - sum);
    if (vec) {
        uint32_t o[kScanItems];
#pragma unroll
        for (int i = 0; i < kScanItems; ++i) { o[i] = run; run += v[i]; }
#pragma unroll
        for (int q = 0; q < kScanItems / 4; ++q)
            __stcs(reinterpret_cast<uint4 *>(out + base) + q, make_uint4(o[4 * q], o[4 * q + 1], o[4 * q + 2], o[4 * q + 3]));
    } else {
#pragma unroll
        for (int i = 0; i < kScanItems; ++i) {
            if (base + i < n) out[base + i] = run;
            run += v[i];
        }
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
