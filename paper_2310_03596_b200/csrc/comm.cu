// Stage 3: communication hash and the MGPU boundary-particle list (step c,
// PAPER.md:22).
//
// The paper's test "particles from other GPUs are present in the particle's bucket or in the
// surrounding buckets" is a per-BUCKET property (I5: the particle itself is in its
// own stencil, so "a different owner exists" == "the stencil holds >= 2 distinct owners").
// So: (1) one owner bitmask per bucket (warp-aggregated atomicOr), (2) per bucket the OR over
// the 27-bucket stencil, flag = popcount >= 2, (3) the paper's "sort on that key" yields
// exactly the stable compaction of the already (hash, id)-sorted array (I6): an
// exclusive scan of the flagged buckets' sizes gives every flagged bucket its slot, and its
// particles copy perm[k] there.  Everything is streaming / HBM-bound.
#include "sph_internal.cuh"

namespace sphb {

constexpr int kMaskItems = 8;  // sorted particles per thread

// The array is sorted by hash, so the particles of a bucket are a contiguous run: every thread
// ORs the owner bits of its 8 consecutive particles run by run and issues one atomicOr per run
// end (about 1.4 per thread at 17.6 particles per bucket) -- no warp-wide match needed.
__global__ void __launch_bounds__(256)
owner_mask_kernel(int64_t n, const uint32_t *__restrict__ sorted_hash,
                  const int32_t *__restrict__ sorted_owner, uint32_t *__restrict__ cell_mask)
{
    const int64_t k0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * kMaskItems;
    if (k0 >= n) return;
    uint32_t h[kMaskItems];
    int32_t o[kMaskItems];
    const bool vec = k0 + kMaskItems <= n && ((reinterpret_cast<uintptr_t>(sorted_hash) |
                                               reinterpret_cast<uintptr_t>(sorted_owner)) & 15) == 0;
    if (vec) {
        const uint4 a = __ldcs(reinterpret_cast<const uint4 *>(sorted_hash + k0));
        const uint4 b = __ldcs(reinterpret_cast<const uint4 *>(sorted_hash + k0) + 1);
        const int4 c = __ldcs(reinterpret_cast<const int4 *>(sorted_owner + k0));
        const int4 d = __ldcs(reinterpret_cast<const int4 *>(sorted_owner + k0) + 1);
        h[0] = a.x; h[1] = a.y; h[2] = a.z; h[3] = a.w; h[4] = b.x; h[5] = b.y; h[6] = b.z; h[7] = b.w;
        o[0] = c.x; o[1] = c.y; o[2] = c.z; o[3] = c.w; o[4] = d.x; o[5] = d.y; o[6] = d.z; o[7] = d.w;
    } else {
#pragma unroll
        for (int j = 0; j < kMaskItems; ++j) {
            const bool ok = k0 + j < n;
            h[j] = ok ? sorted_hash[k0 + j] : 0xFFFFFFFFu;
            o[j] = ok ? sorted_owner[k0 + j] : 0;
        }
    }
    uint32_t cur = h[0], m = 1u << (o[0] & 31);
#pragma unroll
    for (int j = 1; j < kMaskItems; ++j) {
        if (h[j] != cur) {
            atomicOr(cell_mask + cur, m);
            cur = h[j];
            m = 0u;
        }
        if (cur != 0xFFFFFFFFu) m |= 1u << (o[j] & 31);
    }
    if (cur != 0xFFFFFFFFu) atomicOr(cell_mask + cur, m);
}

// One thread per 4 consecutive buckets of a grid row: the 9 stencil rows are read once as 6 masks
// each (54 loads for 4 buckets instead of 108) and OR-ed with a sliding window.
constexpr int kFlagCells = 4;

// kMaskOut = false: flag_count[c] = flagged particle count of bucket c (stage 3);
// kMaskOut = true:  flag_count[c] = the stencil's owner mask itself (per-destination lists, NEXT-1).
template <bool kMaskOut>
__global__ void __launch_bounds__(256)
stencil_flag_kernel(Grid g, const uint32_t *__restrict__ cell_mask, const uint32_t *__restrict__ cs,
                    const uint32_t *__restrict__ ce, uint32_t *__restrict__ flag_count)
{
    const int groups_x = (g.nx + kFlagCells - 1) / kFlagCells;
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (int64_t)groups_x * g.ny * g.nz) return;
    const int gx = (int)(t % groups_x), cy = (int)((t / groups_x) % g.ny), cz = (int)(t / ((int64_t)groups_x * g.ny));
    const int x0 = gx * kFlagCells;
    uint32_t col[kFlagCells + 2];   // OR over the 9 rows of the masks at x0 - 1 .. x0 + kFlagCells
#pragma unroll
    for (int i = 0; i < kFlagCells + 2; ++i) col[i] = 0u;
#pragma unroll
    for (int dz = -1; dz <= 1; ++dz) {
        const int z = cz + dz;
        if (z < 0 || z >= g.nz) continue;
#pragma unroll
        for (int dy = -1; dy <= 1; ++dy) {
            const int y = cy + dy;
            if (y < 0 || y >= g.ny) continue;
            const uint32_t row = (uint32_t)g.nx * ((uint32_t)y + (uint32_t)g.ny * (uint32_t)z);
#pragma unroll
            for (int i = 0; i < kFlagCells + 2; ++i) {
                const int x = x0 - 1 + i;
                if (x >= 0 && x < g.nx) col[i] |= __ldg(cell_mask + row + x);
            }
        }
    }
    const uint32_t row0 = (uint32_t)g.nx * ((uint32_t)cy + (uint32_t)g.ny * (uint32_t)cz);
#pragma unroll
    for (int i = 0; i < kFlagCells; ++i) {
        const int x = x0 + i;
        if (x >= g.nx) break;
        const uint32_t m = col[i] | col[i + 1] | col[i + 2];
        const uint32_t c = row0 + (uint32_t)x;
        if (kMaskOut) {
            flag_count[c] = m;
        } else {
            // an empty bucket contributes no particles whatever its stencil holds
            flag_count[c] = (__popc(m) >= 2) ? (ce[c] - cs[c]) : 0u;
        }
    }
}

constexpr int kCompItems = 8;  // sorted particles per thread (two 128-bit loads per array in flight)

__global__ void __launch_bounds__(256)
comm_hash_compact_kernel(int64_t n, const uint32_t *__restrict__ sorted_hash,
                         const int32_t *__restrict__ sorted_owner, const uint32_t *__restrict__ perm,
                         const uint32_t *__restrict__ cs, const uint32_t *__restrict__ flag_count,
                         const uint32_t *__restrict__ cell_offset, uint32_t *__restrict__ comm_hash,
                         uint32_t *__restrict__ boundary_ids, uint32_t *__restrict__ owner_counts,
                         int n_owners)
{
    __shared__ uint32_t s_cnt[SPH_MAX_OWNERS];
    if (threadIdx.x < SPH_MAX_OWNERS) s_cnt[threadIdx.x] = 0;
    __syncthreads();
    const int64_t k0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * kCompItems;
    uint32_t h[kCompItems], id[kCompItems];
    int32_t o[kCompItems];
    const bool full = k0 + kCompItems <= n;
    const bool vec = full && ((reinterpret_cast<uintptr_t>(sorted_hash) | reinterpret_cast<uintptr_t>(sorted_owner) |
                               reinterpret_cast<uintptr_t>(perm) | reinterpret_cast<uintptr_t>(comm_hash)) & 15) == 0;
    if (vec) {
#pragma unroll
        for (int v = 0; v < kCompItems / 4; ++v) {
            const uint4 a = __ldcs(reinterpret_cast<const uint4 *>(sorted_hash + k0) + v);
            const uint4 b = __ldcs(reinterpret_cast<const uint4 *>(perm + k0) + v);
            const int4 c = __ldcs(reinterpret_cast<const int4 *>(sorted_owner + k0) + v);
            h[4 * v] = a.x; h[4 * v + 1] = a.y; h[4 * v + 2] = a.z; h[4 * v + 3] = a.w;
            id[4 * v] = b.x; id[4 * v + 1] = b.y; id[4 * v + 2] = b.z; id[4 * v + 3] = b.w;
            o[4 * v] = c.x; o[4 * v + 1] = c.y; o[4 * v + 2] = c.z; o[4 * v + 3] = c.w;
        }
    } else {
#pragma unroll
        for (int j = 0; j < kCompItems; ++j) {
            const bool ok = k0 + j < n;
            h[j] = ok ? sorted_hash[k0 + j] : 0xFFFFFFFFu;
            id[j] = ok ? perm[k0 + j] : 0u;
            o[j] = ok ? sorted_owner[k0 + j] : 0;
        }
    }
    // bucket records of the first and the last bucket of the thread are requested up front
    // (independent loads); buckets in between (rare: 8 particles span 1-2 buckets) on demand
    const uint32_t hf = h[0], hl = h[kCompItems - 1];
    uint32_t fc_f = 0, off_f = 0, cs_f = 0, fc_l = 0, off_l = 0, cs_l = 0;
    if (hf != 0xFFFFFFFFu) { fc_f = __ldg(flag_count + hf); off_f = __ldg(cell_offset + hf); cs_f = __ldg(cs + hf); }
    if (hl != 0xFFFFFFFFu) { fc_l = __ldg(flag_count + hl); off_l = __ldg(cell_offset + hl); cs_l = __ldg(cs + hl); }
    uint32_t ch[kCompItems], dst[kCompItems];
    uint32_t cur = 0xFFFFFFFFu, delta = 0u;   // delta = cell_offset - cell_start of a flagged bucket
    bool flagged = false;
    uint32_t my_owner = 0xFFu, my_cnt = 0u;   // flagged particles of this thread with owner my_owner
#pragma unroll
    for (int j = 0; j < kCompItems; ++j) {
        if (h[j] != cur) {
            cur = h[j];
            flagged = false;
            if (cur != 0xFFFFFFFFu) {
                uint32_t fc, of, c0;
                if (cur == hf) { fc = fc_f; of = off_f; c0 = cs_f; }
                else if (cur == hl) { fc = fc_l; of = off_l; c0 = cs_l; }
                else { fc = __ldg(flag_count + cur); of = __ldg(cell_offset + cur); c0 = __ldg(cs + cur); }
                flagged = fc != 0u;
                delta = of - c0;
            }
        }
        ch[j] = flagged ? cur : SPH_GARBAGE_HASH;
        dst[j] = flagged ? delta + (uint32_t)(k0 + j) : 0xFFFFFFFFu;
        if (flagged) {
            const uint32_t oo = (uint32_t)o[j] & 31u;
            if (my_cnt == 0u) my_owner = oo;
            if (oo == my_owner) ++my_cnt; else atomicAdd(&s_cnt[oo], 1u);
        }
    }
    // boundary ids: 128-bit stores where 4 consecutive slots are flagged, contiguous and aligned
#pragma unroll
    for (int v = 0; v < kCompItems / 4; ++v) {
        const uint32_t d0 = dst[4 * v];
        const bool run4 = d0 != 0xFFFFFFFFu && (d0 & 3u) == 0u && dst[4 * v + 1] == d0 + 1u &&
                          dst[4 * v + 2] == d0 + 2u && dst[4 * v + 3] == d0 + 3u &&
                          (reinterpret_cast<uintptr_t>(boundary_ids) & 15) == 0;
        if (run4) {
            __stcs(reinterpret_cast<uint4 *>(boundary_ids + d0),
                   make_uint4(id[4 * v], id[4 * v + 1], id[4 * v + 2], id[4 * v + 3]));
        } else {
#pragma unroll
            for (int j = 4 * v; j < 4 * v + 4; ++j)
                if (dst[j] != 0xFFFFFFFFu) boundary_ids[dst[j]] = id[j];
        }
    }
    if (vec) {
#pragma unroll
        for (int v = 0; v < kCompItems / 4; ++v)
            __stcs(reinterpret_cast<uint4 *>(comm_hash + k0) + v,
                   make_uint4(ch[4 * v], ch[4 * v + 1], ch[4 * v + 2], ch[4 * v + 3]));
    } else {
#pragma unroll
        for (int j = 0; j < kCompItems; ++j)
            if (k0 + j < n) comm_hash[k0 + j] = ch[j];
    }
    // owner counts: one atomic for the warp when every lane saw the same single owner (slab-like
    // labels), per-lane shared-memory atomics otherwise
    const uint32_t o0 = __shfl_sync(0xffffffffu, my_owner, 0);
    if (__all_sync(0xffffffffu, my_owner == o0)) {
        const uint32_t tot = __reduce_add_sync(0xffffffffu, my_cnt);
        if ((threadIdx.x & 31) == 0 && tot) atomicAdd(&s_cnt[o0 & 31u], tot);
    } else if (my_cnt) {
        atomicAdd(&s_cnt[my_owner], my_cnt);
    }
    __syncthreads();
    if (threadIdx.x < n_owners && s_cnt[threadIdx.x]) atomicAdd(owner_counts + threadIdx.x, s_cnt[threadIdx.x]);
}

int launch_comm_hash(sph_ctx *c, int64_t n, const uint32_t *sorted_hash, const int32_t *sorted_owner,
                     const uint32_t *perm, const uint32_t *cs, const uint32_t *ce,
                     uint32_t *comm_hash, uint32_t *boundary_ids, uint32_t *boundary_count,
                     uint32_t *owner_counts)
{
    const uint32_t cells = c->grid.n_cells;
    SPH_CUDA_TRY(c, cudaMemsetAsync(owner_counts, 0, sizeof(uint32_t) * c->params.n_owners, c->stream));
    if (n == 0) {
        SPH_CUDA_TRY(c, cudaMemsetAsync(boundary_count, 0, sizeof(uint32_t), c->stream));
        return SPH_OK;
    }
    SPH_CUDA_TRY(c, cudaMemsetAsync(c->cell_mask, 0, sizeof(uint32_t) * cells, c->stream));
    owner_mask_kernel<<<div_up(div_up(n, kMaskItems), 256), 256, 0, c->stream>>>(n, sorted_hash, sorted_owner, c->cell_mask);
    SPH_CHECK_LAUNCH(c);
    {
        const int64_t groups = (int64_t)((c->grid.nx + kFlagCells - 1) / kFlagCells) * c->grid.ny * c->grid.nz;
        stencil_flag_kernel<false><<<div_up(groups, 256), 256, 0, c->stream>>>(c->grid, c->cell_mask, cs, ce,
                                                                               c->cell_flag_count);
    }
    SPH_CHECK_LAUNCH(c);
    int rc = launch_scan_exclusive(c, cells, c->cell_flag_count, c->cell_offset, boundary_count);
    if (rc != SPH_OK) return rc;
    comm_hash_compact_kernel<<<div_up(div_up(n, kCompItems), 256), 256, 0, c->stream>>>(
        n, sorted_hash, sorted_owner, perm, cs, c->cell_flag_count, c->cell_offset, comm_hash,
        boundary_ids, owner_counts, c->params.n_owners);
    SPH_CHECK_LAUNCH(c);
    return SPH_OK;
}

// ---- NEXT-1, second half: per-DESTINATION send lists (PAPER.md:23 step d; reading D1) --------
// Particle k goes to destination g iff g != owner_k and bit g is set in the owner mask of the
// 27-bucket stencil of k's bucket -- the mask stencil_flag_kernel ORs together anyway.  List g
// holds the ids of its particles in sorted order, so the whole product is a stable multi-way
// split in which one particle may enter several lists:
//   pass 1  per tile of 256 sorted particles, the number of entries for each destination
//           (warp ballots), stored destination-major: counts[g * tiles + tile];
//   scan    one exclusive scan over that array gives every (destination, tile) its first slot,
//           the lists back to back by ascending g;
//   pass 2  the same ballots again give each entry its rank inside the tile.
constexpr int kDestThreads = 256;

__device__ __forceinline__ uint32_t dest_bits(int64_t k, int64_t n, const uint32_t *__restrict__ sorted_hash,
                                              const int32_t *__restrict__ sorted_owner,
                                              const uint32_t *__restrict__ stencil_mask)
{
    if (k >= n) return 0u;
    return __ldg(stencil_mask + sorted_hash[k]) & ~(1u << (sorted_owner[k] & 31));
}

__global__ void __launch_bounds__(kDestThreads)
dest_count_kernel(int64_t n, const uint32_t *__restrict__ sorted_hash, const int32_t *__restrict__ sorted_owner,
                  const uint32_t *__restrict__ stencil_mask, uint32_t *__restrict__ counts, uint32_t tiles,
                  int n_owners)
{
    __shared__ uint32_t s_cnt[kDestThreads / 32][SPH_MAX_OWNERS];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t k = (int64_t)blockIdx.x * kDestThreads + threadIdx.x;
    const uint32_t bits = dest_bits(k, n, sorted_hash, sorted_owner, stencil_mask);
    uint32_t mine = 0u;   // lane g keeps the warp's count for destination g
    uint32_t any = __reduce_or_sync(0xffffffffu, bits);
    while (any) {
        const int g = __ffs(any) - 1;
        any &= any - 1;
        const uint32_t votes = __ballot_sync(0xffffffffu, (bits >> g) & 1u);
        if (lane == g) mine = __popc(votes);
    }
    s_cnt[warp][lane] = mine;
    __syncthreads();
    if (threadIdx.x < n_owners) {
        uint32_t tot = 0;
#pragma unroll
        for (int w = 0; w < kDestThreads / 32; ++w) tot += s_cnt[w][threadIdx.x];
        counts[(size_t)threadIdx.x * tiles + blockIdx.x] = tot;
    }
}

__global__ void __launch_bounds__(kDestThreads)
dest_scatter_kernel(int64_t n, const uint32_t *__restrict__ sorted_hash, const int32_t *__restrict__ sorted_owner,
                    const uint32_t *__restrict__ perm, const uint32_t *__restrict__ stencil_mask,
                    const uint32_t *__restrict__ offsets, uint32_t tiles, int n_owners,
                    uint32_t *__restrict__ dest_offsets, uint32_t *__restrict__ dest_ids, uint32_t cap)
{
    __shared__ uint32_t s_cnt[kDestThreads / 32][SPH_MAX_OWNERS];
    __shared__ uint32_t s_base[kDestThreads / 32][SPH_MAX_OWNERS];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t k = (int64_t)blockIdx.x * kDestThreads + threadIdx.x;
    const uint32_t bits = dest_bits(k, n, sorted_hash, sorted_owner, stencil_mask);
    const uint32_t id = k < n ? perm[k] : 0u;
    const uint32_t warp_any = __reduce_or_sync(0xffffffffu, bits);
    uint32_t mine = 0u;
    for (uint32_t any = warp_any; any;) {
        const int g = __ffs(any) - 1;
        any &= any - 1;
        const uint32_t votes = __ballot_sync(0xffffffffu, (bits >> g) & 1u);
        if (lane == g) mine = __popc(votes);
    }
    s_cnt[warp][lane] = mine;
    __syncthreads();
    if (threadIdx.x < n_owners) {   // first slot of every warp of this tile in list g
        uint32_t run = offsets[(size_t)threadIdx.x * tiles + blockIdx.x];
        if (blockIdx.x == 0) dest_offsets[threadIdx.x] = run;   // list g starts where its tile 0 does
#pragma unroll
        for (int w = 0; w < kDestThreads / 32; ++w) {
            s_base[w][threadIdx.x] = run;
            run += s_cnt[w][threadIdx.x];
        }
    }
    __syncthreads();
    if (!dest_ids) return;
    for (uint32_t any = warp_any; any;) {
        const int g = __ffs(any) - 1;
        any &= any - 1;
        const uint32_t votes = __ballot_sync(0xffffffffu, (bits >> g) & 1u);
        if ((bits >> g) & 1u) {
            const uint32_t slot = s_base[warp][g] + __popc(votes & lanemask_lt());
            if (slot < cap) dest_ids[slot] = id;
        }
    }
}

int launch_pack_destinations(sph_ctx *c, int64_t n, const uint32_t *sorted_hash, const int32_t *sorted_owner,
                             const uint32_t *perm, uint32_t *dest_offsets, uint32_t *dest_ids, int64_t cap)
{
    const int G = c->params.n_owners;
    if (n == 0) {
        SPH_CUDA_TRY(c, cudaMemsetAsync(dest_offsets, 0, sizeof(uint32_t) * (G + 1), c->stream));
        return SPH_OK;
    }
    const uint32_t cells = c->grid.n_cells;
    const uint32_t tiles = (uint32_t)div_up(n, kDestThreads);
    uint32_t *counts = c->dest_counts, *offsets = c->dest_counts + (size_t)G * tiles;
    uint32_t *stencil_mask = c->cell_flag_count;   // stage 3's per-bucket scratch, free outside sph_comm_hash
    SPH_CUDA_TRY(c, cudaMemsetAsync(c->cell_mask, 0, sizeof(uint32_t) * cells, c->stream));
    owner_mask_kernel<<<div_up(div_up(n, kMaskItems), 256), 256, 0, c->stream>>>(n, sorted_hash, sorted_owner, c->cell_mask);
    SPH_CHECK_LAUNCH(c);
    {
        const int64_t groups = (int64_t)((c->grid.nx + kFlagCells - 1) / kFlagCells) * c->grid.ny * c->grid.nz;
        stencil_flag_kernel<true><<<div_up(groups, 256), 256, 0, c->stream>>>(c->grid, c->cell_mask, nullptr, nullptr,
                                                                              stencil_mask);
    }
    SPH_CHECK_LAUNCH(c);
    dest_count_kernel<<<tiles, kDestThreads, 0, c->stream>>>(n, sorted_hash, sorted_owner, stencil_mask, counts, tiles, G);
    SPH_CHECK_LAUNCH(c);
    int rc = launch_scan_exclusive(c, (int64_t)G * tiles, counts, offsets, dest_offsets + G);
    if (rc != SPH_OK) return rc;
    const uint32_t cap32 = (uint32_t)(cap > 0xffffffffll ? 0xffffffffll : cap);
    dest_scatter_kernel<<<tiles, kDestThreads, 0, c->stream>>>(n, sorted_hash, sorted_owner, perm, stencil_mask, offsets,
                                                               tiles, G, dest_offsets, dest_ids, cap32);
    SPH_CHECK_LAUNCH(c);
    return SPH_OK;
}

}  // namespace sphb
