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

__global__ void __launch_bounds__(256)
owner_mask_kernel(int64_t n, const uint32_t *__restrict__ sorted_hash,
                  const int32_t *__restrict__ sorted_owner, uint32_t *__restrict__ cell_mask)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = k < n;
    const uint32_t h = valid ? sorted_hash[k] : 0xFFFFFFFFu;
    const uint32_t bit = valid ? (1u << (sorted_owner[k] & 31)) : 0u;
    const uint32_t peers = __match_any_sync(0xffffffffu, h);
    const uint32_t m = __reduce_or_sync(peers, bit);
    if (valid && (peers & lanemask_lt()) == 0) atomicOr(cell_mask + h, m);
}

__global__ void __launch_bounds__(256)
stencil_flag_kernel(Grid g, const uint32_t *__restrict__ cell_mask, const uint32_t *__restrict__ cs,
                    const uint32_t *__restrict__ ce, uint32_t *__restrict__ flag_count)
{
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= g.n_cells) return;
    const int cx = c % g.nx, cy = (c / g.nx) % g.ny, cz = c / (g.nx * g.ny);
    uint32_t m = 0;
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
            for (int dx = -1; dx <= 1; ++dx) {
                const int x = cx + dx;
                if (x < 0 || x >= g.nx) continue;
                m |= __ldg(cell_mask + row + x);
            }
        }
    }
    // an empty bucket contributes no particles whatever its stencil holds
    flag_count[c] = (__popc(m) >= 2) ? (ce[c] - cs[c]) : 0u;
}

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
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = k < n;
    bool flagged = false;
    uint32_t o = 0xFFu;
    if (valid) {
        const uint32_t h = sorted_hash[k];
        flagged = __ldg(flag_count + h) != 0u;
        comm_hash[k] = flagged ? h : SPH_GARBAGE_HASH;
        if (flagged) {
            boundary_ids[__ldg(cell_offset + h) + ((uint32_t)k - __ldg(cs + h))] = perm[k];
            o = (uint32_t)sorted_owner[k] & 31u;
        }
    }
    const uint32_t peers = __match_any_sync(0xffffffffu, o);
    if (flagged && (peers & lanemask_lt()) == 0) atomicAdd(&s_cnt[o], __popc(peers));
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
    owner_mask_kernel<<<div_up(n, 256), 256, 0, c->stream>>>(n, sorted_hash, sorted_owner, c->cell_mask);
    SPH_CHECK_LAUNCH(c);
    stencil_flag_kernel<<<div_up(cells, 256), 256, 0, c->stream>>>(c->grid, c->cell_mask, cs, ce,
                                                                   c->cell_flag_count);
    SPH_CHECK_LAUNCH(c);
    int rc = launch_scan_exclusive(c, cells, c->cell_flag_count, c->cell_offset, boundary_count);
    if (rc != SPH_OK) return rc;
    comm_hash_compact_kernel<<<div_up(n, 256), 256, 0, c->stream>>>(
        n, sorted_hash, sorted_owner, perm, cs, c->cell_flag_count, c->cell_offset, comm_hash,
        boundary_ids, owner_counts, c->params.n_owners);
    SPH_CHECK_LAUNCH(c);
    return SPH_OK;
}

}  // namespace sphb
