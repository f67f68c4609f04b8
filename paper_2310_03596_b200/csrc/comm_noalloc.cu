// sph_comm_hash_noalloc: the communication hash (step c) for callers
// that must not allocate device memory.
//
// Who that is: code that runs where cudaMalloc / cudaFree are off limits -- a solver that handed
// all of its device memory to its own pool at start-up and has none left for the driver to give
// out, a plug-in running inside a host application whose rules forbid allocations (and the
// implicit device-wide synchronisation of cudaFree) in the time loop, or a thread that drives a
// latency-critical stream and cannot afford the allocator's locks.  Every other entry point of
// this library needs an sph_ctx, and sph_create allocates the ctx's scratch arena with
// cudaMalloc.  This one needs no ctx.
//
// How: the only scratch the communication hash needs is one owner bitmask per bucket
// (I5).  Here it lives in a file-scope __device__ array of fixed size
// (SPH_NOALLOC_MAX_CELLS words = 16 MiB), part of the library image: every GPU that loads the
// library's module carries it until the process exits, whether or not this entry point is used.
// The kernels are variants of owner_mask_kernel / stencil_flag_kernel of comm.cu: same bucket
// masks, but the 27-stencil OR is taken per particle, so no per-bucket flag / offset tables (and
// no cell_start / cell_end) are needed; the boundary LIST is not produced, only comm_hash and
// the number of boundary particles.
//
// Consequences the caller must know (also in include/sph.h):
//  - the array is shared by every call on a device and keeps the previous call's masks: each
//    call clears the words of its own grid first (a cudaMemsetAsync on the caller's stream);
//  - two calls whose work overlaps on one GPU (two streams, two host threads) race on it;
//  - a grid with more buckets than the array holds is refused with SPH_ELIMIT;
//  - the array's device address is looked up once per device, by the first call made while that
//    device is current (cudaGetSymbolAddress); make that first call outside any stream capture.
#include <mutex>

#include "sph_internal.cuh"

namespace sphb {

// The scratch.  In HOST code this name is only a handle for cudaGetSymbolAddress -- it is not a
// device address and must never be passed to a kernel or to cudaMemset as a pointer.
static __device__ __align__(256) uint32_t g_noalloc_cell_mask[SPH_NOALLOC_MAX_CELLS];

constexpr int kNoallocMaxDevices = 64;
static std::mutex g_noalloc_mu;
static uint32_t *g_noalloc_ptr[kNoallocMaxDevices];   // device address of the array, per device ordinal

// Device address of the scratch on the CURRENT device; resolved on the first call per device.
static int noalloc_scratch(uint32_t **out)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return SPH_ECUDA;
    if (dev < 0 || dev >= kNoallocMaxDevices) return SPH_EINVAL;
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (g_noalloc_ptr[dev] == nullptr) {
        void *p = nullptr;
        if (cudaGetSymbolAddress(&p, g_noalloc_cell_mask) != cudaSuccess || p == nullptr) return SPH_ECUDA;
        g_noalloc_ptr[dev] = static_cast<uint32_t *>(p);
    }
    *out = g_noalloc_ptr[dev];
    return SPH_OK;
}

constexpr int kNaItems = 8;   // sorted particles per thread

// Variant of owner_mask_kernel (comm.cu): the sorted array holds every bucket as one run, so a
// thread ORs the owner bits of its 8 consecutive particles run by run and issues one atomicOr per
// run end.  `cell_mask` is the static scratch, passed in by its looked-up device address.
__global__ void __launch_bounds__(256)
noalloc_owner_mask_kernel(int64_t n, uint32_t n_cells, const uint32_t *__restrict__ sorted_hash,
                          const int32_t *__restrict__ sorted_owner, uint32_t *__restrict__ cell_mask)
{
    const int64_t k0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * kNaItems;
    if (k0 >= n) return;
    uint32_t cur = sorted_hash[k0], m = 1u << (sorted_owner[k0] & 31);
#pragma unroll
    for (int j = 1; j < kNaItems; ++j) {
        if (k0 + j >= n) break;
        const uint32_t hj = sorted_hash[k0 + j];
        if (hj != cur) {
            if (cur < n_cells) atomicOr(cell_mask + cur, m);   // a hash outside the grid is ignored, never a fault
            cur = hj;
            m = 0u;
        }
        m |= 1u << (sorted_owner[k0 + j] & 31);
    }
    if (cur < n_cells) atomicOr(cell_mask + cur, m);
}

// One thread per sorted particle: OR of the owner masks over the 27-bucket stencil of its bucket
// (out-of-grid buckets skipped, reading S9), comm hash = own hash if two or more owners are
// present (the particle's own bit is one of them, I5), else the garbage hash.
// Neighbouring threads sit in the same bucket, so the 27 loads are L1 hits for most of a warp.
__global__ void __launch_bounds__(256)
noalloc_comm_hash_kernel(int64_t n, Grid g, const uint32_t *__restrict__ sorted_hash,
                         const uint32_t *__restrict__ cell_mask, uint32_t *__restrict__ comm_hash,
                         uint32_t *__restrict__ boundary_count)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool flagged = false;
    const uint32_t c = k < n ? sorted_hash[k] : SPH_GARBAGE_HASH;
    if (k < n && c >= g.n_cells) comm_hash[k] = SPH_GARBAGE_HASH;   // not a bucket of this grid
    if (c < g.n_cells) {
        const int cx = (int)(c % (uint32_t)g.nx);
        const int cy = (int)((c / (uint32_t)g.nx) % (uint32_t)g.ny);
        const int cz = (int)(c / ((uint32_t)g.nx * (uint32_t)g.ny));
        uint32_t m = 0u;
        for (int dz = -1; dz <= 1; ++dz) {
            const int z = cz + dz;
            if (z < 0 || z >= g.nz) continue;
            for (int dy = -1; dy <= 1; ++dy) {
                const int y = cy + dy;
                if (y < 0 || y >= g.ny) continue;
                const uint32_t row = (uint32_t)g.nx * ((uint32_t)y + (uint32_t)g.ny * (uint32_t)z);
                for (int dx = -1; dx <= 1; ++dx) {
                    const int x = cx + dx;
                    if (x >= 0 && x < g.nx) m |= cell_mask[row + (uint32_t)x];
                }
            }
        }
        flagged = __popc(m) >= 2;
        comm_hash[k] = flagged ? c : SPH_GARBAGE_HASH;
    }
    const uint32_t votes = __ballot_sync(0xffffffffu, flagged);
    if ((threadIdx.x & 31) == 0 && votes) atomicAdd(boundary_count, (uint32_t)__popc(votes));
}

}  // namespace sphb

using namespace sphb;

extern "C" int sph_comm_hash_noalloc(const sph_params *params, int64_t n, const uint32_t *sorted_hash,
                                     const int32_t *sorted_owner, uint32_t *comm_hash,
                                     uint32_t *boundary_count, void *cuda_stream)
{
    // argument checks first: none of them touches the CUDA runtime
    if (!params || !boundary_count || n < 0 || n > ((int64_t)1 << 30)) return SPH_EINVAL;
    if (params->n_owners < 1 || params->n_owners > SPH_MAX_OWNERS) return SPH_EINVAL;
    for (int a = 0; a < 3; ++a)
        if (params->dims[a] <= 0) return SPH_EINVAL;
    uint64_t cells = 1;   // bounded after every factor, so the product cannot wrap
    for (int a = 0; a < 3; ++a) {
        cells *= (uint64_t)params->dims[a];
        if (cells > (uint64_t)SPH_NOALLOC_MAX_CELLS) return SPH_ELIMIT;
    }
    if (n > 0 && (!sorted_hash || !sorted_owner || !comm_hash)) return SPH_EINVAL;

    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    uint32_t *mask = nullptr;
    const int rc = noalloc_scratch(&mask);
    if (rc != SPH_OK) return rc;

    if (cudaMemsetAsync(boundary_count, 0, sizeof(uint32_t), stream) != cudaSuccess) return SPH_ECUDA;
    if (n == 0) return SPH_OK;
    // the array still holds the masks of whatever call came before: clear this grid's words
    if (cudaMemsetAsync(mask, 0, sizeof(uint32_t) * cells, stream) != cudaSuccess) return SPH_ECUDA;

    Grid g{};
    g.nx = params->dims[0];
    g.ny = params->dims[1];
    g.nz = params->dims[2];
    g.n_cells = (uint32_t)cells;
    noalloc_owner_mask_kernel<<<div_up(div_up(n, kNaItems), 256), 256, 0, stream>>>(n, g.n_cells, sorted_hash, sorted_owner, mask);
    if (cudaPeekAtLastError() != cudaSuccess) return SPH_ECUDA;
    noalloc_comm_hash_kernel<<<div_up(n, 256), 256, 0, stream>>>(n, g, sorted_hash, mask, comm_hash, boundary_count);
    if (cudaPeekAtLastError() != cudaSuccess) return SPH_ECUDA;
    return SPH_OK;
}
