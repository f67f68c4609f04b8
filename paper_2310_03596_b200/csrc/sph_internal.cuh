// Internal declarations shared by the CUDA translation units of libsph_b200.so.
// (Nothing here is visible to, or shared with, oracle/.)
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "sph.h"

namespace sphb {

constexpr int kRadixBits = 8;
constexpr int kRadix = 1 << kRadixBits;
constexpr int kMaxPasses = 4;

// onesweep tile geometry
constexpr int kSortThreads = 384;
constexpr int kSortItems = 16;
constexpr int kSortTile = kSortThreads * kSortItems;  // 6144 keys per tile

// decoupled look-back status word: 2 flag bits + 30 value bits
constexpr uint32_t kFlagAgg = 1u << 30;
constexpr uint32_t kFlagPrefix = 2u << 30;
constexpr uint32_t kFlagMask = 3u << 30;
constexpr uint32_t kValueMask = ~kFlagMask;

constexpr int kScanThreads = 256;
constexpr int kScanItems = 16;
constexpr int kScanTile = kScanThreads * kScanItems;

struct Grid {
    float ox, oy, oz;
    float inv_edge;      // 1.0f / (2.0f * h), rounded once (reading S2)
    int nx, ny, nz;
    uint32_t n_cells;
};

struct Consts {
    float support2;      // (2h)^2 in fp32
    float half_inv_h;    // 0.5 / h
    float cF;            // -(5 alpha / h^2),  alpha = 21 / (16 pi h^3)
    float cF_varh;       // -105 / (16 pi): the same constant with h_ij^-5 left to the pair (NEXT-4)
    float K, G;
};

// Stage events of the most recent steps: a ring of kTimingSlots event sets so that a caller can
// time many steps back to back without a host sync in between (sph_get_timing averages them).
constexpr int kTimingSlots = 32;
struct Timing {
    bool on = false;
    bool created = false;
    int64_t count = 0;                       // steps recorded since the last sph_get_timing
    cudaEvent_t ev[kTimingSlots][9] = {};
};

}  // namespace sphb

struct sph_ctx {
    sph_params params;
    sphb::Grid grid;
    sphb::Consts consts;
    int64_t max_n;
    cudaStream_t stream;
    int device;
    int num_sms;
    int key_bits;        // live bits of the hash
    int n_passes;
    int64_t launches;
    cudaError_t last_err;
    // sph_step_host: a second stream uploads velr / sig / owner while hash + sort (which need posm
    // only) already run; step_impl waits for `wait_before_reorder` (if set) before the reorder pass
    cudaStream_t copy_stream;
    cudaEvent_t ev_posm, ev_rest;
    bool host_streams_ready;
    uint32_t *h_count;           // pinned host word: landing place of the boundary count (sph_step_host)
    cudaEvent_t wait_before_reorder;

    // ---- scratch (device) ----
    void *arena;                 // one allocation, carved below
    size_t arena_bytes;
    uint32_t *alt_keys, *alt_vals;            // radix ping-pong
    uint32_t *hist;                           // [kMaxPasses][256] digit histograms -> exclusive
    uint32_t *tile_status;                    // [passes][tiles][256]
    uint32_t *tile_counter;                   // [kMaxPasses + 2] dynamic tile tickets
    uint32_t *cell_mask;                      // [cells] owner bitmask per bucket
    uint32_t *cell_flag_count;                // [cells] flagged particle count per bucket
    uint32_t *cell_offset;                    // [cells] exclusive scan of the above
    uint32_t *scan_status;                    // [scan tiles]
    uint32_t *dest_counts;                    // [2][n_owners][ceil(n / 256)] per-destination tile counts and their scan (NEXT-1)
    // step-internal products (used when the caller passes NULL)
    uint32_t *s_hash, *s_sorted_hash, *s_perm, *s_cell_start, *s_cell_end, *s_comm_hash;
    uint32_t *s_boundary_ids, *s_boundary_count, *s_owner_counts;
    float *s_drho, *s_acc, *s_dsig[6];
    unsigned long long *s_pair_count;
    sph_state sorted;                         // sorted copy of the state
    float *sorted_h;                          // sorted per-particle smoothing lengths (NEXT-4)
    float4 *rec_B, *rec_C;                    // packed neighbour records of the interaction kernel
    float4 *rec_D;
    void *bal;                                // control block of the balancing sweep (balance.cu)
    const uint32_t *hist_for;                 // the digit histograms in `hist` belong to this hash array (written by the fused hash kernel of sph_step), else NULL
    bool rec_fresh;                           // rec_B/C/D already hold the records of `sorted` (written by reorder)
    bool attr_sort, attr_interact;            // >48 KB dynamic shared memory opted in on THIS ctx's device
    // host-API staging (lazy)
    sph_state staging;
    bool staging_ready;
    sphb::Timing timing;
};

namespace sphb {

#define SPH_CUDA_TRY(ctx, expr)                                  \
    do {                                                         \
        cudaError_t e__ = (expr);                                \
        if (e__ != cudaSuccess) { (ctx)->last_err = e__; return SPH_ECUDA; } \
    } while (0)

#define SPH_CHECK_LAUNCH(ctx)                                    \
    do {                                                         \
        cudaError_t e__ = cudaPeekAtLastError();                 \
        (ctx)->launches++;                                       \
        if (e__ != cudaSuccess) { (ctx)->last_err = cudaGetLastError(); return SPH_ECUDA; } \
    } while (0)

static inline int div_up(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }

#ifdef __CUDACC__
__device__ __forceinline__ uint32_t bucket_coord(float x, float o, float inv, int n)
{
    // fp32 sequence pinned by reading S2: sub, mul (no contraction possible), then floor and clamp.
    // floor + clamp + conversion are exact operations, so they are done as ONE conversion
    // (round towards minus infinity, saturating; NaN -> 0) and two integer clamps: the same integer
    // as the oracle's clamp(floorf(u), 0, n - 1) for every finite input as long as n - 1 is exact in
    // fp32 (sph_create refuses dims above 2^24); 5 instead of 9 instructions.  A NaN position is
    // outside the contract (sph.h: "unspecified hash").
    const float t = __fsub_rn(x, o);
    const float u = __fmul_rn(t, inv);
    const int i = __float2int_rd(u);
    return (uint32_t)min(max(i, 0), n - 1);
}

__device__ __forceinline__ uint32_t bucket_hash(const float4 &p, const Grid &g)
{
    const uint32_t cx = bucket_coord(p.x, g.ox, g.inv_edge, g.nx);
    const uint32_t cy = bucket_coord(p.y, g.oy, g.inv_edge, g.ny);
    const uint32_t cz = bucket_coord(p.z, g.oz, g.inv_edge, g.nz);
    return cx + (uint32_t)g.nx * (cy + (uint32_t)g.ny * cz);
}
#endif

// stage launchers (each enqueues on ctx->stream, returns SPH_*)
int launch_hash(sph_ctx *c, int64_t n, const float *posm, uint32_t *hash);
int launch_hash_hist(sph_ctx *c, int64_t n, const float *posm, uint32_t *hash);   // hash + the sort's digit histograms
int launch_sort(sph_ctx *c, int64_t n, const uint32_t *hash, uint32_t *sorted_hash, uint32_t *perm);
int launch_reorder(sph_ctx *c, int64_t n, const uint32_t *perm, const sph_state *in,
                   const sph_state *out, const float *h_in = nullptr /* id order */, float *h_out = nullptr);
int launch_cell_ranges(sph_ctx *c, int64_t n, const uint32_t *sorted_hash, uint32_t *cs,
                       uint32_t *ce);
int launch_comm_hash(sph_ctx *c, int64_t n, const uint32_t *sorted_hash, const int32_t *sorted_owner,
                     const uint32_t *perm, const uint32_t *cs, const uint32_t *ce,
                     uint32_t *comm_hash, uint32_t *boundary_ids, uint32_t *boundary_count,
                     uint32_t *owner_counts);
int launch_pack_destinations(sph_ctx *c, int64_t n, const uint32_t *sorted_hash, const int32_t *sorted_owner,
                             const uint32_t *perm, uint32_t *dest_offsets, uint32_t *dest_ids, int64_t cap);
int launch_interact(sph_ctx *c, int64_t n, const sph_state *sorted, const uint32_t *sorted_hash,
                    const uint32_t *cs, const uint32_t *ce, float *drho, float *acc,
                    float *const dsig[6], unsigned long long *pair_count,
                    const sph_state *fuse_out /* NULL = rates only */, const uint32_t *perm, float dt,
                    int mode = 0 /* 0 all, 1 same-owner, 2 other-owner neighbours */,
                    const float *sorted_h = nullptr /* NEXT-4: per-particle smoothing lengths */,
                    float *drho_f = nullptr, float *acc_f = nullptr, float *const dsig_f[6] = nullptr /* mode 3 */);
int launch_integrate(sph_ctx *c, int64_t n, float dt, const sph_state *in, const float *drho,
                     const float *acc, const float *const dsig[6], const sph_state *out,
                     const uint32_t *scatter_perm /* NULL = elementwise */);
int launch_partition_by_label(sph_ctx *c, int64_t m, const uint32_t *ids, const int32_t *label, int n_labels,
                              uint32_t *offsets, uint32_t *dest /* [m] scatter map */);
int launch_partition_keys(sph_ctx *c, int64_t m, int n_labels /* keys in c->alt_keys, < 256 */, uint32_t *offsets,
                          uint32_t *dest /* optional */, uint32_t **order /* out: indices in partition order */);
int launch_scatter_records(sph_ctx *c, int64_t m, const uint32_t *ids, const uint32_t *dest,
                           const sph_state *in, const sph_state *out, uint32_t *packed_ids);
int launch_balance(sph_ctx *c, int64_t n, const float *posm, int32_t *owner, const int32_t *ptype, int n_types,
                   double alpha, int hmax, int32_t *bal_hash, unsigned long long *swapped);
size_t balance_scratch_bytes();
int launch_scan_exclusive(sph_ctx *c, int64_t n, const uint32_t *in, uint32_t *out,
                          uint32_t *total /* dev scalar */);

// ---- device helpers ----
// look-back status words carry flag and value in ONE 32-bit word, so relaxed gpu-scope accesses
// (served by L2) are enough; ld.volatile would be a system-scope load
__device__ __forceinline__ uint32_t ld_volatile_u32(const uint32_t *p)
{
    uint32_t v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_volatile_u32(uint32_t *p, uint32_t v)
{
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t lanemask_lt()
{
    uint32_t m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}
__device__ __forceinline__ float4 ldg_f4(const float *p)
{
    return __ldg(reinterpret_cast<const float4 *>(p));
}

}  // namespace sphb
