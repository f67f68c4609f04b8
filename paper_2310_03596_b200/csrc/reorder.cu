// Stage 2b: gather the particle state into sorted order ("The particles are then sorted",
// PAPER.md:13), so that the interaction loop reads coalesced SoA arrays.
// 4 B (perm) + 60 B gathered + 60 B written per particle; HBM-bound.  The gather has good
// sector locality because id order and bucket order are both spatially coherent.
#include "sph_internal.cuh"

namespace sphb {

struct StatePtrs {
    const float4 *posm, *velr;
    const float *sig[6];
    const int32_t *owner;
};
struct StatePtrsOut {
    float4 *posm, *velr;
    float *sig[6];
    int32_t *owner;
};

// PACK: also write the packed neighbour records of the interaction kernel (B = vx, vy, vz, Szz;
// C = Sxx, Sxy, Sxy, Syy; D = Sxz, Syz, m, V with S = sigma / rho^2, V = m / rho; layout of
// PairAccum2 in interact_math.cuh) while the state is in registers anyway: inside sph_step this
// replaces the separate pack pass (56 B read + 48 B written per particle) by 48 B written.
template <bool PACK>
__global__ void __launch_bounds__(256)
reorder_kernel(int64_t n, const uint32_t *__restrict__ perm, StatePtrs in, StatePtrsOut out,
               float4 *__restrict__ recB, float4 *__restrict__ recC, float4 *__restrict__ recD,
               const float *__restrict__ h_in, float *__restrict__ h_out)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const uint32_t id = __ldcs(perm + k);
    // issue every gather before the first store
    const float4 p = __ldg(in.posm + id);
    const float4 v = __ldg(in.velr + id);
    float s[6];
#pragma unroll
    for (int c = 0; c < 6; ++c) s[c] = __ldg(in.sig[c] + id);
    const int32_t o = __ldg(in.owner + id);
    float hk = 0.f;   // NEXT-4: per-particle smoothing length (C.z of the record carries it)
    if (h_in) { hk = __ldg(h_in + id); h_out[k] = hk; }
    out.posm[k] = p;
    out.velr[k] = v;
#pragma unroll
    for (int c = 0; c < 6; ++c) out.sig[c][k] = s[c];
    out.owner[k] = o;
    if (PACK) {
        const float inv_rho = 1.0f / v.w;
        const float ir2 = inv_rho * inv_rho;
        const float sxy = s[3] * ir2;
        recB[k] = make_float4(v.x, v.y, v.z, s[2] * ir2);
        recC[k] = make_float4(s[0] * ir2, sxy, h_in ? hk : sxy, s[1] * ir2);
        recD[k] = make_float4(s[4] * ir2, s[5] * ir2, p.w, p.w * inv_rho);
    }
}

// NEXT-1: record packing.  Entry k of the boundary list goes to slot dest[k] of the
// label-segmented buffers.  A tile of kPackTile consecutive list entries is gathered in list order
// (the same sector-friendly gather as the reorder pass), staged in shared memory sorted by
// destination -- inside a tile the entries of one label have CONSECUTIVE destinations, because the
// partition is stable -- and leaves as one contiguous run per label and array.  (A plain gather by
// packed ids re-read every sector once per label, a plain scatter wrote 8-byte pieces: both
// measured ~7 ms at 64 M boundary particles with 16 random labels.)
// Tile geometry as measured at 64 M boundary particles, 16 random owners (whole sph_pack_boundary,
// round 3): 2048 / 1024 threads 2.85 ms, 1024 / 512 2.66, 512 / 256 2.55, 384 / 192 2.53, 256 / 128
// 2.62, 512 / 512 2.78, 256 / 256 2.48 ms (61.5 % of HBM peak).  The load and the store phase of a
// CTA do not overlap, so many small CTAs per SM (17 KB of shared memory each) hide each other's
// phases better than three big ones; the per-label runs of a tile (16 entries at 16 labels) are
// still whole sectors for the 16-byte fields.
constexpr int kPackTile = 256;
constexpr int kPackThreads = 256;
struct PackSmem {
    float4 posm[kPackTile], velr[kPackTile];
    float sig[6][kPackTile];
    int32_t owner[kPackTile];
    uint32_t id[kPackTile], gdst[kPackTile];
    uint32_t lmin[SPH_MAX_OWNERS], lcnt[SPH_MAX_OWNERS], lbase[SPH_MAX_OWNERS];
};

__global__ void __launch_bounds__(kPackThreads)
pack_records_kernel(int64_t m, const uint32_t *__restrict__ ids, const uint32_t *__restrict__ dest,
                    const uint32_t *__restrict__ label, StatePtrs in, StatePtrsOut out,
                    uint32_t *__restrict__ packed_ids)
{
    extern __shared__ __align__(16) unsigned char pack_smem_raw[];
    PackSmem &sm = *reinterpret_cast<PackSmem *>(pack_smem_raw);
    const int tid = threadIdx.x;
    const int64_t base = (int64_t)blockIdx.x * kPackTile;
    const int cnt = (int)min((int64_t)kPackTile, m - base);
    if (tid < SPH_MAX_OWNERS) { sm.lmin[tid] = 0xFFFFFFFFu; sm.lcnt[tid] = 0u; }
    __syncthreads();
    constexpr int kPer = kPackTile / kPackThreads;
    uint32_t id[kPer], d[kPer], o[kPer];
#pragma unroll
    for (int j = 0; j < kPer; ++j) {
        const int e = tid + j * kPackThreads;
        if (e < cnt) {
            id[j] = __ldcs(ids + base + e);
            d[j] = __ldcs(dest + base + e);
            o[j] = __ldcs(label + base + e) & (SPH_MAX_OWNERS - 1);
            atomicMin(&sm.lmin[o[j]], d[j]);
            atomicAdd(&sm.lcnt[o[j]], 1u);
        }
    }
    __syncthreads();
    if (tid < 32) {   // exclusive scan of the per-label counts (SPH_MAX_OWNERS == 32)
        const uint32_t c0 = sm.lcnt[tid];
        uint32_t inc = c0;
#pragma unroll
        for (int s = 1; s < 32; s <<= 1) {
            const uint32_t x = __shfl_up_sync(0xffffffffu, inc, s);
            if (tid >= s) inc += x;
        }
        sm.lbase[tid] = inc - c0;
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < kPer; ++j) {
        const int e = tid + j * kPackThreads;
        if (e < cnt) {
            const uint32_t slot = sm.lbase[o[j]] + (d[j] - sm.lmin[o[j]]);
            sm.posm[slot] = __ldg(in.posm + id[j]);
            sm.velr[slot] = __ldg(in.velr + id[j]);
#pragma unroll
            for (int c = 0; c < 6; ++c) sm.sig[c][slot] = __ldg(in.sig[c] + id[j]);
            sm.owner[slot] = __ldg(in.owner + id[j]);
            sm.id[slot] = id[j];
            sm.gdst[slot] = d[j];
        }
    }
    __syncthreads();
    for (int slot = tid; slot < cnt; slot += kPackThreads) {
        const uint32_t g = sm.gdst[slot];
        packed_ids[g] = sm.id[slot];
        out.posm[g] = sm.posm[slot];
        out.velr[g] = sm.velr[slot];
#pragma unroll
        for (int c = 0; c < 6; ++c) out.sig[c][g] = sm.sig[c][slot];
        out.owner[g] = sm.owner[slot];
    }
}

int launch_scatter_records(sph_ctx *c, int64_t m, const uint32_t *ids, const uint32_t *dest,
                           const sph_state *in, const sph_state *out, uint32_t *packed_ids)
{
    if (m == 0) return SPH_OK;
    static_assert(SPH_MAX_OWNERS == 32, "one warp scans the per-label counts");
    StatePtrs a;
    StatePtrsOut b;
    a.posm = reinterpret_cast<const float4 *>(in->posm);
    a.velr = reinterpret_cast<const float4 *>(in->velr);
    a.owner = in->owner;
    b.posm = reinterpret_cast<float4 *>(out->posm);
    b.velr = reinterpret_cast<float4 *>(out->velr);
    b.owner = out->owner;
    for (int i = 0; i < 6; ++i) { a.sig[i] = in->sig[i]; b.sig[i] = out->sig[i]; }
    SPH_CUDA_TRY(c, cudaFuncSetAttribute(pack_records_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)sizeof(PackSmem)));
    // c->alt_keys still holds the label of every list entry (written by the partition)
    pack_records_kernel<<<div_up(m, kPackTile), kPackThreads, sizeof(PackSmem), c->stream>>>(
        m, ids, dest, c->alt_keys, a, b, packed_ids);
    SPH_CHECK_LAUNCH(c);
    return SPH_OK;
}

int launch_reorder(sph_ctx *c, int64_t n, const uint32_t *perm, const sph_state *in,
                   const sph_state *out, const float *h_in, float *h_out)
{
    if (n == 0) return SPH_OK;
    StatePtrs a;
    StatePtrsOut b;
    a.posm = reinterpret_cast<const float4 *>(in->posm);
    a.velr = reinterpret_cast<const float4 *>(in->velr);
    a.owner = in->owner;
    b.posm = reinterpret_cast<float4 *>(out->posm);
    b.velr = reinterpret_cast<float4 *>(out->velr);
    b.owner = out->owner;
    for (int i = 0; i < 6; ++i) { a.sig[i] = in->sig[i]; b.sig[i] = out->sig[i]; }
    // the ctx's own sorted copy (sph_step) gets its interaction records in the same pass
    const bool pack = out->posm == c->sorted.posm;
    if (pack)
        reorder_kernel<true><<<div_up(n, 256), 256, 0, c->stream>>>(n, perm, a, b, c->rec_B, c->rec_C, c->rec_D,
                                                                    h_in, h_out);
    else
        reorder_kernel<false><<<div_up(n, 256), 256, 0, c->stream>>>(n, perm, a, b, nullptr, nullptr, nullptr,
                                                                     h_in, h_out);
    SPH_CHECK_LAUNCH(c);
    c->rec_fresh = pack;
    return SPH_OK;
}

}  // namespace sphb
