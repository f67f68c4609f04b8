// Stage 4a, main kernel: SPH interaction loops over the 27-bucket stencil ("the search
// for the neighboring particles is restricted to its bucket and to the surrounding buckets";
// steps e/f PAPER.md:24-25; "several interaction loops"; equations DESIGN.md O6-O8).
//
// Layout of the work (DESIGN.md section 6 gives the measurements that led here):
//  * x-fastest hashing makes the 27 buckets of a stencil 9 contiguous runs of the sorted arrays.
//    A CTA owns kTB consecutive buckets of one grid row; its candidate window is the 9 runs
//    widened by one bucket on each side.  The window's packed records (A = x,y,z,m;
//    B = vx,vy,vz,V; C = Sxx,Syy,Szz,Sxy; D = Sxz,Syz with V = m/rho, S = sigma/rho^2, written by
//    pack_kernel) are brought to shared memory with 1-D TMA bulk copies (cp.async.bulk +
//    mbarrier), no register staging.
//  * Phase 1 (distance tests): the warp holds 4 target particles of ONE bucket in registers;
//    lane l tests candidate v = 32 s + l of the bucket's candidate table against all 4 targets
//    (one 128-bit shared load per 128 tests) and records the outcome as one bit per target.
//  * The bit masks are exchanged with 3 shuffles so that quarter-warp q holds the complete
//    neighbour mask of target q, lane t of the quarter owning the candidates v = t (mod 8).
//  * Phase 2 (pair arithmetic): every lane pops one of its set bits per round and evaluates that
//    pair; the 8 lanes of a quarter touch 8 distinct 16-byte slots, so the 128-bit record
//    gathers are bank-conflict free.  The 16 partial sums are reduced over the 8 lanes, parked in
//    shared memory, and a lane-per-target epilogue forms the rates (O8) and stores them.
//  * No pair is skipped or evaluated twice: the self pair is accepted like any other (it
//    contributes exactly zero because x_ii = 0) and is subtracted from pair_count.
// Tiles whose window does not fit the shared-memory budget fall back to the direct walk.
#include "sph_internal.cuh"
#include "interact_math.cuh"

namespace sphb {

constexpr int kTB = 4;                 // buckets per tile along x
constexpr int kTW = 8;                 // warps per CTA (two per bucket)
constexpr int kCap = 1280;             // window records held in shared memory
constexpr int kCandCap = 1024;         // candidate-table entries per bucket
constexpr int kDrain = 512;            // candidates per phase-1/phase-2 round trip (16 x 32)
constexpr int kSlots = 16;             // targets parked per warp before the epilogue
constexpr int kAccStride = 17;         // 16 sums + 1 pad word (bank-conflict free)
constexpr int kDummy = kCap;           // record index of the far-away dummy candidate

struct Packed {
    const float4 *A;                   // sorted posm (x, y, z, m)
    float4 *B;                         // vx, vy, vz, V = m / rho
    float4 *C;                         // Sxx, Syy, Szz, Sxy     (S = sigma / rho^2)
    float2 *D;                         // Sxz, Syz
};

// ------------------------------------------------------------------------------------ pack
__global__ void __launch_bounds__(256)
pack_kernel(int64_t n, InteractIn in, float4 *__restrict__ B, float4 *__restrict__ C,
            float2 *__restrict__ D)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const float m = in.posm[k].w;
    const float4 v = in.velr[k];
    const float inv_rho = 1.0f / v.w;
    const float ir2 = inv_rho * inv_rho;
    B[k] = make_float4(v.x, v.y, v.z, m * inv_rho);
    C[k] = make_float4(in.sig[0][k] * ir2, in.sig[1][k] * ir2, in.sig[2][k] * ir2, in.sig[3][k] * ir2);
    D[k] = make_float2(in.sig[4][k] * ir2, in.sig[5][k] * ir2);
}

// ------------------------------------------------------------------------------------ PTX
__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_1d(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
            smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

// ------------------------------------------------------------------------------------ smem
struct __align__(16) TileSmem {
    float4 A[kCap + 2];
    float4 B[kCap + 2];
    float4 C[kCap + 2];
    float2 D[kCap + 2];
    float acc[kTW][kSlots][kAccStride];
    uint16_t cand[kTB][kCandCap];
    int run_lo[9];            // first sorted index copied for run r (even)
    int run_off[9];           // its record offset in shared memory (even)
    int run_hi[9];            // one past the last sorted index of run r
    uint64_t bar;
};


// ------------------------------------------------------------------------------------ kernel
__device__ __forceinline__ void reduce8(float &v)
{
    v += __shfl_xor_sync(0xffffffffu, v, 4);
    v += __shfl_xor_sync(0xffffffffu, v, 2);
    v += __shfl_xor_sync(0xffffffffu, v, 1);
}

__global__ void __launch_bounds__(kTW * 32, 2)
interact_tiled_kernel(Packed rec, InteractIn in, const uint32_t *__restrict__ cs,
                      const uint32_t *__restrict__ ce, Grid g, Consts k, InteractOut out,
                      unsigned long long *pair_count, int tiles_x)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TileSmem &sm = *reinterpret_cast<TileSmem *>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tx = blockIdx.x % tiles_x, yz = blockIdx.x / tiles_x;
    const int cy = yz % g.ny, cz = yz / g.ny;
    const int cx0 = tx * kTB;
    const int nb = min(kTB, g.nx - cx0);
    const uint32_t center = (uint32_t)g.nx * ((uint32_t)cy + (uint32_t)g.ny * (uint32_t)cz);
    const uint32_t t_lo = cs[center + cx0], t_hi = ce[center + cx0 + nb - 1];
    if (t_lo == t_hi) return;  // no target particle in this tile (uniform over the CTA)

    // ---- the 9 runs of the tile's window -------------------------------------------------
    if (tid < 9) {
        const int y = cy + (tid % 3) - 1, z = cz + (tid / 3) - 1;
        int lo = 0, hi = 0;
        if (y >= 0 && y < g.ny && z >= 0 && z < g.nz) {
            const uint32_t row = (uint32_t)g.nx * ((uint32_t)y + (uint32_t)g.ny * (uint32_t)z);
            lo = (int)cs[row + max(cx0 - 1, 0)];
            hi = (int)ce[row + min(cx0 + nb, g.nx - 1)];
        }
        if (hi <= lo) lo = hi = 0;
        sm.run_lo[tid] = lo & ~1;  // even start: 16-byte aligned source for the 8-byte D records
        sm.run_hi[tid] = hi;
    }
    if (tid == 0) {
        mbar_init(&sm.bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    if (tid == 32) sm.A[kDummy] = make_float4(1e18f, 1e18f, 1e18f, 0.f);
    __syncthreads();
    int total = 0;
    int run_off[9];
#pragma unroll
    for (int r = 0; r < 9; ++r) {
        run_off[r] = total;
        total += (sm.run_hi[r] - sm.run_lo[r] + 1) & ~1;
    }
    unsigned long long my_pairs = 0;
    if (total > kCap) {
        // window too large for shared memory (very dense region): direct walk for the tile
        for (uint32_t i = t_lo + tid; i < t_hi; i += kTW * 32) {
            int cx = cx0;
            while (i >= ce[center + cx]) ++cx;
            my_pairs += direct_particle((int64_t)i, cx, cy, cz, in, cs, ce, g, k, out);
        }
    } else {
        if (tid == 0) {
            uint32_t bytes = 0;
#pragma unroll
            for (int r = 0; r < 9; ++r) {
                const int len = sm.run_hi[r] - sm.run_lo[r];
                bytes += (uint32_t)len * 48u + (uint32_t)((len + 1) & ~1) * 8u;
            }
            mbar_expect_tx(&sm.bar, bytes);
#pragma unroll
            for (int r = 0; r < 9; ++r) {
                const int lo = sm.run_lo[r], len = sm.run_hi[r] - lo;
                if (len <= 0) continue;
                tma_load_1d(&sm.A[run_off[r]], rec.A + lo, (uint32_t)len * 16u, &sm.bar);
                tma_load_1d(&sm.B[run_off[r]], rec.B + lo, (uint32_t)len * 16u, &sm.bar);
                tma_load_1d(&sm.C[run_off[r]], rec.C + lo, (uint32_t)len * 16u, &sm.bar);
                tma_load_1d(&sm.D[run_off[r]], rec.D + lo, (uint32_t)((len + 1) & ~1) * 8u, &sm.bar);
            }
        }
        const int b = warp % kTB, half = warp / kTB;
        const int cx = cx0 + b;
        uint32_t tb0 = 0, nt = 0;
        if (b < nb) {
            tb0 = cs[center + cx];
            nt = ce[center + cx] - tb0;
        }
        if (nt > 0) {
            // ---- candidate table of bucket cx: its 27-bucket stencil as shared-memory indices,
            //      every run shifted so that (table position) == (record index) mod 8 ----------
            uint16_t *cand = sm.cand[b];
            int W = 0;
            bool overflow = false;
#pragma unroll
            for (int r = 0; r < 9; ++r) {
                const int y = cy + (r % 3) - 1, z = cz + (r / 3) - 1;
                if (y < 0 || y >= g.ny || z < 0 || z >= g.nz) continue;
                const uint32_t row = (uint32_t)g.nx * ((uint32_t)y + (uint32_t)g.ny * (uint32_t)z);
                const int sg = (int)cs[row + max(cx - 1, 0)], eg = (int)ce[row + min(cx + 1, g.nx - 1)];
                const int len = eg - sg;
                if (len <= 0) continue;
                const int s = run_off[r] + (sg - sm.run_lo[r]);
                const int pad = (s - W) & 7;
                if (W + pad + len > kCandCap - 32) { overflow = true; break; }
                if (lane < pad) cand[W + lane] = (uint16_t)kDummy;
                W += pad;
                for (int o = lane; o < len; o += 32) cand[W + o] = (uint16_t)(s + o);
                W += len;
            }
            if (overflow) {
                if (half == 0)
                    for (uint32_t i = tb0 + lane; i < tb0 + nt; i += 32)
                        my_pairs += direct_particle((int64_t)i, cx, cy, cz, in, cs, ce, g, k, out);
            } else {
                const int Wp = (W + 31) & ~31;
                if (W + lane < Wp) cand[W + lane] = (uint16_t)kDummy;
                __syncwarp();
                mbar_wait(&sm.bar, 0);

                const int q = lane >> 3, t = lane & 7;
                const int tbase = run_off[4] + ((int)tb0 - sm.run_lo[4]);  // targets sit in the centre run
                float(*acc)[kAccStride] = sm.acc[warp];
                int parked = 0;
                for (uint32_t p = half; 4 * p < nt; p += 2) {
                    // quarter q works for target 4p + q; T[d] is the position of target 4p + (q ^ d)
                    float Tx[4], Ty[4], Tz[4];
#pragma unroll
                    for (int d = 0; d < 4; ++d) {
                        const uint32_t ti = 4 * p + (uint32_t)(q ^ d);
                        float4 pa = make_float4(-1e18f, -1e18f, -1e18f, 0.f);
                        if (ti < nt) pa = sm.A[tbase + ti];
                        Tx[d] = pa.x; Ty[d] = pa.y; Tz[d] = pa.z;
                    }
                    const uint32_t my_t = 4 * p + (uint32_t)q;
                    const bool my_valid = my_t < nt;
                    float4 tv = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (my_valid) tv = sm.B[tbase + my_t];
                    PairAccum S;
                    S.clear();
                    for (int base = 0; base < Wp; base += kDrain) {
                        // ---- phase 1: distance tests, one bit per (target, candidate) --------
                        uint32_t M0 = 0, M1 = 0, M2 = 0, M3 = 0;
                        const int nch = min(kDrain, Wp - base) >> 5;
                        for (int s = 0; s < nch; ++s) {
                            const float4 pa = sm.A[cand[base + 32 * s + lane]];
                            const uint32_t bit = 1u << s;
                            {
                                const float dx = Tx[0] - pa.x, dy = Ty[0] - pa.y, dz = Tz[0] - pa.z;
                                if (dx * dx + dy * dy + dz * dz < k.support2) M0 |= bit;
                            }
                            {
                                const float dx = Tx[1] - pa.x, dy = Ty[1] - pa.y, dz = Tz[1] - pa.z;
                                if (dx * dx + dy * dy + dz * dz < k.support2) M1 |= bit;
                            }
                            {
                                const float dx = Tx[2] - pa.x, dy = Ty[2] - pa.y, dz = Tz[2] - pa.z;
                                if (dx * dx + dy * dy + dz * dz < k.support2) M2 |= bit;
                            }
                            {
                                const float dx = Tx[3] - pa.x, dy = Ty[3] - pa.y, dz = Tz[3] - pa.z;
                                if (dx * dx + dy * dy + dz * dz < k.support2) M3 |= bit;
                            }
                        }
                        // ---- hand every quarter the masks of its own target ------------------
                        const uint32_t R1 = __shfl_xor_sync(0xffffffffu, M1, 8);
                        const uint32_t R2 = __shfl_xor_sync(0xffffffffu, M2, 16);
                        const uint32_t R3 = __shfl_xor_sync(0xffffffffu, M3, 24);
                        uint32_t lo = M0 | (R1 << 16), hi = R2 | (R3 << 16);
                        my_pairs += __popc(lo) + __popc(hi);
                        // ---- phase 2: one accepted pair per lane and round -------------------
                        while (__any_sync(0xffffffffu, (lo | hi) != 0u)) {
                            if ((lo | hi) != 0u) {
                                int bp;
                                if (lo) { bp = __ffs(lo) - 1; lo &= lo - 1; }
                                else    { bp = 31 + __ffs(hi); hi &= hi - 1; }
                                const int v = base + ((bp & 15) << 5) + (((bp >> 4) ^ q) << 3) + t;
                                const int j = cand[v];
                                const float4 pa = sm.A[j];
                                const float4 pb = sm.B[j];
                                const float4 pc = sm.C[j];
                                const float2 pd = sm.D[j];
                                const float dx = Tx[0] - pa.x, dy = Ty[0] - pa.y, dz = Tz[0] - pa.z;
                                const float r2 = dx * dx + dy * dy + dz * dz;
                                const float Sj[6] = {pc.x, pc.y, pc.z, pc.w, pd.x, pd.y};
                                S.add(dx, dy, dz, r2, pa.w, pb.w, pb.x - tv.x, pb.y - tv.y, pb.z - tv.z,
                                      Sj, k.half_inv_h);
                            }
                        }
                    }
                    // ---- reduce the 16 sums over the quarter, park them ----------------------
                    reduce8(S.dr);
#pragma unroll
                    for (int c = 0; c < 9; ++c) reduce8(S.L[c]);
#pragma unroll
                    for (int c = 0; c < 3; ++c) { reduce8(S.g[c]); reduce8(S.a[c]); }
                    if (t == 0) {
                        float *row = acc[parked * 4 + q];
                        row[0] = S.dr;
#pragma unroll
                        for (int c = 0; c < 9; ++c) row[1 + c] = S.L[c];
#pragma unroll
                        for (int c = 0; c < 3; ++c) { row[10 + c] = S.g[c]; row[13 + c] = S.a[c]; }
                        row[16] = __int_as_float(my_valid ? (int)(tb0 + my_t) : -1);
                    }
                    if (my_valid && t == 0) my_pairs -= 1;  // the self pair (reading S15)
                    ++parked;
                    const bool last = 4 * (p + 2) >= nt;
                    if (parked == kSlots / 4 || last) {
                        // ---- epilogue: one lane per parked target (O8, stores) ---------------
                        __syncwarp();
                        if (lane < parked * 4) {
                            const float *row = acc[lane];
                            const int i = __float_as_int(row[16]);
                            if (i >= 0) {
                                PairAccum R;
                                R.dr = row[0];
#pragma unroll
                                for (int c = 0; c < 9; ++c) R.L[c] = row[1 + c];
#pragma unroll
                                for (int c = 0; c < 3; ++c) { R.g[c] = row[10 + c]; R.a[c] = row[13 + c]; }
                                float si[6];
#pragma unroll
                                for (int c = 0; c < 6; ++c) si[c] = in.sig[c][i];
                                finish_particle(R, si, in.velr[i].w, k, out, (int64_t)i);
                            }
                        }
                        __syncwarp();
                        parked = 0;
                    }
                }
            }
        }
    }
    if (total <= kCap && tid == 0) mbar_wait(&sm.bar, 0);  // never leave with copies in flight
    if (pair_count) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) my_pairs += __shfl_xor_sync(0xffffffffu, my_pairs, o);
        if (lane == 0 && my_pairs) atomicAdd(pair_count, my_pairs);
    }
}

int launch_interact_tiled(sph_ctx *c, int64_t n, const InteractIn &in, const uint32_t *sorted_hash,
                          const uint32_t *cs, const uint32_t *ce, const InteractOut &out,
                          unsigned long long *pair_count)
{
    (void)sorted_hash;
    Packed rec;
    rec.A = in.posm;
    rec.B = c->rec_B;
    rec.C = c->rec_C;
    rec.D = c->rec_D;
    pack_kernel<<<div_up(n, 256), 256, 0, c->stream>>>(n, in, rec.B, rec.C, rec.D);
    SPH_CHECK_LAUNCH(c);
    static bool attr_set = false;
    const int smem = (int)sizeof(TileSmem);
    if (!attr_set) {
        SPH_CUDA_TRY(c, cudaFuncSetAttribute(interact_tiled_kernel,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        attr_set = true;
    }
    const int tiles_x = (c->grid.nx + kTB - 1) / kTB;
    const int64_t tiles = (int64_t)tiles_x * c->grid.ny * c->grid.nz;
    if (tiles > 0x7fffffffll) return SPH_EINVAL;
    interact_tiled_kernel<<<(unsigned)tiles, kTW * 32, smem, c->stream>>>(rec, in, cs, ce, c->grid, c->consts,
                                                                       out, pair_count, tiles_x);
    SPH_CHECK_LAUNCH(c);
    return SPH_OK;
}

}  // namespace sphb
