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
    float4 A[kCap + 2];       // x - ox, y - oy, z - oz, m   (tile-local coordinates after the shift)
    float4 B[kCap + 2];
    float4 C[kCap + 2];
    float2 D[kCap + 2];
    float P2[kCap + 2];       // |p'|^2 of the shifted position
    float acc[kTW][kSlots][kAccStride];
    uint16_t cand[kTB][kCandCap];
    int cand_len[kTB];        // padded table length (multiple of 32), -1 = overflow -> direct walk
    uint64_t bar;
};

// ------------------------------------------------------------------------------------ kernel
// Sum 16 values over the 8 lanes of a quarter-warp with 14 shuffles: every stage halves the
// number of values a lane carries.  On return lane t holds in (v[0], v[1]) the complete sums
// of the original indices idx and idx + 1, idx = 8 (t>>2 & 1) + 4 (t>>1 & 1) + 2 (t & 1).
__device__ __forceinline__ void reduce8_transposed(float (&v)[16], int t)
{
    const bool b2 = t & 4, b1 = t & 2, b0 = t & 1;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const float send = b2 ? v[i] : v[i + 8];
        const float keep = b2 ? v[i + 8] : v[i];
        v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float send = b1 ? v[i] : v[i + 4];
        const float keep = b1 ? v[i + 4] : v[i];
        v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 2);
    }
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const float send = b0 ? v[i] : v[i + 2];
        const float keep = b0 ? v[i + 2] : v[i];
        v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 1);
    }
}

// One phase-1 test: sign bit of (|p'|^2 - 2 T'.p' - thr) shifted into the mask (1 = inside).
__device__ __forceinline__ void test_push(uint32_t &mask, const float4 &pa, float p2, float ax, float ay,
                                          float az, float thr)
{
    float acc = fmaf(ax, pa.x, p2);
    acc = fmaf(ay, pa.y, acc);
    acc = fmaf(az, pa.z, acc);
    acc -= thr;
    mask = __funnelshift_l(__float_as_uint(acc), mask, 1);
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

    // ---- the 9 runs of the tile's window: lane r of every warp describes run r ----------------
    const int ry = cy + (lane % 3) - 1, rz = cz + (lane / 3) - 1;
    const bool row_ok = lane < 9 && ry >= 0 && ry < g.ny && rz >= 0 && rz < g.nz;
    const uint32_t rrow = row_ok ? (uint32_t)g.nx * ((uint32_t)ry + (uint32_t)g.ny * (uint32_t)rz) : 0u;
    int run_lo = 0, run_len = 0;  // first sorted index copied (even) and number of records
    if (row_ok) {
        const int lo = (int)cs[rrow + max(cx0 - 1, 0)], hi = (int)ce[rrow + min(cx0 + nb, g.nx - 1)];
        if (hi > lo) { run_lo = lo & ~1; run_len = hi - run_lo; }
    }
    const int run_cnt = (run_len + 1) & ~1;  // even record count: keeps every offset 16-byte aligned
    int run_off = run_cnt;                   // exclusive prefix over lanes 0..8
#pragma unroll
    for (int o = 1; o < 16; o <<= 1) {
        const int x = __shfl_up_sync(0xffffffffu, run_off, o);
        if (lane >= o) run_off += x;
    }
    const int total = __shfl_sync(0xffffffffu, run_off, 8);
    run_off -= run_cnt;

    if (tid == 0) {
        mbar_init(&sm.bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    uint32_t my_pairs = 0, my_self = 0;
    if (total > kCap) {
        // window too large for shared memory (very dense region): direct walk for the tile
        for (uint32_t i = t_lo + tid; i < t_hi; i += kTW * 32) {
            int cx = cx0;
            while (i >= ce[center + cx]) ++cx;
            my_pairs += direct_particle((int64_t)i, cx, cy, cz, in, cs, ce, g, k, out);
        }
    } else {
        if (warp == 0) {
            const uint32_t bytes = __reduce_add_sync(0xffffffffu, (uint32_t)run_len * 48u + (uint32_t)run_cnt * 8u);
            if (lane == 0) mbar_expect_tx(&sm.bar, bytes);
            __syncwarp();
            if (run_len > 0) {
                tma_load_1d(&sm.A[run_off], rec.A + run_lo, (uint32_t)run_len * 16u, &sm.bar);
                tma_load_1d(&sm.B[run_off], rec.B + run_lo, (uint32_t)run_len * 16u, &sm.bar);
                tma_load_1d(&sm.C[run_off], rec.C + run_lo, (uint32_t)run_len * 16u, &sm.bar);
                tma_load_1d(&sm.D[run_off], rec.D + run_lo, (uint32_t)run_cnt * 8u, &sm.bar);
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
            //      every run shifted so that (table position) == (record index) mod 8.  Lane r
            //      looks run r up; the two warps of the bucket fill alternate runs. -------------
            int s_r = 0, len_r = 0;
            if (row_ok) {
                const int sg = (int)cs[rrow + max(cx - 1, 0)], eg = (int)ce[rrow + min(cx + 1, g.nx - 1)];
                len_r = max(eg - sg, 0);
                s_r = run_off + (sg - run_lo);
            }
            uint16_t *cand = sm.cand[b];
            int W = 0;
#pragma unroll
            for (int r = 0; r < 9; ++r) {
                const int s = __shfl_sync(0xffffffffu, s_r, r), len = __shfl_sync(0xffffffffu, len_r, r);
                if (len == 0) continue;
                const int pad = (s - W) & 7;
                if ((r & 1) == half && W + pad + len <= kCandCap - 32) {
                    if (lane < pad) cand[W + lane] = (uint16_t)kDummy;
                    for (int o = lane; o < len; o += 32) cand[W + pad + o] = (uint16_t)(s + o);
                }
                W += pad + len;
            }
            const bool overflow = W > kCandCap - 32;
            const int Wp = (W + 31) & ~31;
            if (half == 0) {
                if (!overflow && W + lane < Wp) cand[W + lane] = (uint16_t)kDummy;
                if (lane == 0) sm.cand_len[b] = overflow ? -1 : Wp;
            }
        }
        // ---- wait for the window, shift it to tile-local coordinates, form |p'|^2 ---------------
        __syncthreads();  // mbarrier initialised before anyone waits on it
        mbar_wait(&sm.bar, 0);
        {
            const float edge = 1.0f / g.inv_edge;
            const float ox = g.ox + (float)cx0 * edge, oy = g.oy + (float)cy * edge,
                        oz = g.oz + (float)cz * edge;
            for (int j = tid; j < total; j += kTW * 32) {
                float4 pa = sm.A[j];
                pa.x -= ox; pa.y -= oy; pa.z -= oz;
                sm.A[j] = pa;
                sm.P2[j] = pa.x * pa.x + pa.y * pa.y + pa.z * pa.z;
            }
            if (tid == 0) {
                sm.A[kDummy] = make_float4(1e18f, 1e18f, 1e18f, 0.f);
                sm.B[kDummy] = make_float4(0.f, 0.f, 0.f, 0.f);
                sm.C[kDummy] = make_float4(0.f, 0.f, 0.f, 0.f);
                sm.D[kDummy] = make_float2(0.f, 0.f);
                sm.P2[kDummy] = 3e36f;
            }
        }
        __syncthreads();

        if (nt > 0 && sm.cand_len[b] < 0) {
            if (half == 0)
                for (uint32_t i = tb0 + lane; i < tb0 + nt; i += 32)
                    my_pairs += direct_particle((int64_t)i, cx, cy, cz, in, cs, ce, g, k, out);
        } else if (nt > 0) {
            const uint16_t *cand = sm.cand[b];
            const int Wp = sm.cand_len[b];
            const int q = lane >> 3, t = lane & 7;
            // targets sit in the centre run (r = 4)
            const int tbase = __shfl_sync(0xffffffffu, run_off, 4) + ((int)tb0 - __shfl_sync(0xffffffffu, run_lo, 4));
            float(*acc)[kAccStride] = sm.acc[warp];
            int parked = 0;
            for (uint32_t p = half; 4 * p < nt; p += 2) {
                // quarter q works for target 4p + q; slot d of the phase-1 registers holds target
                // 4p + (q ^ d):  a = -2 T', thr = support^2 - |T'|^2 + rounding margin
                float ax[4], ay[4], az[4], th[4];
#pragma unroll
                for (int d = 0; d < 4; ++d) {
                    const uint32_t ti = 4 * p + (uint32_t)(q ^ d);
                    ax[d] = ay[d] = az[d] = 0.f;
                    th[d] = -1.f;  // |p'|^2 >= 0 > -1: an absent target accepts nothing
                    if (ti < nt) {
                        const float4 pa = sm.A[tbase + ti];
                        const float t2 = pa.x * pa.x + pa.y * pa.y + pa.z * pa.z;
                        ax[d] = -2.0f * pa.x; ay[d] = -2.0f * pa.y; az[d] = -2.0f * pa.z;
                        // margin >= 1e-6 (2|T'| + 2h)^2, the rounding bound of the expanded form
                        th[d] = k.support2 - t2 + 1e-6f * (8.0f * t2 + 3.0f * k.support2);
                    }
                }
                const uint32_t my_t = 4 * p + (uint32_t)q;
                const bool my_valid = my_t < nt;
                float4 tp = make_float4(0.f, 0.f, 0.f, 0.f), tv = tp;
                if (my_valid) { tp = sm.A[tbase + my_t]; tv = sm.B[tbase + my_t]; }
                PairAccum S;
                S.clear();
                for (int base = 0; base < Wp; base += kDrain) {
                    // ---- phase 1: bit 4 s + d of (lo | hi << 32) <- candidate chunk s, slot d -----
                    uint32_t lo = 0, hi = 0;
                    const int nch = min(kDrain, Wp - base) >> 5;
                    const uint16_t *cb = cand + base + lane;
#pragma unroll 2
                    for (int s = nch - 1; s >= 8; --s) {
                        const int j = cb[32 * s];
                        const float4 pa = sm.A[j];
                        const float p2 = sm.P2[j];
                        test_push(hi, pa, p2, ax[3], ay[3], az[3], th[3]);
                        test_push(hi, pa, p2, ax[2], ay[2], az[2], th[2]);
                        test_push(hi, pa, p2, ax[1], ay[1], az[1], th[1]);
                        test_push(hi, pa, p2, ax[0], ay[0], az[0], th[0]);
                    }
#pragma unroll 2
                    for (int s = min(nch, 8) - 1; s >= 0; --s) {
                        const int j = cb[32 * s];
                        const float4 pa = sm.A[j];
                        const float p2 = sm.P2[j];
                        test_push(lo, pa, p2, ax[3], ay[3], az[3], th[3]);
                        test_push(lo, pa, p2, ax[2], ay[2], az[2], th[2]);
                        test_push(lo, pa, p2, ax[1], ay[1], az[1], th[1]);
                        test_push(lo, pa, p2, ax[0], ay[0], az[0], th[0]);
                    }
                    // ---- every quarter collects the bits of its own target: slot d of the lanes
                    //      of quarter q ^ d -------------------------------------------------------
                    {
                        const uint32_t l1 = __shfl_xor_sync(0xffffffffu, lo, 8), h1 = __shfl_xor_sync(0xffffffffu, hi, 8);
                        const uint32_t l2 = __shfl_xor_sync(0xffffffffu, lo, 16), h2 = __shfl_xor_sync(0xffffffffu, hi, 16);
                        const uint32_t l3 = __shfl_xor_sync(0xffffffffu, lo, 24), h3 = __shfl_xor_sync(0xffffffffu, hi, 24);
                        lo = (lo & 0x11111111u) | (l1 & 0x22222222u) | (l2 & 0x44444444u) | (l3 & 0x88888888u);
                        hi = (hi & 0x11111111u) | (h1 & 0x22222222u) | (h2 & 0x44444444u) | (h3 & 0x88888888u);
                    }
                    // ---- phase 2: two pairs per lane and round; bit beta of the word being popped
                    //      <-> candidate vb + 8 (beta ^ q); lanes that ran dry evaluate the dummy
                    //      record, which contributes exactly zero ------------------------------------
                    uint32_t w = lo, w2 = hi;
                    int vb = base + t;
                    while (__any_sync(0xffffffffu, (w | w2) != 0u)) {
#pragma unroll
                        for (int u = 0; u < 2; ++u) {
                            if (w == 0u) { w = w2; w2 = 0u; vb += 256; }
                            int j = kDummy;
                            if (w != 0u) {
                                const int beta = __ffs(w) - 1;
                                w &= w - 1;
                                j = cand[vb + ((beta ^ q) << 3)];
                            }
                            const float4 pa = sm.A[j];
                            const float4 pb = sm.B[j];
                            const float4 pc = sm.C[j];
                            const float2 pd = sm.D[j];
                            const float dx = tp.x - pa.x, dy = tp.y - pa.y, dz = tp.z - pa.z;
                            const float r2 = dx * dx + dy * dy + dz * dz;
                            if (r2 < k.support2) ++my_pairs;  // exact test (phase 1 has a rounding margin)
                            const float Sj[6] = {pc.x, pc.y, pc.z, pc.w, pd.x, pd.y};
                            S.add(dx, dy, dz, r2, pa.w, pb.w, pb.x - tv.x, pb.y - tv.y, pb.z - tv.z, Sj,
                                  k.half_inv_h);
                        }
                    }
                }
                // ---- reduce the 16 sums over the quarter, park them ---------------------------
                {
                    float v[16];
                    v[0] = S.dr;
#pragma unroll
                    for (int c = 0; c < 9; ++c) v[1 + c] = S.L[c];
#pragma unroll
                    for (int c = 0; c < 3; ++c) { v[10 + c] = S.g[c]; v[13 + c] = S.a[c]; }
                    reduce8_transposed(v, t);
                    float *row = acc[parked * 4 + q];
                    const int idx = ((t & 4) << 1) + ((t & 2) << 1) + ((t & 1) << 1);
                    row[idx] = v[0];
                    row[idx + 1] = v[1];
                    if (t == 0) row[16] = __int_as_float(my_valid ? (int)(tb0 + my_t) : -1);
                }
                if (my_valid && t == 0) ++my_self;  // the self pair is not a pair (reading S15)
                ++parked;
                const bool last = 4 * (p + 2) >= nt;
                if (parked == kSlots / 4 || last) {
                    // ---- epilogue: one lane per parked target (O8, stores) --------------------
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
    if (pair_count) {
        const uint32_t tot = __reduce_add_sync(0xffffffffu, my_pairs) - __reduce_add_sync(0xffffffffu, my_self);
        if (lane == 0 && tot) atomicAdd(pair_count, (unsigned long long)tot);
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
