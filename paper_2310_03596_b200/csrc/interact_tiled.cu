// Stage 4a, main kernel: SPH interaction loops over the 27-bucket stencil ("the search
// for the neighboring particles is restricted to its bucket and to the surrounding buckets";
// steps e/f PAPER.md:24-25; "several interaction loops"; equations DESIGN.md O6-O8).
//
// Layout of the work (DESIGN.md section 6.1 gives the measurements that led here):
//  * x-fastest hashing makes the three buckets (cx-1, cx, cx+1) contiguous in the sorted arrays.
//    A CTA owns a tile of kTBX x kTBY buckets of one z-layer; its candidate window is the
//    3 (kTBY + 2) rows of kTBX + 2 buckets around it, i.e. 12 contiguous runs of the sorted arrays.
//    The window's packed records (A = x,y,z,m; B = vx,vy,vz,V; C = Sxx,Syy,Szz,Sxy; D = Sxz,Syz
//    with V = m/rho, S = sigma/rho^2, written by pack_kernel) are brought to shared memory with
//    1-D TMA bulk copies (cp.async.bulk + mbarrier), no register staging.
//  * Warp b builds the candidate table of bucket b once: the 27-bucket stencil as shared-memory
//    record offsets, every run padded so that (table position) == (record index) mod 8.
//  * Work unit = 4 consecutive targets of one bucket, dealt round-robin to the 8 warps.
//    Phase 1 (distance tests): lane l tests candidate 32 s + l of the table against the 4 targets
//    held in registers (one 128-bit shared load per 128 tests, expanded-form test in tile-local
//    coordinates) and records the outcome as one bit per target; 3 shuffles give quarter-warp q
//    the complete mask of target q, lane t owning the table positions = t (mod 8).
//  * Compaction: every lane pops its bits into the target's neighbour list in shared memory
//    (positions from an 8-lane prefix sum), so the list is grouped by record index mod 8.
//  * Phase 2 (pair arithmetic): lane t of the quarter walks list[t R .. (t + 1) R), R =
//    ceil(len / 8): all lanes carry the same number of pairs (the v3 kernel ran at 61 % lane
//    efficiency because a lane was tied to its residue class) and the 8 record gathers of a
//    quarter-warp still fall mostly into 8 distinct 16-byte bank groups.  The 16 partial sums
//    are reduced over the 8 lanes, parked in shared memory, and a lane-per-target epilogue forms
//    the rates (O8) and stores them.
//  * No pair is skipped or evaluated twice: the self pair is accepted like any other (it
//    contributes exactly zero because x_ii = 0) and is subtracted from pair_count.
// Tiles whose window does not fit the shared-memory budget, buckets whose table overflows and
// targets with more than kListCap neighbours fall back to the direct walk.
#include "sph_internal.cuh"
#include "interact_math.cuh"

namespace sphb {

constexpr int kTBX = 4, kTBY = 2;      // buckets per tile along x and y
constexpr int kNB = kTBX * kTBY;       // target buckets per tile
constexpr int kRowsY = kTBY + 2;       // window rows along y
constexpr int kRuns = 3 * kRowsY;      // contiguous runs of the window
constexpr int kTW = 8;                 // warps per CTA (== kNB: warp b builds the table of bucket b)
constexpr int kCap = 1472;             // window records held in shared memory
constexpr int kCandCap = 640;          // candidate-table entries per bucket
constexpr int kDrain = 512;            // candidates per phase-1 / compaction round trip (16 x 32)
constexpr int kListCap = 128;          // neighbour-list entries per target
constexpr int kSlots = 8;              // targets parked per warp before the epilogue
constexpr int kAccStride = 17;         // 16 sums + 1 pad word (bank-conflict free)
constexpr int kDummy = kCap;           // record index of the far-away dummy candidate
static_assert(kTW == kNB, "warp b builds the candidate table of bucket b");
static_assert((kCap + 1) * 8 < 65536, "table entries are record index * 8 in 16 bits");

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
    uint16_t cand[kNB][kCandCap];      // record index * 8
    uint16_t list[kTW][4][kListCap];   // record index * 8, per warp and quarter
    int cand_len[kNB];        // padded table length (multiple of 32), -1 = overflow -> direct walk
    int bkt_nt[kNB];          // targets in bucket b
    int bkt_tsm[kNB];         // shared-memory record index of its first target
    uint32_t bkt_tb0[kNB];    // sorted index of its first target
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

// byte-offset views of the record arrays (table and list entries are record index * 8)
__device__ __forceinline__ float4 ld_rec16(const float4 *base, uint32_t e8)
{
    return *reinterpret_cast<const float4 *>(reinterpret_cast<const char *>(base) + 2u * e8);
}
__device__ __forceinline__ float2 ld_rec8(const float2 *base, uint32_t e8)
{
    return *reinterpret_cast<const float2 *>(reinterpret_cast<const char *>(base) + e8);
}
__device__ __forceinline__ float ld_rec4(const float *base, uint32_t e8)
{
    return *reinterpret_cast<const float *>(reinterpret_cast<const char *>(base) + (e8 >> 1));
}

template <bool kCount>
__global__ void __launch_bounds__(kTW * 32, 2)
interact_tiled_kernel(Packed rec, InteractIn in, const uint32_t *__restrict__ cs,
                      const uint32_t *__restrict__ ce, Grid g, Consts k, InteractOut out,
                      unsigned long long *pair_count, int tiles_x, int tiles_y)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TileSmem &sm = *reinterpret_cast<TileSmem *>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tx = blockIdx.x % tiles_x, tyz = blockIdx.x / tiles_x;
    const int ty = tyz % tiles_y, cz = tyz / tiles_y;
    const int cx0 = tx * kTBX, cy0 = ty * kTBY;
    const int nbx = min(kTBX, g.nx - cx0), nby = min(kTBY, g.ny - cy0);

    // ---- the 12 runs of the tile's window: lane r of every warp describes run r ---------------
    // run r: window row iy = r % kRowsY (grid row cy0 - 1 + iy), layer iz = r / kRowsY (cz - 1 + iz)
    const int ry = cy0 - 1 + (lane % kRowsY), rz = cz - 1 + (lane / kRowsY);
    const bool row_ok = lane < kRuns && ry >= 0 && ry < g.ny && rz >= 0 && rz < g.nz;
    const uint32_t rrow = row_ok ? (uint32_t)g.nx * ((uint32_t)ry + (uint32_t)g.ny * (uint32_t)rz) : 0u;
    int run_lo = 0, run_len = 0;  // first sorted index copied (even) and number of records
    if (row_ok) {
        const int lo = (int)cs[rrow + max(cx0 - 1, 0)], hi = (int)ce[rrow + min(cx0 + nbx, g.nx - 1)];
        if (hi > lo) { run_lo = lo & ~1; run_len = hi - run_lo; }
    }
    const int run_cnt = (run_len + 1) & ~1;  // even record count: keeps every offset 16-byte aligned
    int run_off = run_cnt;                   // exclusive prefix over lanes 0..kRuns-1
#pragma unroll
    for (int o = 1; o < 16; o <<= 1) {
        const int x = __shfl_up_sync(0xffffffffu, run_off, o);
        if (lane >= o) run_off += x;
    }
    const int total = __shfl_sync(0xffffffffu, run_off, kRuns - 1);
    run_off -= run_cnt;

    // ---- bucket b = warp: targets, work units ---------------------------------------------------
    const int bx = warp % kTBX, by = warp / kTBX;
    const int cxb = cx0 + bx, cyb = cy0 + by;
    const bool b_ok = bx < nbx && by < nby;
    const int rc = (by + 1) + kRowsY;        // the run holding the targets of bucket b
    uint32_t tb0 = 0;
    int nt = 0;
    if (b_ok) {
        const uint32_t c = (uint32_t)cxb + (uint32_t)g.nx * ((uint32_t)cyb + (uint32_t)g.ny * (uint32_t)cz);
        tb0 = cs[c];
        nt = (int)(ce[c] - tb0);
    }
    if (__syncthreads_or(nt) == 0) return;   // no target particle in this tile

    if (tid == 0) {
        mbar_init(&sm.bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    uint32_t my_pairs = 0, my_self = 0;
    if (total > kCap) {
        // window too large for shared memory (very dense region): direct walk, warp = bucket
        for (int i = lane; i < nt; i += 32)
            my_pairs += direct_particle((int64_t)tb0 + i, cxb, cyb, cz, in, cs, ce, g, k, out);
    } else {
        __syncthreads();  // mbarrier initialised before the copies are issued against it
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
        // ---- candidate table of bucket b: its 27-bucket stencil as record offsets, every run
        //      shifted so that (table position) == (record index) mod 8.  Lane r' < 9 looks up
        //      stencil row r' = (dy + 1) + 3 (dz + 1), i.e. window run (by + r' % 3) + kRowsY (r' / 3).
        {
            int s_r = 0, len_r = 0;
            if (nt > 0 && lane < 9) {
                const int wr = (by + lane % 3) + kRowsY * (lane / 3);
                const int y = cy0 - 1 + (wr % kRowsY), z = cz - 1 + (wr / kRowsY);
                if (y >= 0 && y < g.ny && z >= 0 && z < g.nz) {
                    const uint32_t row = (uint32_t)g.nx * ((uint32_t)y + (uint32_t)g.ny * (uint32_t)z);
                    const int sg = (int)cs[row + max(cxb - 1, 0)], eg = (int)ce[row + min(cxb + 1, g.nx - 1)];
                    len_r = max(eg - sg, 0);
                    // offset of the stencil row inside window run wr (held by lane wr)
                    s_r = sg;
                }
            }
            // window run descriptors of the 9 rows (every lane fetches the one of its row)
            const int wr_l = (lane < 9) ? (by + lane % 3) + kRowsY * (lane / 3) : 0;
            const int w_off = __shfl_sync(0xffffffffu, run_off, wr_l);
            const int w_lo = __shfl_sync(0xffffffffu, run_lo, wr_l);
            s_r = w_off + (s_r - w_lo);
            uint16_t *cand = sm.cand[warp];
            int W = 0;
            if (nt > 0) {
#pragma unroll
                for (int r = 0; r < 9; ++r) {
                    const int s = __shfl_sync(0xffffffffu, s_r, r), len = __shfl_sync(0xffffffffu, len_r, r);
                    if (len == 0) continue;
                    const int pad = (s - W) & 7;
                    if (W + pad + len <= kCandCap - 32) {
                        uint16_t *cw = cand + W + pad + lane;
                        const int e0 = (s + lane) * 8;
                        if (lane < pad) cand[W + lane] = (uint16_t)(kDummy * 8);
                        if (lane < len) cw[0] = (uint16_t)e0;
                        if (lane + 32 < len) cw[32] = (uint16_t)(e0 + 256);
                        for (int o = lane + 64; o < len; o += 32) cw[o - lane] = (uint16_t)(e0 + 8 * (o - lane));
                    }
                    W += pad + len;
                }
                const bool overflow = W > kCandCap - 32;
                const int Wp = (W + 31) & ~31;
                if (!overflow && W + lane < Wp) cand[W + lane] = (uint16_t)(kDummy * 8);
                if (lane == 0) sm.cand_len[warp] = overflow ? -1 : Wp;
            }
            // shared-memory index of the first target: it sits in window run rc
            const int t_off = __shfl_sync(0xffffffffu, run_off, rc), t_lo = __shfl_sync(0xffffffffu, run_lo, rc);
            if (lane == 0) {
                sm.bkt_nt[warp] = nt;
                sm.bkt_tb0[warp] = tb0;
                sm.bkt_tsm[warp] = t_off + ((int)tb0 - t_lo);
            }
        }
        // ---- wait for the window, shift it to tile-local coordinates, form |p'|^2 ---------------
        mbar_wait(&sm.bar, 0);
        {
            const float edge = 1.0f / g.inv_edge;
            const float ox = g.ox + ((float)cx0 + 0.5f * kTBX) * edge, oy = g.oy + ((float)cy0 + 0.5f * kTBY) * edge,
                        oz = g.oz + ((float)cz + 0.5f) * edge;
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
        __syncthreads();  // window shifted, tables and bucket records visible to every warp

        // a bucket whose table overflowed is walked directly by its own warp
        if (nt > 0 && sm.cand_len[warp] < 0)
            for (int i = lane; i < nt; i += 32)
                my_pairs += direct_particle((int64_t)tb0 + i, cxb, cyb, cz, in, cs, ce, g, k, out);

        // ---- work units: lane b < kNB keeps the record of bucket b -----------------------------
        int l_nt = 0, l_tsm = 0, l_wp = 0, l_ng = 0;
        uint32_t l_tb0 = 0;
        if (lane < kNB) {
            l_nt = sm.bkt_nt[lane];
            l_tsm = sm.bkt_tsm[lane];
            l_tb0 = sm.bkt_tb0[lane];
            l_wp = sm.cand_len[lane];
            l_ng = (l_nt > 0 && l_wp > 0) ? (l_nt + 3) >> 2 : 0;
        }
        int l_gend = l_ng;  // inclusive prefix over the buckets
#pragma unroll
        for (int o = 1; o < kNB; o <<= 1) {
            const int x = __shfl_up_sync(0xffffffffu, l_gend, o);
            if (lane >= o) l_gend += x;
        }
        const int NG = __shfl_sync(0xffffffffu, l_gend, kNB - 1);

        const int q = lane >> 3, t = lane & 7;
        float(*acc)[kAccStride] = sm.acc[warp];
        uint16_t *lst = sm.list[warp][q];
        int parked = 0;
        for (int gi = warp; gi < NG; gi += kTW) {
            // bucket of work unit gi = number of buckets that end at or before it
            const int b = __popc(__ballot_sync(0xffffffffu, lane < kNB && l_gend <= gi));
            const int p = gi - (__shfl_sync(0xffffffffu, l_gend, b) - __shfl_sync(0xffffffffu, l_ng, b));
            const int bnt = __shfl_sync(0xffffffffu, l_nt, b);
            const int tbase = __shfl_sync(0xffffffffu, l_tsm, b);
            const uint32_t btb0 = __shfl_sync(0xffffffffu, l_tb0, b);
            const int Wp = __shfl_sync(0xffffffffu, l_wp, b);
            const uint16_t *cand = sm.cand[b];

            // quarter q works for target 4p + q; slot d of the phase-1 registers holds target
            // 4p + (q ^ d):  a = -2 T', thr = support^2 - |T'|^2 + rounding margin
            const int my_t = 4 * p + q;
            const bool my_valid = my_t < bnt;
            float4 tp = make_float4(0.f, 0.f, 0.f, 0.f);
            float ax[4], ay[4], az[4], th[4];
            ax[0] = ay[0] = az[0] = 0.f;
            th[0] = -1.f;  // |p'|^2 >= 0 > -1: an absent target accepts nothing
            if (my_valid) {
                tp = sm.A[tbase + my_t];
                const float t2 = tp.x * tp.x + tp.y * tp.y + tp.z * tp.z;
                ax[0] = -2.0f * tp.x; ay[0] = -2.0f * tp.y; az[0] = -2.0f * tp.z;
                // margin >= 1e-6 (2|T'| + 2h)^2, the rounding bound of the expanded form
                th[0] = k.support2 - t2 + 1e-6f * (8.0f * t2 + 3.0f * k.support2);
            }
#pragma unroll
            for (int d = 1; d < 4; ++d) {
                ax[d] = __shfl_xor_sync(0xffffffffu, ax[0], 8 * d);
                ay[d] = __shfl_xor_sync(0xffffffffu, ay[0], 8 * d);
                az[d] = __shfl_xor_sync(0xffffffffu, az[0], 8 * d);
                th[d] = __shfl_xor_sync(0xffffffffu, th[0], 8 * d);
            }

            // ---- phase 1 + compaction, kDrain table positions at a time -----------------------
            int len = 0;          // entries in this quarter's list (uniform over its 8 lanes)
            bool ovf = false;
            for (int base = 0; base < Wp; base += kDrain) {
                // bit 4 s + d of (lo | hi << 32) <- candidate chunk s, slot d
                uint32_t lo = 0, hi = 0;
                const int nch = min(kDrain, Wp - base) >> 5;
                const uint16_t *cb = cand + base + lane;
#pragma unroll 2
                for (int s = nch - 1; s >= 8; --s) {
                    const uint32_t e = cb[32 * s];
                    const float4 pa = ld_rec16(sm.A, e);
                    const float p2 = ld_rec4(sm.P2, e);
                    test_push(hi, pa, p2, ax[3], ay[3], az[3], th[3]);
                    test_push(hi, pa, p2, ax[2], ay[2], az[2], th[2]);
                    test_push(hi, pa, p2, ax[1], ay[1], az[1], th[1]);
                    test_push(hi, pa, p2, ax[0], ay[0], az[0], th[0]);
                }
#pragma unroll 2
                for (int s = min(nch, 8) - 1; s >= 0; --s) {
                    const uint32_t e = cb[32 * s];
                    const float4 pa = ld_rec16(sm.A, e);
                    const float p2 = ld_rec4(sm.P2, e);
                    test_push(lo, pa, p2, ax[3], ay[3], az[3], th[3]);
                    test_push(lo, pa, p2, ax[2], ay[2], az[2], th[2]);
                    test_push(lo, pa, p2, ax[1], ay[1], az[1], th[1]);
                    test_push(lo, pa, p2, ax[0], ay[0], az[0], th[0]);
                }
                // every quarter collects the bits of its own target: slot d of the lanes of
                // quarter q ^ d.  Afterwards bit beta of lo <-> table position
                // base + t + 8 (beta ^ q), of hi <-> the same + 256.
                {
                    const uint32_t l1 = __shfl_xor_sync(0xffffffffu, lo, 8), h1 = __shfl_xor_sync(0xffffffffu, hi, 8);
                    const uint32_t l2 = __shfl_xor_sync(0xffffffffu, lo, 16), h2 = __shfl_xor_sync(0xffffffffu, hi, 16);
                    const uint32_t l3 = __shfl_xor_sync(0xffffffffu, lo, 24), h3 = __shfl_xor_sync(0xffffffffu, hi, 24);
                    lo = (lo & 0x11111111u) | (l1 & 0x22222222u) | (l2 & 0x44444444u) | (l3 & 0x88888888u);
                    hi = (hi & 0x11111111u) | (h1 & 0x22222222u) | (h2 & 0x44444444u) | (h3 & 0x88888888u);
                }
                // ---- compaction: 8-lane prefix sum of the bit counts, then every lane pops its
                //      bits into list[pos ..) -----------------------------------------------------
                const int c = __popc(lo) + __popc(hi);
                int inc = c;
#pragma unroll
                for (int o = 1; o < 8; o <<= 1) {
                    const int x = __shfl_up_sync(0xffffffffu, inc, o, 8);
                    if (t >= o) inc += x;
                }
                const int tot = __shfl_sync(0xffffffffu, inc, 7, 8);
                if (__any_sync(0xffffffffu, len + tot > kListCap)) { ovf = true; break; }
                uint16_t *lw = lst + (len + inc - c);
                len += tot;
                const uint16_t *cq = cand + base + t;
                uint32_t w = lo, w2 = hi;
                while (w | w2) {
                    if (w == 0u) { w = w2; w2 = 0u; cq += 256; }
                    const int beta = 31 - __clz(w);
                    w ^= 1u << beta;
                    *lw++ = cq[(beta ^ q) << 3];
                }
            }
            __syncwarp();
            if (ovf) {
                // a target with more than kListCap neighbours (very dense spot): direct walk
                if (lane < 4 && 4 * p + lane < bnt)
                    my_pairs += direct_particle((int64_t)btb0 + 4 * p + lane, cx0 + b % kTBX, cy0 + b / kTBX, cz,
                                                in, cs, ce, g, k, out);
                continue;
            }

            // ---- phase 2: lane t walks list[t R .. (t + 1) R), two pairs per round; lanes past
            //      the end evaluate the dummy record, which contributes exactly zero -------------
            float4 tv = make_float4(0.f, 0.f, 0.f, 0.f);
            if (my_valid) tv = sm.B[tbase + my_t];
            PairAccum S;
            S.clear();
            {
                const int R = (len + 7) >> 3;
                int Rmax = max(R, __shfl_xor_sync(0xffffffffu, R, 8));
                Rmax = max(Rmax, __shfl_xor_sync(0xffffffffu, Rmax, 16));
                const int p0 = t * R;
                const int mine = max(min(R, len - p0), 0);   // entries this lane owns
                const uint16_t *lp = lst + p0;
                auto eval = [&](uint32_t e) {
                    const float4 pa = ld_rec16(sm.A, e);
                    const float4 pb = ld_rec16(sm.B, e);
                    const float4 pc = ld_rec16(sm.C, e);
                    const float2 pd = ld_rec8(sm.D, e);
                    const float dx = tp.x - pa.x, dy = tp.y - pa.y, dz = tp.z - pa.z;
                    const float r2 = dx * dx + dy * dy + dz * dz;
                    if (kCount && r2 < k.support2) ++my_pairs;  // exact test (phase 1 has a rounding margin)
                    const float Sj[6] = {pc.x, pc.y, pc.z, pc.w, pd.x, pd.y};
                    S.add(dx, dy, dz, r2, pa.w, pb.w, pb.x - tv.x, pb.y - tv.y, pb.z - tv.z, Sj, k.half_inv_h);
                };
                int r = 0;
                for (; r + 2 <= Rmax; r += 2) {
                    uint32_t e0 = (uint32_t)kDummy * 8u, e1 = e0;
                    if (r < mine) e0 = lp[r];
                    if (r + 1 < mine) e1 = lp[r + 1];
                    eval(e0);
                    eval(e1);
                }
                if (r < Rmax) {
                    uint32_t e0 = (uint32_t)kDummy * 8u;
                    if (r < mine) e0 = lp[r];
                    eval(e0);
                }
            }
            // ---- reduce the 16 sums over the quarter, park them -------------------------------
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
                if (t == 0) row[16] = __int_as_float(my_valid ? (int)(btb0 + my_t) : -1);
            }
            if (my_valid && t == 0) ++my_self;  // the self pair is not a pair (reading S15)
            ++parked;
            if (parked == kSlots / 4 || gi + kTW >= NG) {
                // ---- epilogue: one lane per parked target (O8, stores) ------------------------
                __syncwarp();
                if (lane < parked * 4) {
                    const float *row = acc[lane];
                    const int i = __float_as_int(row[16]);
                    if (i >= 0) {
                        PairAccum Rr;
                        Rr.dr = row[0];
#pragma unroll
                        for (int c = 0; c < 9; ++c) Rr.L[c] = row[1 + c];
#pragma unroll
                        for (int c = 0; c < 3; ++c) { Rr.g[c] = row[10 + c]; Rr.a[c] = row[13 + c]; }
                        float si[6];
#pragma unroll
                        for (int c = 0; c < 6; ++c) si[c] = in.sig[c][i];
                        finish_particle(Rr, si, in.velr[i].w, k, out, (int64_t)i);
                    }
                }
                __syncwarp();
                parked = 0;
            }
        }
        // a warp whose last work unit overflowed may still hold parked targets
        if (parked > 0) {
            __syncwarp();
            if (lane < parked * 4) {
                const float *row = acc[lane];
                const int i = __float_as_int(row[16]);
                if (i >= 0) {
                    PairAccum Rr;
                    Rr.dr = row[0];
#pragma unroll
                    for (int c = 0; c < 9; ++c) Rr.L[c] = row[1 + c];
#pragma unroll
                    for (int c = 0; c < 3; ++c) { Rr.g[c] = row[10 + c]; Rr.a[c] = row[13 + c]; }
                    float si[6];
#pragma unroll
                    for (int c = 0; c < 6; ++c) si[c] = in.sig[c][i];
                    finish_particle(Rr, si, in.velr[i].w, k, out, (int64_t)i);
                }
            }
        }
    }
    if (kCount) {
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
        SPH_CUDA_TRY(c, cudaFuncSetAttribute(interact_tiled_kernel<true>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        SPH_CUDA_TRY(c, cudaFuncSetAttribute(interact_tiled_kernel<false>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        attr_set = true;
    }
    const int tiles_x = (c->grid.nx + kTBX - 1) / kTBX, tiles_y = (c->grid.ny + kTBY - 1) / kTBY;
    const int64_t tiles = (int64_t)tiles_x * tiles_y * c->grid.nz;
    if (tiles > 0x7fffffffll) return SPH_EINVAL;
    if (pair_count)
        interact_tiled_kernel<true><<<(unsigned)tiles, kTW * 32, smem, c->stream>>>(
            rec, in, cs, ce, c->grid, c->consts, out, pair_count, tiles_x, tiles_y);
    else
        interact_tiled_kernel<false><<<(unsigned)tiles, kTW * 32, smem, c->stream>>>(
            rec, in, cs, ce, c->grid, c->consts, out, pair_count, tiles_x, tiles_y);
    SPH_CHECK_LAUNCH(c);
    return SPH_OK;
}

}  // namespace sphb
