// Stage 4a, main kernel: SPH interaction loops over the 27-bucket stencil ("the search
// for the neighboring particles is restricted to its bucket and to the surrounding buckets";
// steps e/f PAPER.md:24-25; "several interaction loops"; equations DESIGN.md O6-O8).
//
// Layout of the work (DESIGN.md section 6.1 gives the measurements that led here):
//  * x-fastest hashing makes the three buckets (cx-1, cx, cx+1) contiguous in the sorted arrays.
//    A CTA owns a tile of kTBX x kTBY buckets of one z-layer; its candidate window is the
//    3 (kTBY + 2) rows of kTBX + 2 buckets around it, i.e. 12 contiguous runs of the sorted arrays.
//    The window's packed records, four 16-byte parts per particle (A = x,y,z,m -> after the shift
//    x',y',z',|p'|^2; B = vx,vy,vz,Szz; C = Sxx,Sxy,Sxy,Syy; D = Sxz,Syz,m,V with V = m/rho,
//    S = sigma/rho^2; B, C, D written by the reorder pass inside sph_step, else by pack_kernel, in
//    the pair layout of PairAccum2) are brought
//    to shared memory with 1-D TMA bulk copies (cp.async.bulk + mbarrier), no register staging.
//  * Warp b builds the candidate table of bucket b once: the 27-bucket stencil as shared-memory
//    record offsets, every run padded so that (table position) == (record index) mod 8.
//  * Work unit = 4 consecutive targets of one bucket, dealt round-robin to the 12 warps.
//    Phase 1 (distance tests): lane l tests candidate 32 s + l of the table against the 4 targets
//    held in registers as two fp32 pairs (one 128-bit shared load per 128 tests; expanded-form
//    test in tile-local coordinates, 4 FFMA2 per 2 tests) and records the outcome as one bit per
//    target; 3 shuffles give quarter-warp q the complete mask of target q, lane t owning the table
//    positions = t (mod 8).  The whole table (up to 640 positions) is tested before one drain.
//  * Phase 2 (pair arithmetic): lane t of quarter q pops the set bits of its own mask words and
//    evaluates those pairs directly, two per round -- no neighbour list, no compaction pass.
//    Because lane t only ever gathers records whose index is = t (mod 8), the 8 128-bit gathers
//    of a quarter-warp always hit 8 distinct bank groups: the gathers are conflict-free by
//    construction (the list-based v4 / v5 variants measured 7-8 wavefronts per gather
//    instruction against the ideal 4, profiles/r01c).  The price is lane imbalance (the warp runs
//    max-over-lanes rounds; idle lanes evaluate the dummy record of their class), paid on a pair
//    body that is packed (PairAccum2: FFMA2 / FMUL2 / FADD2, 30 issue slots per pair instead
//    of 46).  The 16 partial sums are reduced over the 8 lanes, parked in shared memory, and a
//    lane-per-target epilogue forms the rates (O8), stores them if asked to, and -- inside
//    sph_step -- integrates the particle (O9) and scatters it to id order through perm.
//  * No pair is skipped or evaluated twice: the self pair is accepted like any other (it
//    contributes exactly zero because x_ii = 0) and is subtracted from pair_count.
// Tiles whose window does not fit the shared-memory budget and buckets whose table overflows
// fall back to the direct walk.
#include "sph_internal.cuh"
#include "interact_math.cuh"

namespace sphb {

constexpr int kTBX = 4, kTBY = 2;      // buckets per tile along x and y
constexpr int kNB = kTBX * kTBY;       // target buckets per tile
constexpr int kRowsY = kTBY + 2;       // window rows along y
constexpr int kRuns = 3 * kRowsY;      // contiguous runs of the window
constexpr int kTW = 12;                // warps per CTA (warp b < kNB builds the table of bucket b)
constexpr int kCap = 1496;             // window records held in shared memory (64 B each)
constexpr int kCandCap = 640;          // candidate-table entries per bucket
constexpr int kSlots = 8;              // targets parked per warp before the epilogue
constexpr int kAccStride = 19;         // 16 sums, particle index, record index, 1 pad word (odd: conflict-free)
constexpr int kDummy = kCap;           // kDummy + c: far-away dummy candidate of bank class c = 0..7
static_assert(kTW >= kNB, "warp b builds the candidate table of bucket b");
static_assert((kCap + 8) * 16 < 65536 && kCap % 8 == 0, "table entries are record index * 16 in 16 bits");
static_assert(kCandCap == 640, "three mask words cover 20 chunks of 32 table positions");

struct Packed {
    const float4 *A;                   // sorted posm (x, y, z, m)
    float4 *B;                         // vx, vy, vz, Szz
    float4 *C;                         // Sxx, Sxy, Sxy, Syy     (S = sigma / rho^2)
    float4 *D;                         // Sxz, Syz, m, V
};

// ------------------------------------------------------------------------------------ pack
__global__ void __launch_bounds__(256)
pack_kernel(int64_t n, InteractIn in, float4 *__restrict__ B, float4 *__restrict__ C,
            float4 *__restrict__ D)
{
    // (NEXT-4: with per-particle smoothing lengths C.z carries h instead of the second Sxy)
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const float m = in.posm[k].w;
    const float4 v = in.velr[k];
    const float inv_rho = 1.0f / v.w;
    const float ir2 = inv_rho * inv_rho;
    const float sxy = in.sig[3][k] * ir2;
    B[k] = make_float4(v.x, v.y, v.z, in.sig[2][k] * ir2);
    C[k] = make_float4(in.sig[0][k] * ir2, sxy, in.h ? in.h[k] : sxy, in.sig[1][k] * ir2);
    D[k] = make_float4(in.sig[4][k] * ir2, in.sig[5][k] * ir2, m, m * inv_rho);
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
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity), "r"(0x989680u)   // suspend-time hint: the warp sleeps until the phase completes
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
    float4 A[kCap + 8];       // x - ox, y - oy, z - oz (tile-local coordinates), |p'|^2
    float4 B[kCap + 8];
    float4 C[kCap + 8];
    float4 D[kCap + 8];
    float acc[kTW][kSlots][kAccStride];
    uint16_t cand[kNB][kCandCap];      // record index * 16 (byte offset into A / B / C / D)
    int cand_len[kNB];        // padded table length (multiple of 32), -1 = overflow -> direct walk
    int bkt_nt[kNB];          // targets in bucket b
    int bkt_tsm[kNB];         // shared-memory record index of its first target
    uint32_t bkt_tb0[kNB];    // sorted index of its first target
    uint64_t bar;
    uint8_t own[kCap + 8];    // owner label of every window record (split passes only, NEXT-3)
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

// Phase-1 tests of one candidate against two targets held as an fp32 pair:
// acc = -thr + a . p' + |p'|^2 per target (a = -2 T', expanded form), the two sign bits are
// shifted into the mask (1 = inside), the higher slot first.
__device__ __forceinline__ void test_push2(uint32_t &mask, const float4 &pa, f32x2 ax, f32x2 ay, f32x2 az,
                                           f32x2 nth)
{
    f32x2 acc = fma2(bc(pa.x), ax, nth);
    acc = fma2(bc(pa.y), ay, acc);
    acc = fma2(bc(pa.z), az, acc);
    acc = add2(acc, bc(pa.w));
    mask = __funnelshift_l(__float_as_uint(hi_of(acc)), mask, 1);
    mask = __funnelshift_l(__float_as_uint(lo_of(acc)), mask, 1);
}

// byte-offset view of the record arrays (table entries are record index * 16)
__device__ __forceinline__ float4 ld_rec(const float4 *base, uint32_t e16)
{
    return *reinterpret_cast<const float4 *>(reinterpret_cast<const char *>(base) + e16);
}

template <bool kCount, int kMode, bool kVarH>
__global__ void __launch_bounds__(kTW * 32, 2)
interact_tiled_kernel(Packed rec, InteractIn in, const uint32_t *__restrict__ cs,
                      const uint32_t *__restrict__ ce, Grid g, Consts k, InteractOut out,
                      unsigned long long *pair_count, int tiles_x, int tiles_y, InteractOut out_f)
{
    // kMode == kPassBoth: step e goes to `out`, step f to `out_f`; pair_count[0] / [1] likewise
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TileSmem &sm = *reinterpret_cast<TileSmem *>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // tile order: x fastest, then z, then y -- the three z-layers of a window are then touched by
    // consecutive waves of CTAs (reuse distance one tile row) and the y-neighbours one slab of
    // tiles_x * nz tiles later, which the 126 MB L2 holds; with z outermost a record came back
    // from DRAM ~3 times (12.4 GB read at 64 M particles against 4.1 GB of records)
    const int tx = blockIdx.x % tiles_x, tyz = blockIdx.x / tiles_x;
    const int cz = tyz % g.nz, ty = tyz / g.nz;
    const int cx0 = tx * kTBX, cy0 = ty * kTBY;
    const int nbx = min(kTBX, g.nx - cx0), nby = min(kTBY, g.ny - cy0);

    // ---- the 12 runs of the tile's window: lane r of every warp describes run r ---------------
    // run r: window row iy = r % kRowsY (grid row cy0 - 1 + iy), layer iz = r / kRowsY (cz - 1 + iz)
    const int ry = cy0 - 1 + (lane % kRowsY), rz = cz - 1 + (lane / kRowsY);
    const bool row_ok = lane < kRuns && ry >= 0 && ry < g.ny && rz >= 0 && rz < g.nz;
    const uint32_t rrow = row_ok ? (uint32_t)g.nx * ((uint32_t)ry + (uint32_t)g.ny * (uint32_t)rz) : 0u;
    int run_lo = 0, run_len = 0;  // first sorted index copied and number of records (16-byte parts)
    if (row_ok) {
        const int lo = (int)cs[rrow + max(cx0 - 1, 0)], hi = (int)ce[rrow + min(cx0 + nbx, g.nx - 1)];
        if (hi > lo) { run_lo = lo; run_len = hi - lo; }
    }
    // stencil rows of bucket b = warp (candidate table below): lane r' < 9 looks up stencil row
    // r' = (dy + 1) + 3 (dz + 1).  Issued here so that every global load of the tile set-up is in
    // flight at once (one round trip instead of three).
    int rowq_sg = 0, rowq_len = 0;
    {
        const int bx_ = warp % kTBX, by_ = warp / kTBX;
        if (lane < 9 && bx_ < nbx && by_ < nby) {
            const int wr = (by_ + lane % 3) + kRowsY * (lane / 3);
            const int y = cy0 - 1 + (wr % kRowsY), z = cz - 1 + (wr / kRowsY);
            if (y >= 0 && y < g.ny && z >= 0 && z < g.nz) {
                const uint32_t row = (uint32_t)g.nx * ((uint32_t)y + (uint32_t)g.ny * (uint32_t)z);
                const int cxb_ = cx0 + bx_;
                rowq_sg = (int)cs[row + max(cxb_ - 1, 0)];
                rowq_len = max((int)ce[row + min(cxb_ + 1, g.nx - 1)] - rowq_sg, 0);
            }
        }
    }
    const int run_cnt = run_len;
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
    uint32_t my_pairs = 0, my_self = 0, my_pairs_f = 0;
    if (total > kCap) {
        // window too large for shared memory (very dense region): direct walk, warp = bucket
        for (int i = lane; i < nt; i += 32) {
            if (kMode == kPassBoth) {
                my_pairs += direct_particle((int64_t)tb0 + i, cxb, cyb, cz, in, cs, ce, g, k, out, kPassLocal);
                my_pairs_f += direct_particle((int64_t)tb0 + i, cxb, cyb, cz, in, cs, ce, g, k, out_f, kPassRemote);
            } else {
                my_pairs += direct_particle((int64_t)tb0 + i, cxb, cyb, cz, in, cs, ce, g, k, out, kMode);
            }
        }
    } else {
        __syncthreads();  // mbarrier initialised before the copies are issued against it
        if (warp == 0) {
            const uint32_t bytes = __reduce_add_sync(0xffffffffu, (uint32_t)run_len * 64u);
            if (lane == 0) mbar_expect_tx(&sm.bar, bytes);
            __syncwarp();
            if (run_len > 0) {
                tma_load_1d(&sm.A[run_off], rec.A + run_lo, (uint32_t)run_len * 16u, &sm.bar);
                tma_load_1d(&sm.B[run_off], rec.B + run_lo, (uint32_t)run_len * 16u, &sm.bar);
                tma_load_1d(&sm.C[run_off], rec.C + run_lo, (uint32_t)run_len * 16u, &sm.bar);
                tma_load_1d(&sm.D[run_off], rec.D + run_lo, (uint32_t)run_len * 16u, &sm.bar);
            }
        }
        // ---- candidate table of bucket b: its 27-bucket stencil as record offsets, every run
        //      shifted so that (table position) == (record index) mod 8.  Lane r' < 9 looks up
        //      stencil row r' = (dy + 1) + 3 (dz + 1), i.e. window run (by + r' % 3) + kRowsY (r' / 3).
        {
            int s_r = rowq_sg;   // (loaded at the top of the kernel, together with the run descriptors)
            const int len_r = nt > 0 ? rowq_len : 0;
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
                        const int e0 = (s + lane) * 16;
                        if (lane < pad) cand[W + lane] = (uint16_t)((kDummy + ((W + lane) & 7)) * 16);
                        if (lane < len) cw[0] = (uint16_t)e0;
                        if (lane + 32 < len) cw[32] = (uint16_t)(e0 + 512);
                        for (int o = lane + 64; o < len; o += 32) cw[o - lane] = (uint16_t)(e0 + 16 * (o - lane));
                    }
                    W += pad + len;
                }
                const bool overflow = W > kCandCap - 32;
                const int Wp = (W + 31) & ~31;
                if (!overflow && W + lane < Wp) cand[W + lane] = (uint16_t)((kDummy + ((W + lane) & 7)) * 16);
                if (lane == 0) sm.cand_len[warp] = overflow ? -1 : Wp;
            }
            // shared-memory index of the first target: it sits in window run rc
            const int t_off = __shfl_sync(0xffffffffu, run_off, rc), t_lo = __shfl_sync(0xffffffffu, run_lo, rc);
            if (lane == 0 && warp < kNB) {
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
                pa.w = pa.x * pa.x + pa.y * pa.y + pa.z * pa.z;   // the mass travels in D.z
                sm.A[j] = pa;
            }
            if (kMode != kPassAll) {
                // owner labels of the window records, run by run (lane r of every warp describes run r)
                for (int r = 0; r < kRuns; ++r) {
                    const int lo = __shfl_sync(0xffffffffu, run_lo, r), off = __shfl_sync(0xffffffffu, run_off, r);
                    const int len = __shfl_sync(0xffffffffu, run_len, r);
                    for (int i = tid; i < len; i += kTW * 32) sm.own[off + i] = (uint8_t)in.owner[lo + i];
                }
            }
            if (tid < 8) {
                sm.A[kDummy + tid] = make_float4(1e18f, 1e18f, 1e18f, 3e36f);
                sm.B[kDummy + tid] = make_float4(0.f, 0.f, 0.f, 0.f);
                sm.C[kDummy + tid] = make_float4(0.f, 0.f, kVarH ? 1.f : 0.f, 0.f);
                sm.D[kDummy + tid] = make_float4(0.f, 0.f, 0.f, 0.f);
            }
        }
        __syncthreads();  // window shifted, tables and bucket records visible to every warp

        // a bucket whose table overflowed is walked directly by its own warp
        if (nt > 0 && sm.cand_len[warp] < 0)
            for (int i = lane; i < nt; i += 32) {
                if (kMode == kPassBoth) {
                    my_pairs += direct_particle((int64_t)tb0 + i, cxb, cyb, cz, in, cs, ce, g, k, out, kPassLocal);
                    my_pairs_f += direct_particle((int64_t)tb0 + i, cxb, cyb, cz, in, cs, ce, g, k, out_f, kPassRemote);
                } else {
                    my_pairs += direct_particle((int64_t)tb0 + i, cxb, cyb, cz, in, cs, ce, g, k, out, kMode);
                }
            }

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
            // 4p + (q ^ d):  a = -2 T', nth = -(support^2 - |T'|^2 + rounding margin)
            const int my_t = 4 * p + q;
            const bool my_valid = my_t < bnt;
            float4 tp = make_float4(0.f, 0.f, 0.f, 0.f);
            float ax0 = 0.f, ay0 = 0.f, az0 = 0.f;
            float nt0 = 1.f;  // |p'|^2 + 1 > 0: an absent target accepts nothing
            if (my_valid) {
                tp = sm.A[tbase + my_t];
                const float t2 = tp.w;
                ax0 = -2.0f * tp.x; ay0 = -2.0f * tp.y; az0 = -2.0f * tp.z;
                // margin >= 1e-6 (2|T'| + 2h)^2, the rounding bound of the expanded form
                nt0 = t2 - k.support2 - 1e-6f * (8.0f * t2 + 3.0f * k.support2);
            }
            f32x2 ax01, ay01, az01, nt01, ax23, ay23, az23, nt23;
            {
                const float ax1 = __shfl_xor_sync(0xffffffffu, ax0, 8), ay1 = __shfl_xor_sync(0xffffffffu, ay0, 8);
                const float az1 = __shfl_xor_sync(0xffffffffu, az0, 8), nt1 = __shfl_xor_sync(0xffffffffu, nt0, 8);
                ax01 = pk(ax0, ax1); ay01 = pk(ay0, ay1); az01 = pk(az0, az1); nt01 = pk(nt0, nt1);
                // slots 2, 3 = slots 0, 1 of the lane 16 away
                ax23 = __shfl_xor_sync(0xffffffffu, ax01, 16); ay23 = __shfl_xor_sync(0xffffffffu, ay01, 16);
                az23 = __shfl_xor_sync(0xffffffffu, az01, 16); nt23 = __shfl_xor_sync(0xffffffffu, nt01, 16);
            }

            // split passes: owner labels of the 4 slots, one byte each (0xFF = absent target)
            uint32_t own4 = 0;
            if (kMode != kPassAll) {
                const uint32_t o0 = my_valid ? (uint32_t)sm.own[tbase + my_t] : 0xFFu;
                const uint32_t o1 = __shfl_xor_sync(0xffffffffu, o0, 8);
                const uint32_t o01 = o0 | (o1 << 8);
                own4 = o01 | (__shfl_xor_sync(0xffffffffu, o01, 16) << 16);
            }
            // keeps, of the 4 fresh mask bits of one candidate, those the pass takes:
            // same-owner pairs (step e) or other-owner pairs (step f)
            // (kPassBoth keeps every accepted pair and records the equality nibble in a second word)
            auto owner_filter = [&](uint32_t &mask, uint32_t &eqw, uint32_t e) {
                if (kMode == kPassAll) return;
                const uint32_t oj = sm.own[e >> 4];
                // four byte compares at once: (own4 ^ oj oj oj oj) has a zero byte where the labels
                // agree (labels < 32, absent targets 0xFF never match); exact per-byte zero test
                // (no carry crosses a byte), then the four flags are gathered into a nibble
                const uint32_t x = own4 ^ (oj * 0x01010101u);
                const uint32_t nz = ((x & 0x7F7F7F7Fu) + 0x7F7F7F7Fu) | x;     // bit 7 of a byte set <=> byte != 0
                const uint32_t eq = (((~nz & 0x80808080u) >> 7) * 0x01020408u) >> 24;   // byte d -> bit d
                if (kMode == kPassBoth) eqw = (eqw << 4) | eq;
                else mask &= ~0xFu | (kMode == kPassLocal ? eq : ~eq);
            };

            // ---- phase 1: the whole table, bit 4 s + d of mask word s / 8 <- chunk s, slot d ----
            uint32_t m0 = 0, m1 = 0, m2 = 0;
            uint32_t q0 = 0, q1 = 0, q2 = 0;   // kPassBoth: same-owner bits, aligned with m0..m2
            const int nch = Wp >> 5;
            const uint16_t *cb = cand + lane;
#pragma unroll 1
            for (int s = nch - 1; s >= 16; --s) {
                const uint32_t ce_ = cb[32 * s];
                const float4 pa = ld_rec(sm.A, ce_);
                test_push2(m2, pa, ax23, ay23, az23, nt23);
                test_push2(m2, pa, ax01, ay01, az01, nt01);
                owner_filter(m2, q2, ce_);
            }
#pragma unroll 4
            for (int s = min(nch, 16) - 1; s >= 8; --s) {
                const uint32_t ce_ = cb[32 * s];
                const float4 pa = ld_rec(sm.A, ce_);
                test_push2(m1, pa, ax23, ay23, az23, nt23);
                test_push2(m1, pa, ax01, ay01, az01, nt01);
                owner_filter(m1, q1, ce_);
            }
#pragma unroll 4
            for (int s = min(nch, 8) - 1; s >= 0; --s) {
                const uint32_t ce_ = cb[32 * s];
                const float4 pa = ld_rec(sm.A, ce_);
                test_push2(m0, pa, ax23, ay23, az23, nt23);
                test_push2(m0, pa, ax01, ay01, az01, nt01);
                owner_filter(m0, q0, ce_);
            }
            // every quarter collects the bits of its own target: slot d of the lanes of quarter
            // q ^ d.  Afterwards bit beta of word w <-> table position 256 w + t + 8 (beta ^ q).
            {
                const uint32_t a1 = __shfl_xor_sync(0xffffffffu, m0, 8), b1 = __shfl_xor_sync(0xffffffffu, m1, 8);
                const uint32_t a2 = __shfl_xor_sync(0xffffffffu, m0, 16), b2 = __shfl_xor_sync(0xffffffffu, m1, 16);
                const uint32_t a3 = __shfl_xor_sync(0xffffffffu, m0, 24), b3 = __shfl_xor_sync(0xffffffffu, m1, 24);
                m0 = (m0 & 0x11111111u) | (a1 & 0x22222222u) | (a2 & 0x44444444u) | (a3 & 0x88888888u);
                m1 = (m1 & 0x11111111u) | (b1 & 0x22222222u) | (b2 & 0x44444444u) | (b3 & 0x88888888u);
                if (nch > 16) {  // warp-uniform
                    const uint32_t c1 = __shfl_xor_sync(0xffffffffu, m2, 8), c2 = __shfl_xor_sync(0xffffffffu, m2, 16);
                    const uint32_t c3 = __shfl_xor_sync(0xffffffffu, m2, 24);
                    m2 = (m2 & 0x11111111u) | (c1 & 0x22222222u) | (c2 & 0x44444444u) | (c3 & 0x88888888u);
                }
                if (kMode == kPassBoth) {
                    auto xch = [&](uint32_t v) {
                        const uint32_t v1 = __shfl_xor_sync(0xffffffffu, v, 8), v2 = __shfl_xor_sync(0xffffffffu, v, 16);
                        const uint32_t v3 = __shfl_xor_sync(0xffffffffu, v, 24);
                        return (v & 0x11111111u) | (v1 & 0x22222222u) | (v2 & 0x44444444u) | (v3 & 0x88888888u);
                    };
                    q0 = xch(q0); q1 = xch(q1); q2 = xch(q2);
                }
            }
            // ---- phase 2: lane t of quarter q owns the accepted candidates of target q whose record
            //      index is = t (mod 8) and evaluates them straight from its mask words, two per
            //      round.  The 8 gathers of a quarter-warp always fall into 8 distinct 16-byte bank
            //      groups (conflict-free by construction); a lane that has run out of bits gathers
            //      the dummy record of its own class, which contributes exactly zero. -------------
            float4 tv = make_float4(0.f, 0.f, 0.f, 0.f);
            float th = 1.0f;   // the target's own smoothing length (NEXT-4)
            if (my_valid) tv = sm.B[tbase + my_t];
            if (kVarH && my_valid) th = sm.C[tbase + my_t].z;
            const f32x2 tpxy = pk(tp.x, tp.y), tvxy = pk(tv.x, tv.y);
            // phase 2 + reduction + parking of one set of mask words (kPassBoth runs it twice)
            auto pass2 = [&](uint32_t u0, uint32_t u1, uint32_t u2, int slot, uint32_t &cnt) {
            const int c = __popc(u0) + __popc(u1) + __popc(u2);
            const int rounds = (int)__reduce_max_sync(0xffffffffu, (unsigned)((c + 1) >> 1));
            PairAccum2 S;
            S.clear();
            {
                // three (mask word, table base) pairs, the non-empty words first; pop() is
                // branch-free: refill the head word when it has run dry, take its highest bit
                const uint32_t dummy = (uint32_t)(kDummy + t) * 16u;
                const uint32_t cbase = smem_u32(cand + t);
                uint32_t w = u0, w1 = u1, w2 = u2;
                uint32_t c0 = cbase, c1 = cbase + 512u, c2 = cbase + 1024u;
                if (w1 == 0u) { w1 = w2; c1 = c2; w2 = 0u; }
                if (w == 0u) { w = w1; c0 = c1; w1 = w2; c1 = c2; w2 = 0u; }
                auto pop = [&]() -> uint32_t {
                    const bool z = (w == 0u);
                    w = z ? w1 : w;   c0 = z ? c1 : c0;
                    w1 = z ? w2 : w1; c1 = z ? c2 : c1;
                    w2 = z ? 0u : w2;
                    const uint32_t beta = 31u - (uint32_t)__clz(w);   // 0xffffffff when w == 0
                    const bool valid = (w != 0u);
                    w &= ~(1u << (beta & 31u));
                    uint32_t e = dummy;
                    if (valid) {
                        uint16_t v;
                        asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(c0 + ((beta ^ (uint32_t)q) << 4)));
                        e = v;
                    }
                    return e;
                };
                auto eval = [&](uint32_t e) {
                    const float4 pa = ld_rec(sm.A, e);
                    const float4 pb = ld_rec(sm.B, e);
                    const float4 pc = ld_rec(sm.C, e);
                    const float4 pd = ld_rec(sm.D, e);
                    const float r2 = S.template add<kVarH>(tpxy, tp.z, tvxy, tv.z, pa, pb, pc, pd, -k.half_inv_h, th);
                    // exact test (phase 1 has a rounding margin; with per-particle lengths it runs on 2 h_max)
                    const float hs = th + pc.z;
                    if (kCount && r2 < (kVarH ? hs * hs : k.support2)) ++cnt;
                };
#pragma unroll 1
                for (int r = 0; r < rounds; ++r) {
                    const uint32_t e0 = pop();
                    const uint32_t e1 = pop();
                    eval(e0);
                    eval(e1);
                }
            }
            // ---- reduce the 16 sums over the quarter, park them -------------------------------
            {
                float v[16];
                S.unpack(v);
                reduce8_transposed(v, t);
                float *row = acc[slot * 4 + q];
                const int idx = ((t & 4) << 1) + ((t & 2) << 1) + ((t & 1) << 1);
                row[idx] = v[0];
                row[idx + 1] = v[1];
                if (t == 0) {
                    row[16] = __int_as_float(my_valid ? (int)(btb0 + my_t) : -1);
                    row[17] = __int_as_float(tbase + my_t);
                }
            }
            };
            if (kMode == kPassBoth) {
                // step e: same-owner pairs -> slot 0 -> out; step f: the others -> slot 1 -> out_f
                pass2(m0 & q0, m1 & q1, m2 & q2, 0, my_pairs);
                pass2(m0 & ~q0, m1 & ~q1, m2 & ~q2, 1, my_pairs_f);
            } else {
                pass2(m0, m1, m2, parked, my_pairs);
            }
            if (kMode != kPassRemote && my_valid && t == 0) ++my_self;  // the self pair is not a pair (reading S15)
            parked = kMode == kPassBoth ? 2 : parked + 1;   // kPassBoth parked two sets of this unit
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
                        for (int c = 0; c < 6; ++c) si[c] = 0.f;
                        // sigma_i and rho_i come back from the target's own record in shared memory
                        // (S = sigma / rho^2, m, V = m / rho): no global load on the epilogue's path
                        const int rs = __float_as_int(row[17]);
                        const float4 rb = sm.B[rs], rc = sm.C[rs], rd = sm.D[rs];
                        const float rho = rd.z / rd.w, rho2 = rho * rho;
                        si[0] = rc.x * rho2; si[1] = rc.w * rho2; si[2] = rb.w * rho2;
                        si[3] = rc.y * rho2; si[4] = rd.x * rho2; si[5] = rd.y * rho2;
                        float4 pos_i = make_float4(0.f, 0.f, 0.f, 0.f);
                        if (out.perm) pos_i = __ldg(in.posm + i);
                        const InteractOut &oo = (kMode == kPassBoth && lane >= 4) ? out_f : out;
                        finish_particle(Rr, si, rho, k, oo, (int64_t)i, pos_i, rb.x, rb.y, rb.z);
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
                    for (int c = 0; c < 6; ++c) si[c] = 0.f;
                    const int rs = __float_as_int(row[17]);
                    const float4 rb = sm.B[rs], rc = sm.C[rs], rd = sm.D[rs];
                    const float rho = rd.z / rd.w, rho2 = rho * rho;
                    si[0] = rc.x * rho2; si[1] = rc.w * rho2; si[2] = rb.w * rho2;
                    si[3] = rc.y * rho2; si[4] = rd.x * rho2; si[5] = rd.y * rho2;
                    float4 pos_i = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (out.perm) pos_i = __ldg(in.posm + i);
                    // same routing as the in-loop epilogue: kPassBoth parks step e in slot 0, step f in slot 1
                    const InteractOut &oo = (kMode == kPassBoth && lane >= 4) ? out_f : out;
                    finish_particle(Rr, si, rho, k, oo, (int64_t)i, pos_i, rb.x, rb.y, rb.z);
                }
            }
        }
    }
    if (kCount) {
        const uint32_t tot = __reduce_add_sync(0xffffffffu, my_pairs) - __reduce_add_sync(0xffffffffu, my_self);
        if (lane == 0 && tot) atomicAdd(pair_count, (unsigned long long)tot);
        if (kMode == kPassBoth) {
            const uint32_t tf = __reduce_add_sync(0xffffffffu, my_pairs_f);
            if (lane == 0 && tf) atomicAdd(pair_count + 1, (unsigned long long)tf);
        }
    }
}

int launch_interact_tiled(sph_ctx *c, int64_t n, const InteractIn &in, const uint32_t *sorted_hash,
                          const uint32_t *cs, const uint32_t *ce, const InteractOut &out,
                          unsigned long long *pair_count, int mode, const InteractOut *out_f)
{
    (void)sorted_hash;
    Packed rec;
    rec.A = in.posm;
    rec.B = c->rec_B;
    rec.C = c->rec_C;
    rec.D = c->rec_D;
    if (!(c->rec_fresh && in.posm == reinterpret_cast<const float4 *>(c->sorted.posm))) {
        pack_kernel<<<div_up(n, 256), 256, 0, c->stream>>>(n, in, rec.B, rec.C, rec.D);
        SPH_CHECK_LAUNCH(c);
    }
    c->rec_fresh = false;
    const int smem = (int)sizeof(TileSmem);
    const bool vh = in.h != nullptr;
    if (!c->attr_interact) {   // per device: once per ctx
        const void *fns[] = {
            (const void *)interact_tiled_kernel<true, kPassAll, false>, (const void *)interact_tiled_kernel<false, kPassAll, false>,
            (const void *)interact_tiled_kernel<true, kPassLocal, false>, (const void *)interact_tiled_kernel<true, kPassRemote, false>,
            (const void *)interact_tiled_kernel<true, kPassAll, true>, (const void *)interact_tiled_kernel<false, kPassAll, true>,
            (const void *)interact_tiled_kernel<true, kPassLocal, true>, (const void *)interact_tiled_kernel<true, kPassRemote, true>,
            (const void *)interact_tiled_kernel<true, kPassBoth, false>, (const void *)interact_tiled_kernel<true, kPassBoth, true>};
        for (const void *f : fns) SPH_CUDA_TRY(c, cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        c->attr_interact = true;
    }
    const int tiles_x = (c->grid.nx + kTBX - 1) / kTBX, tiles_y = (c->grid.ny + kTBY - 1) / kTBY;
    const int64_t tiles = (int64_t)tiles_x * tiles_y * c->grid.nz;
    if (tiles > 0x7fffffffll) return SPH_EINVAL;
    const unsigned gr = (unsigned)tiles;
    Consts kc = c->consts;
    if (vh) kc.cF = kc.cF_varh;   // h_ij^-5 is applied per pair (reading H2)
    // the split passes always count (one instantiation each); without a caller buffer the count
    // goes to ctx scratch
    unsigned long long *pc = (mode == kPassAll || pair_count) ? pair_count : c->s_pair_count;
#define SPH_LAUNCH_TILED(CNT, MODE, VH)                                                        \
    interact_tiled_kernel<CNT, MODE, VH><<<gr, kTW * 32, smem, c->stream>>>(                     \
        rec, in, cs, ce, c->grid, kc, out, pc, tiles_x, tiles_y, out_f ? *out_f : out)
    if (mode == kPassAll) {
        if (pair_count) { if (vh) SPH_LAUNCH_TILED(true, kPassAll, true); else SPH_LAUNCH_TILED(true, kPassAll, false); }
        else            { if (vh) SPH_LAUNCH_TILED(false, kPassAll, true); else SPH_LAUNCH_TILED(false, kPassAll, false); }
    } else if (mode == kPassLocal) {
        if (vh) SPH_LAUNCH_TILED(true, kPassLocal, true); else SPH_LAUNCH_TILED(true, kPassLocal, false);
    } else if (mode == kPassBoth) {
        if (!out_f || !pair_count) return SPH_EINVAL;   // two rate sets, pair_count[2]
        if (vh) SPH_LAUNCH_TILED(true, kPassBoth, true); else SPH_LAUNCH_TILED(true, kPassBoth, false);
    } else {
        if (vh) SPH_LAUNCH_TILED(true, kPassRemote, true); else SPH_LAUNCH_TILED(true, kPassRemote, false);
    }
#undef SPH_LAUNCH_TILED
    SPH_CHECK_LAUNCH(c);
    return SPH_OK;
}

}  // namespace sphb
