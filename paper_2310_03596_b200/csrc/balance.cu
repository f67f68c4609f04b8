// NEXT-2 / NEXT-4: one sweep of the paper's communication-load balancing heuristic
// on the owner labels (section III.A; multi-type variant PAPER.md:54-57; readings
// B1-B10 in DESIGN.md section 6.5).
//
// For every owner pair (A, B), A < B, in lexicographic order:
//   Cg_A, Cg_B        unweighted mean positions, kept as EXACT 2^-16 fixed-point int64 sums per owner
//                     (computed once per sweep, then updated by the swaps), so that the value does
//                     not depend on the order of any reduction and matches the oracle bit for bit;
//   balancing hash    projection s of the particle on the line Cg_own -> Cg_other in fp64 with a
//                     pinned operation sequence (no contraction): 0 if !(s > 1/2), hmax if s >= 1,
//                     else ceil(hmax (2 s - 1)) in [1, hmax];
//   n = min(nA, nB)   particles with a positive hash on each side; the n first of each side in
//                     the order (hash descending, id ascending) swap labels.
// The paper sorts by the balancing hash; the same selection is done here without a sort: a
// histogram over the <= 1024 hash values gives the threshold hash of each side, and among the ties
// at the threshold the ones with the SMALLEST ids move (a three-level radix select on the id).
//
// Layout: in the paper every GPU holds its own particles; here the labels are scattered over the
// id-ordered arrays, and a pair only concerns the particles of two owners.  The sweep therefore
// starts with ONE stable partition of the ids by (type, owner) (a single onesweep pass) and a
// gather of the positions into that grouped order.  A pair then streams two contiguous segments
// (hash, select, mark, swap); a swap exchanges two ENTRIES between the segments, so every segment
// keeps its size and offset, and the labels are written back once at the end of the sweep.  (The
// first two versions walked all n particles per pair: 1.4-1.9 ms and 0.5-1.0 ms per pair at 64 M
// particles; this one touches 2 n / G of them.)  The segment sizes are read back once per sweep
// (one small copy + stream synchronisation) to size the launches.
#include "sph_internal.cuh"

namespace sphb {

constexpr int kBalBins = 1024;  // hash values 0 .. hmax <= 1023

// device control block of a sweep (lives in ctx->bal)
constexpr int kBalTypes = 8;    // particle types of the multi-type variant

struct BalCtl {
    long long sum[SPH_MAX_OWNERS][kBalTypes][3];   // fixed-point coordinate sums per owner and type
    unsigned long long cnt[SPH_MAX_OWNERS][kBalTypes];
    unsigned long long swapped;         // pairs of particles swapped so far
    // per pair:
    double cgA[3], cgB[3];
    int valid;                          // both owners non-empty, distinct Cgs (B5)
    uint32_t thrA, thrB, quotaA, quotaB;  // threshold hash and how many of its ties move
    uint32_t tiesA, tiesB;              // particles AT the threshold hash (quota < ties: select by id)
    uint32_t m;                         // particles moving each way in this pair
    uint32_t hist[2][kBalBins];
    uint32_t sel[3][2][kBalBins];       // radix select on the id among the ties: 3 levels of 10 bits
    uint32_t seg[SPH_MAX_OWNERS * kBalTypes + 1];   // offsets of the (type, owner) segments
    uint32_t sel_active[2], sel_prefix[2], sel_rem[2];   // state of the select per side
    uint32_t sel_done[3];                             // blocks of level L that have finished
};

__device__ __forceinline__ long long fixed16(float x)
{
    return __double2ll_rn(__dmul_rn((double)x, 65536.0));
}

// one block: centres of gravity of the pair, validity, cleared histograms and look-back words
__global__ void bal_pair_begin_kernel(BalCtl *ctl, int A, int B, int T, int typed, double alpha,
                                      uint32_t *status, int64_t n_status, uint32_t *ticket)
{
    for (int i = threadIdx.x; i < 2 * kBalBins; i += blockDim.x) (&ctl->hist[0][0])[i] = 0;
    for (int i = threadIdx.x; i < 6 * kBalBins; i += blockDim.x) (&ctl->sel[0][0][0])[i] = 0;
    for (int64_t i = threadIdx.x; i < n_status; i += blockDim.x) status[i] = 0;   // look-back words of the mark pass
    if (threadIdx.x == 0) *ticket = 0;
    if (threadIdx.x != 0) return;
    const unsigned long long ca = ctl->cnt[A][T], cb = ctl->cnt[B][T];
    int valid = ca != 0 && cb != 0;   // B5 / B10
    if (valid) {
        const int own[2] = {A, B};
        for (int side = 0; side < 2; ++side)
            for (int a = 0; a < 3; ++a) {
                const int o = own[side];
                const double ctyp = __dmul_rn(__ddiv_rn((double)ctl->sum[o][T][a], (double)ctl->cnt[o][T]), 1.0 / 65536.0);
                double cg = ctyp;
                if (typed) {   // Cg' = alpha Cg_alltypes + (1 - alpha) Cg_type
                    long long sa = 0;
                    unsigned long long na = 0;
                    for (int t = 0; t < kBalTypes; ++t) { sa += ctl->sum[o][t][a]; na += ctl->cnt[o][t]; }
                    const double call = __dmul_rn(__ddiv_rn((double)sa, (double)na), 1.0 / 65536.0);
                    cg = __dadd_rn(__dmul_rn(alpha, call), __dmul_rn(__dsub_rn(1.0, alpha), ctyp));
                }
                (side == 0 ? ctl->cgA : ctl->cgB)[a] = cg;
            }
        if (ctl->cgA[0] == ctl->cgB[0] && ctl->cgA[1] == ctl->cgB[1] && ctl->cgA[2] == ctl->cgB[2]) valid = 0;
    }
    ctl->valid = valid;
    ctl->thrA = ctl->thrB = 0xFFFFFFFFu;
    ctl->quotaA = ctl->quotaB = 0;
    ctl->tiesA = ctl->tiesB = 0;
    ctl->m = 0;
    for (int i = 0; i < 2; ++i) { ctl->sel_active[i] = 0; ctl->sel_prefix[i] = 0; ctl->sel_rem[i] = 0; }
    for (int i = 0; i < 3; ++i) ctl->sel_done[i] = 0;
}

__device__ __forceinline__ int32_t balance_hash(const float4 &p, const double *own, const double *oth, int hmax)
{
    const double d0 = __dsub_rn(oth[0], own[0]), d1 = __dsub_rn(oth[1], own[1]), d2 = __dsub_rn(oth[2], own[2]);
    const double dd = __dadd_rn(__dadd_rn(__dmul_rn(d0, d0), __dmul_rn(d1, d1)), __dmul_rn(d2, d2));
    const double e0 = __dsub_rn((double)p.x, own[0]), e1 = __dsub_rn((double)p.y, own[1]),
                 e2 = __dsub_rn((double)p.z, own[2]);
    const double s = __ddiv_rn(__dadd_rn(__dadd_rn(__dmul_rn(e0, d0), __dmul_rn(e1, d1)), __dmul_rn(e2, d2)), dd);
    if (!(s > 0.5)) return 0;
    if (s >= 1.0) return hmax;
    double hv = ceil(__dmul_rn((double)hmax, __dsub_rn(__dmul_rn(2.0, s), 1.0)));
    if (hv < 1.0) hv = 1.0;
    if (hv > (double)hmax) hv = (double)hmax;
    return (int32_t)hv;
}

// ---- grouping: slot k of the grouped arrays holds particle gid[k]; the slots of (type T, owner g)
//      are the contiguous segment [seg[T * G + g], seg[T * G + g + 1]) --------------------------------
__global__ void __launch_bounds__(256)
bal_key_kernel(int64_t n, const int32_t *__restrict__ owner, const int32_t *__restrict__ ptype, int G,
               uint32_t *__restrict__ key)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n)
        key[i] = (uint32_t)(owner[i] & (SPH_MAX_OWNERS - 1)) +
                 (uint32_t)G * (uint32_t)(ptype ? (ptype[i] & (kBalTypes - 1)) : 0);
}

__global__ void __launch_bounds__(256)
bal_gather_kernel(int64_t n, const uint32_t *__restrict__ gid, const float4 *__restrict__ posm,
                  float4 *__restrict__ gpos)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) gpos[k] = __ldg(posm + __ldcs(gid + k));
}

// Exact fixed-point coordinate sums and counts per (type, owner) segment from the GROUPED positions
// (dense, one segment after the other): a warp owns 1024 consecutive slots; when they all lie in
// one segment (all but <= n_seg warps) it reduces in registers and issues three atomics.
__global__ void __launch_bounds__(256)
bal_seg_sums_kernel(int64_t n, const float4 *__restrict__ gpos, int n_seg, int G, BalCtl *ctl)
{
    __shared__ uint32_t s_seg[SPH_MAX_OWNERS * kBalTypes + 1];
    for (int i = threadIdx.x; i <= n_seg; i += blockDim.x) s_seg[i] = ctl->seg[i];
    __syncthreads();
    if (blockIdx.x == 0)
        for (int sgi = threadIdx.x; sgi < n_seg; sgi += blockDim.x)
            ctl->cnt[sgi % G][sgi / G] = (unsigned long long)(s_seg[sgi + 1] - s_seg[sgi]);
    auto seg_of = [&](uint32_t k) {
        int lo = 0, hi = n_seg;   // last segment with seg[s] <= k
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (s_seg[mid] <= k) lo = mid; else hi = mid;
        }
        return lo;
    };
    const int lane = threadIdx.x & 31;
    const int64_t wbase = ((int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5)) * 1024;
    if (wbase >= n) return;
    const int64_t wend = min(wbase + 1024, n);
    const int s0 = seg_of((uint32_t)wbase), s1 = seg_of((uint32_t)(wend - 1));
    if (s0 == s1) {
        long long f[3] = {0, 0, 0};
        for (int64_t k = wbase + lane; k < wend; k += 32) {
            const float4 p = __ldcs(gpos + k);
            f[0] += fixed16(p.x); f[1] += fixed16(p.y); f[2] += fixed16(p.z);
        }
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            long long v = f[a];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0 && v)
                atomicAdd(reinterpret_cast<unsigned long long *>(&ctl->sum[s0 % G][s0 / G][a]), (unsigned long long)v);
        }
    } else {
        for (int64_t k = wbase + lane; k < wend; k += 32) {
            const float4 p = __ldcs(gpos + k);
            const int sg = seg_of((uint32_t)k);
            atomicAdd(reinterpret_cast<unsigned long long *>(&ctl->sum[sg % G][sg / G][0]), (unsigned long long)fixed16(p.x));
            atomicAdd(reinterpret_cast<unsigned long long *>(&ctl->sum[sg % G][sg / G][1]), (unsigned long long)fixed16(p.y));
            atomicAdd(reinterpret_cast<unsigned long long *>(&ctl->sum[sg % G][sg / G][2]), (unsigned long long)fixed16(p.z));
        }
    }
}

// slot of element j of the pair's two segments (A first)
__device__ __forceinline__ int64_t pair_slot(int64_t j, int64_t offA, int64_t nA, int64_t offB)
{
    return j < nA ? offA + j : offB + (j - nA);
}

// Pass 1: balancing hash of every particle of the two segments, the two 1024-bin histograms.
__global__ void __launch_bounds__(256)
bal_hash_kernel(const float4 *__restrict__ gpos, const uint32_t *__restrict__ gid, BalCtl *ctl, int64_t offA,
                int64_t nA, int64_t offB, int64_t nB, int hmax, uint16_t *__restrict__ ghash,
                int32_t *__restrict__ bal_hash)
{
    __shared__ uint32_t s_hist[2][kBalBins];
    for (int i = threadIdx.x; i < 2 * kBalBins; i += blockDim.x) (&s_hist[0][0])[i] = 0;
    __syncthreads();
    if (ctl->valid) {
        const double cgA[3] = {ctl->cgA[0], ctl->cgA[1], ctl->cgA[2]};
        const double cgB[3] = {ctl->cgB[0], ctl->cgB[1], ctl->cgB[2]};
        // hash = hmax is by far the most frequent positive value (every particle beyond the other
        // Cg): those are counted per thread and warp-reduced instead of hammering one shared bin
        uint32_t n_max[2] = {0, 0};
        for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < nA + nB; j += (int64_t)gridDim.x * blockDim.x) {
            const int side = j < nA ? 0 : 1;
            const int64_t k = pair_slot(j, offA, nA, offB);
            const float4 p = __ldcs(gpos + k);
            const int32_t hv = side == 0 ? balance_hash(p, cgA, cgB, hmax) : balance_hash(p, cgB, cgA, hmax);
            ghash[k] = (uint16_t)hv;
            if (bal_hash) bal_hash[gid[k]] = hv;   // optional product: a 4-byte scatter per member
            if (hv == hmax) ++n_max[side];
            else if (hv > 0) atomicAdd(&s_hist[side][hv], 1u);
        }
        const uint32_t wa = __reduce_add_sync(0xffffffffu, n_max[0]), wb = __reduce_add_sync(0xffffffffu, n_max[1]);
        if ((threadIdx.x & 31) == 0) {
            if (wa) atomicAdd(&s_hist[0][hmax], wa);
            if (wb) atomicAdd(&s_hist[1][hmax], wb);
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < 2 * kBalBins; i += blockDim.x)
        if ((&s_hist[0][0])[i]) atomicAdd(&ctl->hist[0][0] + i, (&s_hist[0][0])[i]);
}

// one block of kBalBins threads: n = min(nA, nB); per side the threshold hash, the number of its
// ties that move and the number of ties.  Thread j owns hash value h = kBalBins - 1 - j, so an
// inclusive scan over j is the count of particles with a hash >= h.
__global__ void __launch_bounds__(kBalBins) bal_pair_select_kernel(BalCtl *ctl, int hmax)
{
    __shared__ unsigned int s_warp[2][kBalBins / 32];
    __shared__ unsigned int s_tot[2];
    if (!ctl->valid) return;   // uniform
    const int j = threadIdx.x, lane = j & 31, w = j >> 5;
    const int h = kBalBins - 1 - j;
    unsigned int cnt[2], inc[2];
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        cnt[s] = (h >= 1 && h <= hmax) ? ctl->hist[s][h] : 0u;
        unsigned int v = cnt[s];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned int x = __shfl_up_sync(0xffffffffu, v, o);
            if (lane >= o) v += x;
        }
        inc[s] = v;
        if (lane == 31) s_warp[s][w] = v;
    }
    __syncthreads();
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        unsigned int add = 0;
        for (int i = 0; i < w; ++i) add += s_warp[s][i];
        inc[s] += add;                       // particles of side s with a hash >= h
        if (j == kBalBins - 1) s_tot[s] = inc[s];
    }
    __syncthreads();
    const unsigned int m = min(s_tot[0], s_tot[1]);
    if (m == 0) {
        if (j == 0) ctl->valid = 0;
        return;
    }
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        const unsigned int above = inc[s] - cnt[s];            // hash > h
        if (above < m && inc[s] >= m && cnt[s] > 0) {          // h is the threshold of side s
            (s == 0 ? ctl->thrA : ctl->thrB) = (uint32_t)h;
            (s == 0 ? ctl->quotaA : ctl->quotaB) = m - above;
            (s == 0 ? ctl->tiesA : ctl->tiesB) = cnt[s];
            ctl->sel_active[s] = (m - above) < cnt[s];          // fewer movers than ties: the smallest ids
            ctl->sel_rem[s] = m - above;
        }
    }
    if (j == 0) { ctl->swapped += m; ctl->m = m; }
}

// ---- radix select on the id among the ties of a side (reading B6: id ascending) ----------------
// Level L histograms the 10-bit digit L (most significant first; ids < 2^30) of the ties whose
// higher digits equal the digits found so far; the LAST block of the level to finish looks up the
// digit that holds the quota-th tie and leaves prefix / remaining quota in the control block for
// the next level.  After level 2 the prefix IS the cut-off id (ids are distinct).
__device__ __forceinline__ void sel_find(BalCtl *ctl, int side, int L, uint32_t *s_scan /* [256] */,
                                         uint32_t *s_pub /* [2] */)
{
    // smallest digit d with  sum_{x <= d} sel[L][side][x] >= rem   (block-wide, 256 threads x 4 bins)
    const int t = threadIdx.x;
    const uint32_t rem = ctl->sel_rem[side];
    uint32_t c[4], run = 0;
#pragma unroll
    for (int q = 0; q < 4; ++q) { c[q] = __ldcg(&ctl->sel[L][side][4 * t + q]); run += c[q]; }
    s_scan[t] = run;
    __syncthreads();
    if (t < 32) {   // warp 0 scans the 256 partial sums
        uint32_t v[8], tot = 0;
#pragma unroll
        for (int q = 0; q < 8; ++q) { v[q] = s_scan[8 * t + q]; tot += v[q]; }
        uint32_t inc = tot;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t x = __shfl_up_sync(0xffffffffu, inc, o);
            if (t >= o) inc += x;
        }
        uint32_t ex = inc - tot;
#pragma unroll
        for (int q = 0; q < 8; ++q) { const uint32_t y = v[q]; s_scan[8 * t + q] = ex; ex += y; }
    }
    __syncthreads();
    uint32_t ex = s_scan[t];       // ties in bins < 4 t
    // exactly one bin satisfies ex < rem <= ex + c: its thread publishes digit and new rem
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        if (rem > ex && rem <= ex + c[q]) { s_pub[0] = 4 * t + q; s_pub[1] = rem - ex; }
        ex += c[q];
    }
    __syncthreads();
    if (t == 0) {
        ctl->sel_prefix[side] |= s_pub[0] << (20 - 10 * L);
        ctl->sel_rem[side] = s_pub[1];
    }
    __syncthreads();
}

template <int LEVEL>
__global__ void __launch_bounds__(256)
bal_sel_kernel(const uint16_t *__restrict__ ghash, const uint32_t *__restrict__ gid, BalCtl *ctl, int64_t offA,
               int64_t nA, int64_t offB, int64_t nB)
{
    __shared__ uint32_t s_h[2][kBalBins];
    __shared__ uint32_t s_scan[256], s_pub[2];
    __shared__ bool s_last;
    if (!ctl->valid) return;
    const bool actA = ctl->sel_active[0], actB = ctl->sel_active[1];
    if (!actA && !actB) return;   // every tie moves on both sides: nothing to select (uniform)
    for (int i = threadIdx.x; i < 2 * kBalBins; i += blockDim.x) (&s_h[0][0])[i] = 0;
    __syncthreads();
    const uint32_t thrA = ctl->thrA, thrB = ctl->thrB;
    const uint32_t preA = ctl->sel_prefix[0], preB = ctl->sel_prefix[1];
    constexpr int kShift = 20 - 10 * LEVEL;
    const uint32_t himask = LEVEL == 0 ? 0u : ~((1u << (kShift + 10)) - 1u);
    for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < nA + nB; j += (int64_t)gridDim.x * blockDim.x) {
        const int side = j < nA ? 0 : 1;
        if (!(side ? actB : actA)) continue;
        const int64_t k = pair_slot(j, offA, nA, offB);
        if ((uint32_t)ghash[k] != (side ? thrB : thrA)) continue;
        const uint32_t id = gid[k];
        if ((id & himask) != (side ? preB : preA)) continue;
        atomicAdd(&s_h[side][(id >> kShift) & (kBalBins - 1)], 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < 2 * kBalBins; i += blockDim.x)
        if ((&s_h[0][0])[i]) atomicAdd(&ctl->sel[LEVEL][0][0] + i, (&s_h[0][0])[i]);
    // the last block to arrive turns the finished histogram into the next digit
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(&ctl->sel_done[LEVEL], 1u) == gridDim.x - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    if (actA) sel_find(ctl, 0, LEVEL, s_scan, s_pub);
    if (actB) sel_find(ctl, 1, LEVEL, s_scan, s_pub);
}

// ---- mark the movers and list them per side (compaction by decoupled look-back over the tiles
//      of each segment); a particle moves if its hash is above the threshold, or at it and --
//      where the side selects -- its id is not above the cut-off id found by the radix select ----
constexpr int kBalThreads = 256;
constexpr int kBalItems = 16;
constexpr int kBalTile = kBalThreads * kBalItems;   // slots per tile of the mark pass

__global__ void __launch_bounds__(kBalThreads)
bal_mark_kernel(const uint16_t *__restrict__ ghash, const uint32_t *__restrict__ gid, BalCtl *ctl, int64_t offA,
                int64_t nA, int64_t offB, int64_t nB, uint32_t *status /* [tilesA + tilesB] */, uint32_t *ticket,
                uint32_t *__restrict__ listA, uint32_t *__restrict__ listB)
{
    __shared__ uint32_t s_warp[kBalThreads / 32];
    __shared__ uint32_t s_tile, s_excl;
    if (!ctl->valid) return;   // uniform over the grid
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    const uint32_t tilesA = (uint32_t)((nA + kBalTile - 1) / kBalTile);
    const int side = tile < tilesA ? 0 : 1;
    const uint32_t ltile = side ? tile - tilesA : tile;        // tile index inside the segment
    const int64_t seg_off = side ? offB : offA, seg_n = side ? nB : nA;
    const uint32_t thr = side ? ctl->thrB : ctl->thrA;
    const bool sel_on = ctl->sel_active[side];
    const uint32_t cut_id = ctl->sel_prefix[side];   // after the three levels: the quota-th smallest tie id
    const int64_t base = (int64_t)ltile * kBalTile + (int64_t)tid * kBalItems;
    uint32_t mv = 0;   // bit j: item j of this thread moves
#pragma unroll
    for (int j = 0; j < kBalItems; ++j) {
        if (base + j < seg_n) {
            const uint32_t hv = ghash[seg_off + base + j];
            bool move = hv > thr;
            // ids are distinct, so exactly quota ties have an id <= the cut-off id
            if (hv == thr && hv > 0) move = !sel_on || gid[seg_off + base + j] <= cut_id;
            if (move && hv > 0) mv |= 1u << j;
        }
    }
    const uint32_t cnt = __popc(mv);
    uint32_t inc = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t x = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += x;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    uint32_t add = 0, tile_total = 0;
#pragma unroll
    for (int i = 0; i < kBalThreads / 32; ++i) {
        const uint32_t w = s_warp[i];
        add += (i < warp) ? w : 0u;
        tile_total += w;
    }
    if (warp == 0) {
        // warp-parallel decoupled look-back over the tiles of THIS segment (as in scan_exclusive_kernel)
        uint32_t *st_w = status + (side ? tilesA : 0u);
        if (lane == 0) st_volatile_u32(st_w + ltile, (ltile == 0 ? kFlagPrefix : kFlagAgg) | tile_total);
        uint32_t excl = 0;
        if (ltile > 0) {
            int64_t t0 = (int64_t)ltile - 1;
            while (true) {
                const int64_t t = t0 - lane;
                const uint32_t s = t >= 0 ? ld_volatile_u32(st_w + t) : kFlagPrefix;
                const uint32_t f = s & kFlagMask;
                const uint32_t pref = __ballot_sync(0xffffffffu, f == kFlagPrefix);
                const uint32_t unpub = __ballot_sync(0xffffffffu, f == 0);
                const int fp = pref ? __ffs(pref) - 1 : 31;
                const uint32_t need = 0xffffffffu >> (31 - fp);
                if (unpub & need) continue;
                excl += __reduce_add_sync(0xffffffffu, lane <= fp ? (s & kValueMask) : 0u);
                if (pref) break;
                t0 -= 32;
            }
            if (lane == 0) st_volatile_u32(st_w + ltile, kFlagPrefix | (excl + tile_total));
        }
        if (lane == 0) s_excl = excl;
    }
    __syncthreads();
    uint32_t rank = s_excl + add + (inc - cnt);
    uint32_t *list = side ? listB : listA;
#pragma unroll
    for (int j = 0; j < kBalItems; ++j)
        if (mv & (1u << j)) list[rank++] = (uint32_t)(base + j);   // slot index inside the segment
}

// ---- swap: the j-th mover of A and the j-th mover of B exchange their entries -------------------
__global__ void __launch_bounds__(256)
bal_swap_kernel(float4 *__restrict__ gpos, uint32_t *__restrict__ gid, BalCtl *ctl, int A, int B, int T,
                int64_t offA, int64_t offB, const uint32_t *__restrict__ listA, const uint32_t *__restrict__ listB)
{
    // D = (coordinates leaving A) - (coordinates leaving B): sum[A] -= D, sum[B] += D.  Exact
    // integer sums, so the order of the block and grid reductions does not matter.
    __shared__ long long s_d[3];
    if (threadIdx.x < 3) s_d[threadIdx.x] = 0;
    __syncthreads();
    if (!ctl->valid) return;   // uniform over the grid
    const uint32_t m = ctl->m;
    long long f[3] = {0, 0, 0};
    for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < m; j += gridDim.x * blockDim.x) {
        const int64_t a = offA + listA[j], b = offB + listB[j];
        const float4 pa = gpos[a], pb = gpos[b];
        const uint32_t ia = gid[a], ib = gid[b];
        gpos[a] = pb; gpos[b] = pa;
        gid[a] = ib; gid[b] = ia;
        f[0] += fixed16(pa.x) - fixed16(pb.x);
        f[1] += fixed16(pa.y) - fixed16(pb.y);
        f[2] += fixed16(pa.z) - fixed16(pb.z);
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        long long v = f[a];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) == 0 && v) atomicAdd(reinterpret_cast<unsigned long long *>(&s_d[a]), (unsigned long long)v);
    }
    __syncthreads();
    if (threadIdx.x < 3 && s_d[threadIdx.x]) {
        const long long d = s_d[threadIdx.x];
        atomicAdd(reinterpret_cast<unsigned long long *>(&ctl->sum[A][T][threadIdx.x]), (unsigned long long)(-d));
        atomicAdd(reinterpret_cast<unsigned long long *>(&ctl->sum[B][T][threadIdx.x]), (unsigned long long)d);
    }
}

// ---- end of the sweep: the label of every particle is the owner of the segment that holds it ----
__global__ void __launch_bounds__(256)
bal_writeback_kernel(int64_t n, const uint32_t *__restrict__ gid, const uint32_t *__restrict__ seg, int n_seg, int G,
                     int32_t *__restrict__ owner)
{
    __shared__ uint32_t s_seg[SPH_MAX_OWNERS * kBalTypes + 1];
    for (int i = threadIdx.x; i <= n_seg; i += blockDim.x) s_seg[i] = seg[i];
    __syncthreads();
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    int lo = 0, hi = n_seg;   // last segment with seg[s] <= k
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (s_seg[mid] <= (uint32_t)k) lo = mid; else hi = mid;
    }
    owner[gid[k]] = lo % G;
}

__global__ void bal_finish_kernel(const BalCtl *ctl, unsigned long long *swapped_out)
{
    if (swapped_out) *swapped_out = ctl->swapped;
}

int launch_balance(sph_ctx *c, int64_t n, const float *posm, int32_t *owner, const int32_t *ptype, int n_types,
                   double alpha, int hmax, int32_t *bal_hash, unsigned long long *swapped)
{
    // ptype == NULL: single particle type, section III.A (plain Cg); else section III.B: the pair
    // sweep per type with the biased Cg' of PAPER.md:56
    BalCtl *ctl = reinterpret_cast<BalCtl *>(c->bal);
    const float4 *p4 = reinterpret_cast<const float4 *>(posm);
    SPH_CUDA_TRY(c, cudaMemsetAsync(ctl, 0, sizeof(BalCtl), c->stream));
    if (bal_hash) SPH_CUDA_TRY(c, cudaMemsetAsync(bal_hash, 0, sizeof(int32_t) * (size_t)n, c->stream));
    const int G = c->params.n_owners, NT = ptype ? n_types : 1, typed = ptype != nullptr;
    if (n > 0 && G > 1) {
        // ---- group the ids by (type, owner): one stable partition pass, then the positions ----
        const int n_seg = G * NT;
        uint32_t *seg_dev = ctl->seg;                        // [n_seg + 1] segment offsets (device)
        bal_key_kernel<<<div_up(n, 256), 256, 0, c->stream>>>(n, owner, ptype, G, c->alt_keys);
        SPH_CHECK_LAUNCH(c);
        uint32_t *gid = nullptr;
        int rc = launch_partition_keys(c, n, n_seg, seg_dev, nullptr, &gid);
        if (rc != SPH_OK) return rc;
        float4 *gpos = reinterpret_cast<float4 *>(c->sorted.posm);
        bal_gather_kernel<<<div_up(n, 256), 256, 0, c->stream>>>(n, gid, p4, gpos);
        SPH_CHECK_LAUNCH(c);
        bal_seg_sums_kernel<<<div_up(n, 8 * 1024), 256, 0, c->stream>>>(n, gpos, n_seg, G, ctl);
        SPH_CHECK_LAUNCH(c);
        // the segment sizes size the launches of the pairs: one small read-back per sweep
        uint32_t seg_h[SPH_MAX_OWNERS * kBalTypes + 1];
        SPH_CUDA_TRY(c, cudaMemcpyAsync(seg_h, seg_dev, sizeof(uint32_t) * (n_seg + 1), cudaMemcpyDeviceToHost, c->stream));
        SPH_CUDA_TRY(c, cudaStreamSynchronize(c->stream));
        uint16_t *ghash = reinterpret_cast<uint16_t *>(c->alt_keys);          // free again after the partition
        uint32_t *listA = c->s_sorted_hash, *listB = c->s_perm;               // movers of a pair (slot indices)
        uint32_t *status = c->alt_vals;                                       // look-back words of the mark pass
        uint32_t *ticket = c->tile_counter + kMaxPasses;
        for (int T = 0; T < NT; ++T)
            for (int A = 0; A < G; ++A)
                for (int B = A + 1; B < G; ++B) {
                    const int64_t offA = seg_h[T * G + A], nA = seg_h[T * G + A + 1] - offA;
                    const int64_t offB = seg_h[T * G + B], nB = seg_h[T * G + B + 1] - offB;
                    if (nA == 0 || nB == 0) continue;   // B5 / B10: the pair is skipped
                    const int64_t tiles = (nA + kBalTile - 1) / kBalTile + (nB + kBalTile - 1) / kBalTile;
                    const int pb = (int)min((int64_t)c->num_sms * 8, (nA + nB + 255) / 256);
                    bal_pair_begin_kernel<<<1, 256, 0, c->stream>>>(ctl, A, B, T, typed, alpha, status, tiles, ticket);
                    SPH_CHECK_LAUNCH(c);
                    bal_hash_kernel<<<pb, 256, 0, c->stream>>>(gpos, gid, ctl, offA, nA, offB, nB, hmax, ghash, bal_hash);
                    SPH_CHECK_LAUNCH(c);
                    bal_pair_select_kernel<<<1, kBalBins, 0, c->stream>>>(ctl, hmax);
                    SPH_CHECK_LAUNCH(c);
                    bal_sel_kernel<0><<<pb, 256, 0, c->stream>>>(ghash, gid, ctl, offA, nA, offB, nB);
                    SPH_CHECK_LAUNCH(c);
                    bal_sel_kernel<1><<<pb, 256, 0, c->stream>>>(ghash, gid, ctl, offA, nA, offB, nB);
                    SPH_CHECK_LAUNCH(c);
                    bal_sel_kernel<2><<<pb, 256, 0, c->stream>>>(ghash, gid, ctl, offA, nA, offB, nB);
                    SPH_CHECK_LAUNCH(c);
                    bal_mark_kernel<<<(unsigned)tiles, kBalThreads, 0, c->stream>>>(ghash, gid, ctl, offA, nA, offB, nB,
                                                                                  status, ticket, listA, listB);
                    SPH_CHECK_LAUNCH(c);
                    const int sb = (int)min((int64_t)c->num_sms * 4, (min(nA, nB) + 255) / 256);
                    bal_swap_kernel<<<sb, 256, 0, c->stream>>>(gpos, gid, ctl, A, B, T, offA, offB, listA, listB);
                    SPH_CHECK_LAUNCH(c);
                }
        bal_writeback_kernel<<<div_up(n, 256), 256, 0, c->stream>>>(n, gid, seg_dev, n_seg, G, owner);
        SPH_CHECK_LAUNCH(c);
    }
    bal_finish_kernel<<<1, 1, 0, c->stream>>>(ctl, swapped);
    SPH_CHECK_LAUNCH(c);
    return SPH_OK;
}

size_t balance_scratch_bytes() { return sizeof(BalCtl); }

}  // namespace sphb
