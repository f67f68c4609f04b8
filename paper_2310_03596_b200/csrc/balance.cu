// NEXT-2: one sweep of the paper's communication-load balancing heuristic on the
// owner labels (section III.A; readings B1-B7 in DESIGN.md section 6.5).
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
// histogram over the <= 1024 hash values gives the threshold hash of each side, and the ties at
// the threshold are ranked by id with an exclusive scan.  Everything is decided on the device
// (no host synchronisation); a pair with nothing to swap costs its kernels but changes nothing.
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
    uint32_t hist[2][kBalBins];
};

__device__ __forceinline__ long long fixed16(float x)
{
    return __double2ll_rn(__dmul_rn((double)x, 65536.0));
}

__global__ void __launch_bounds__(256)
bal_sums_kernel(int64_t n, const float4 *__restrict__ posm, const int32_t *__restrict__ owner,
                const int32_t *__restrict__ ptype, BalCtl *ctl)
{
    __shared__ long long s_sum[SPH_MAX_OWNERS][kBalTypes][3];
    __shared__ unsigned long long s_cnt[SPH_MAX_OWNERS][kBalTypes];
    for (int i = threadIdx.x; i < SPH_MAX_OWNERS * kBalTypes * 3; i += blockDim.x) (&s_sum[0][0][0])[i] = 0;
    for (int i = threadIdx.x; i < SPH_MAX_OWNERS * kBalTypes; i += blockDim.x) (&s_cnt[0][0])[i] = 0;
    __syncthreads();
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float4 p = posm[i];
        const int o = owner[i] & (SPH_MAX_OWNERS - 1);
        const int t = ptype ? (ptype[i] & (kBalTypes - 1)) : 0;
        atomicAdd(reinterpret_cast<unsigned long long *>(&s_sum[o][t][0]), (unsigned long long)fixed16(p.x));
        atomicAdd(reinterpret_cast<unsigned long long *>(&s_sum[o][t][1]), (unsigned long long)fixed16(p.y));
        atomicAdd(reinterpret_cast<unsigned long long *>(&s_sum[o][t][2]), (unsigned long long)fixed16(p.z));
        atomicAdd(&s_cnt[o][t], 1ull);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < SPH_MAX_OWNERS * kBalTypes * 3; i += blockDim.x)
        if ((&s_sum[0][0][0])[i])
            atomicAdd(reinterpret_cast<unsigned long long *>(&ctl->sum[0][0][0]) + i,
                      (unsigned long long)(&s_sum[0][0][0])[i]);
    for (int i = threadIdx.x; i < SPH_MAX_OWNERS * kBalTypes; i += blockDim.x)
        if ((&s_cnt[0][0])[i]) atomicAdd(&ctl->cnt[0][0] + i, (&s_cnt[0][0])[i]);
}

// one block: centres of gravity of the pair, validity, cleared histograms and look-back words
__global__ void bal_pair_begin_kernel(BalCtl *ctl, int A, int B, int T, int typed, double alpha,
                                      uint32_t *status, int64_t n_status, uint32_t *ticket)
{
    for (int i = threadIdx.x; i < 2 * kBalBins; i += blockDim.x) (&ctl->hist[0][0])[i] = 0;
    for (int64_t i = threadIdx.x; i < n_status; i += blockDim.x) status[i] = 0;   // look-back words of pass 2
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

// Per pair the particles are visited TWICE, both times as a dense stream:
//   pass 1 (bal_hash_kernel): owner labels in, balancing hash of the pair's particles out, plus a
//     dense 16-bit code per particle (0 = takes no part or hash 0; else side bit 14 | hash), plus
//     the two 1024-bin histograms;
//   pass 2 (bal_swap_kernel): codes in; the ties at the threshold hash are ranked by id with a
//     decoupled look-back over the tiles (two status words per tile, one per side) INSIDE the
//     pass, and the labels of the selected particles are flipped at once.
// (The first version ran seven full-length passes per pair: hash, tie indicators, two separate
// scans reading and writing 4 B per particle each, swap: 1.4-1.9 ms per pair at 64 M particles.)
constexpr int kBalThreads = 256;
constexpr int kBalItems = 32;
constexpr int kBalTile = kBalThreads * kBalItems;   // ids per tile of pass 2

__device__ __forceinline__ uint16_t bal_code(int32_t hv, int side)
{
    return hv > 0 ? (uint16_t)((side ? 0x4000 : 0) | hv) : (uint16_t)0;
}

__global__ void __launch_bounds__(256)
bal_hash_kernel(int64_t n, const float4 *__restrict__ posm, const int32_t *__restrict__ owner,
                const int32_t *__restrict__ ptype, BalCtl *ctl, int A, int B, int T, int hmax,
                int32_t *__restrict__ bal_hash, uint16_t *__restrict__ code)
{
    __shared__ uint32_t s_hist[2][kBalBins];
    for (int i = threadIdx.x; i < 2 * kBalBins; i += blockDim.x) (&s_hist[0][0])[i] = 0;
    __syncthreads();
    if (ctl->valid) {
        const double cgA[3] = {ctl->cgA[0], ctl->cgA[1], ctl->cgA[2]};
        const double cgB[3] = {ctl->cgB[0], ctl->cgB[1], ctl->cgB[2]};
        // hash = hmax is by far the most frequent positive value (every particle beyond the other
        // Cg): those are counted per thread and warp-reduced instead of hammering one shared bin
        uint32_t n_max = 0;   // low half: side A, high half: side B
        auto member = [&](int o, int t) -> bool { return (o == A || o == B) && (!ptype || t == T); };
        auto hash_of = [&](int64_t i, int o, const float4 &p) -> uint16_t {
            const int side = o == A ? 0 : 1;
            const int32_t hv = side == 0 ? balance_hash(p, cgA, cgB, hmax) : balance_hash(p, cgB, cgA, hmax);
            if (bal_hash) bal_hash[i] = hv;   // optional product: a 4-byte scatter per member
            if (hv == hmax) n_max += side ? 0x10000u : 1u;
            else if (hv > 0) atomicAdd(&s_hist[side][hv], 1u);
            return bal_code(hv, side);
        };
        // eight particles per thread and iteration: two 128-bit owner loads, then the position
        // gathers of all members in flight together, one 128-bit code store
        const bool vec = ((reinterpret_cast<uintptr_t>(owner) | (ptype ? reinterpret_cast<uintptr_t>(ptype) : 0)) & 15) == 0 &&
                         (reinterpret_cast<uintptr_t>(code) & 15) == 0;
        const int64_t n8 = vec ? (n >> 3) : 0;
        for (int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; g < n8; g += (int64_t)gridDim.x * blockDim.x) {
            const int4 oa = __ldcs(reinterpret_cast<const int4 *>(owner) + 2 * g);
            const int4 ob = __ldcs(reinterpret_cast<const int4 *>(owner) + 2 * g + 1);
            int4 ta = make_int4(0, 0, 0, 0), tb = ta;
            if (ptype) {
                ta = __ldcs(reinterpret_cast<const int4 *>(ptype) + 2 * g);
                tb = __ldcs(reinterpret_cast<const int4 *>(ptype) + 2 * g + 1);
            }
            const int o[8] = {oa.x, oa.y, oa.z, oa.w, ob.x, ob.y, ob.z, ob.w};
            const int t[8] = {ta.x, ta.y, ta.z, ta.w, tb.x, tb.y, tb.z, tb.w};
            const int64_t i = g << 3;
            float4 p[8];
            bool m[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                m[j] = member(o[j], t[j]);
                p[j] = m[j] ? __ldg(posm + i + j) : make_float4(0.f, 0.f, 0.f, 0.f);
            }
            uint32_t c[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) c[j] = m[j] ? hash_of(i + j, o[j], p[j]) : 0u;
            __stcs(reinterpret_cast<uint4 *>(code) + g,
                   make_uint4(c[0] | (c[1] << 16), c[2] | (c[3] << 16), c[4] | (c[5] << 16), c[6] | (c[7] << 16)));
        }
        for (int64_t i = (n8 << 3) + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
             i += (int64_t)gridDim.x * blockDim.x) {
            const int o = owner[i], t = ptype ? ptype[i] : 0;
            code[i] = member(o, t) ? hash_of(i, o, __ldg(posm + i)) : (uint16_t)0;
        }
        // (a thread sees at most n / (grid x 256 x 4) x 4 < 2^16 particles per side for n < 2^30)
        const uint32_t wa = __reduce_add_sync(0xffffffffu, n_max & 0xFFFFu), wb = __reduce_add_sync(0xffffffffu, n_max >> 16);
        if ((threadIdx.x & 31) == 0) {
            if (wa) atomicAdd(&s_hist[0][hmax], wa);
            if (wb) atomicAdd(&s_hist[1][hmax], wb);
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < 2 * kBalBins; i += blockDim.x)
        if ((&s_hist[0][0])[i]) atomicAdd(&ctl->hist[0][0] + i, (&s_hist[0][0])[i]);
}

// one block of kBalBins threads: n = min(nA, nB); per side the threshold hash and the number of
// its ties that move.  Thread j owns hash value h = kBalBins - 1 - j, so an inclusive scan over j is
// the count of particles with a hash >= h.
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
        }
    }
    if (j == 0) ctl->swapped += m;
}

// Pass 2: one tile of kBalTile consecutive ids per block (dynamic ticket).  The ties at the
// threshold hash of each side are ranked by id: block scan of the per-thread tie counts, then a
// decoupled look-back over the preceding tiles (warp 0: side A, warp 1: side B); a particle moves
// if its hash is above the threshold, or equal to it with rank < quota (reading B6).
__global__ void __launch_bounds__(kBalThreads)
bal_swap_kernel(int64_t n, const float4 *__restrict__ posm, int32_t *__restrict__ owner,
                const uint16_t *__restrict__ code, BalCtl *ctl, int A, int B, int T, uint32_t *statusA,
                uint32_t *statusB, uint32_t *ticket)
{
    // D = (coordinates leaving A) - (coordinates leaving B): sum[A] -= D, sum[B] += D.  Exact
    // integer sums, so the order of the block and grid reductions does not matter.
    __shared__ long long s_d[3];
    __shared__ uint32_t s_warp[kBalThreads / 32];
    __shared__ uint32_t s_tile, s_excl[2];
    if (!ctl->valid) return;   // uniform over the grid: nothing to swap for this pair
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    if (tid < 3) s_d[tid] = 0;
    __syncthreads();
    const uint32_t tile = s_tile;
    const int64_t base = (int64_t)tile * kBalTile + (int64_t)tid * kBalItems;
    const uint32_t thrA = ctl->thrA, thrB = ctl->thrB, quotaA = ctl->quotaA, quotaB = ctl->quotaB;
    uint16_t c[kBalItems];
    if (base + kBalItems <= n && (reinterpret_cast<uintptr_t>(code) & 15) == 0) {
#pragma unroll
        for (int q = 0; q < kBalItems / 8; ++q) {
            const uint4 x = __ldcs(reinterpret_cast<const uint4 *>(code + base) + q);
            c[8 * q] = (uint16_t)x.x; c[8 * q + 1] = (uint16_t)(x.x >> 16);
            c[8 * q + 2] = (uint16_t)x.y; c[8 * q + 3] = (uint16_t)(x.y >> 16);
            c[8 * q + 4] = (uint16_t)x.z; c[8 * q + 5] = (uint16_t)(x.z >> 16);
            c[8 * q + 6] = (uint16_t)x.w; c[8 * q + 7] = (uint16_t)(x.w >> 16);
        }
    } else {
#pragma unroll
        for (int j = 0; j < kBalItems; ++j) c[j] = (base + j < n) ? code[base + j] : (uint16_t)0;
    }
    // ties of this thread: side A in the low half, side B in the high half (each <= 16)
    uint32_t ties = 0;
#pragma unroll
    for (int j = 0; j < kBalItems; ++j) {
        const uint32_t hv = c[j] & 0x3FFFu;
        const bool sideB = c[j] & 0x4000u;
        if (c[j] && hv == (sideB ? thrB : thrA)) ties += sideB ? 0x10000u : 1u;
    }
    uint32_t inc = ties;   // block scan (totals <= 4096 per side: 16 bits each are enough)
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
    if (warp < 2) {
        // warp-parallel decoupled look-back (as in scan_exclusive_kernel), one side per warp
        uint32_t *status = warp == 0 ? statusA : statusB;
        const uint32_t mine = warp == 0 ? (tile_total & 0xFFFFu) : (tile_total >> 16);
        if (lane == 0) st_volatile_u32(status + tile, (tile == 0 ? kFlagPrefix : kFlagAgg) | mine);
        uint32_t excl = 0;
        if (tile > 0) {
            int64_t t0 = (int64_t)tile - 1;
            while (true) {
                const int64_t t = t0 - lane;
                const uint32_t s = t >= 0 ? ld_volatile_u32(status + t) : kFlagPrefix;
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
            if (lane == 0) st_volatile_u32(status + tile, kFlagPrefix | (excl + mine));
        }
        if (lane == 0) s_excl[warp] = excl;
    }
    __syncthreads();
    const uint32_t before = add + (inc - ties);
    uint32_t rankA = s_excl[0] + (before & 0xFFFFu), rankB = s_excl[1] + (before >> 16);
    long long f[3] = {0, 0, 0};
#pragma unroll
    for (int j = 0; j < kBalItems; ++j) {
        if (!c[j]) continue;
        const uint32_t hv = c[j] & 0x3FFFu;
        const bool sideB = c[j] & 0x4000u;
        const uint32_t thr = sideB ? thrB : thrA;
        bool move = hv > thr;
        if (hv == thr) {
            move = sideB ? rankB < quotaB : rankA < quotaA;
            if (sideB) ++rankB; else ++rankA;
        }
        if (move) {
            const int64_t i = base + j;
            owner[i] = sideB ? A : B;
            const float4 p = __ldg(posm + i);
            const long long sgn = sideB ? -1 : 1;
            f[0] += sgn * fixed16(p.x); f[1] += sgn * fixed16(p.y); f[2] += sgn * fixed16(p.z);
        }
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        long long v = f[a];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0 && v) atomicAdd(reinterpret_cast<unsigned long long *>(&s_d[a]), (unsigned long long)v);
    }
    __syncthreads();
    if (tid < 3 && s_d[tid]) {
        const long long d = s_d[tid];
        atomicAdd(reinterpret_cast<unsigned long long *>(&ctl->sum[A][T][tid]), (unsigned long long)(-d));
        atomicAdd(reinterpret_cast<unsigned long long *>(&ctl->sum[B][T][tid]), (unsigned long long)d);
    }
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
    int32_t *bh = bal_hash;   // NULL: the hashes are not stored (pass 2 works on the 16-bit codes)
    uint16_t *code = reinterpret_cast<uint16_t *>(c->alt_keys);          // scratch (stream-ordered)
    const int64_t tiles = (n + kBalTile - 1) / kBalTile;
    uint32_t *statusA = c->alt_vals, *statusB = c->alt_vals + tiles;     // tiles <= n / 2
    uint32_t *ticket = c->tile_counter + kMaxPasses;
    SPH_CUDA_TRY(c, cudaMemsetAsync(ctl, 0, sizeof(BalCtl), c->stream));
    if (bal_hash) SPH_CUDA_TRY(c, cudaMemsetAsync(bal_hash, 0, sizeof(int32_t) * (size_t)n, c->stream));
    const int G = c->params.n_owners, NT = ptype ? n_types : 1, typed = ptype != nullptr;
    if (n > 0 && G > 1) {
        const int blocks = (int)min((int64_t)c->num_sms * 8, (n + 255) / 256);
        bal_sums_kernel<<<blocks, 256, 0, c->stream>>>(n, p4, owner, ptype, ctl);
        SPH_CHECK_LAUNCH(c);
        for (int T = 0; T < NT; ++T)
            for (int A = 0; A < G; ++A)
                for (int B = A + 1; B < G; ++B) {
                    bal_pair_begin_kernel<<<1, 256, 0, c->stream>>>(ctl, A, B, T, typed, alpha, statusA, 2 * tiles,
                                                                   ticket);
                    SPH_CHECK_LAUNCH(c);
                    bal_hash_kernel<<<blocks, 256, 0, c->stream>>>(n, p4, owner, ptype, ctl, A, B, T, hmax, bh, code);
                    SPH_CHECK_LAUNCH(c);
                    bal_pair_select_kernel<<<1, kBalBins, 0, c->stream>>>(ctl, hmax);
                    SPH_CHECK_LAUNCH(c);
                    bal_swap_kernel<<<(unsigned)tiles, kBalThreads, 0, c->stream>>>(n, p4, owner, code, ctl, A, B, T,
                                                                                  statusA, statusB, ticket);
                    SPH_CHECK_LAUNCH(c);
                }
    }
    bal_finish_kernel<<<1, 1, 0, c->stream>>>(ctl, swapped);
    SPH_CHECK_LAUNCH(c);
    return SPH_OK;
}

size_t balance_scratch_bytes() { return sizeof(BalCtl); }

}  // namespace sphb
