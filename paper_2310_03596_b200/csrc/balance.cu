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

// one thread: centres of gravity of the pair, validity, cleared histograms
__global__ void bal_pair_begin_kernel(BalCtl *ctl, int A, int B, int T, int typed, double alpha)
{
    for (int i = threadIdx.x; i < 2 * kBalBins; i += blockDim.x) (&ctl->hist[0][0])[i] = 0;
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

__global__ void __launch_bounds__(256)
bal_hash_kernel(int64_t n, const float4 *__restrict__ posm, const int32_t *__restrict__ owner,
                const int32_t *__restrict__ ptype, BalCtl *ctl, int A, int B, int T, int hmax,
                int32_t *__restrict__ bal_hash)
{
    __shared__ uint32_t s_hist[2][kBalBins];
    for (int i = threadIdx.x; i < 2 * kBalBins; i += blockDim.x) (&s_hist[0][0])[i] = 0;
    __syncthreads();
    if (ctl->valid) {
        for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
             i += (int64_t)gridDim.x * blockDim.x) {
            const int o = owner[i];
            if (o != A && o != B) continue;
            if (ptype && ptype[i] != T) continue;
            const float4 p = posm[i];
            const int side = o == A ? 0 : 1;
            const int32_t hv = side == 0 ? balance_hash(p, ctl->cgA, ctl->cgB, hmax)
                                         : balance_hash(p, ctl->cgB, ctl->cgA, hmax);
            bal_hash[i] = hv;
            if (hv > 0) atomicAdd(&s_hist[side][hv], 1u);
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

// indicator arrays of the threshold ties (their exclusive scans rank the ties by id)
__global__ void __launch_bounds__(256)
bal_ties_kernel(int64_t n, const int32_t *__restrict__ owner, const int32_t *__restrict__ ptype,
                const int32_t *__restrict__ bal_hash, const BalCtl *ctl, int A, int B, int T,
                uint32_t *__restrict__ tieA, uint32_t *__restrict__ tieB)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t a = 0, b = 0;
    if (ctl->valid) {
        const int o = owner[i];
        const bool mine = !ptype || ptype[i] == T;
        if (mine && o == A) a = (uint32_t)bal_hash[i] == ctl->thrA;
        else if (mine && o == B) b = (uint32_t)bal_hash[i] == ctl->thrB;
    }
    tieA[i] = a;
    tieB[i] = b;
}

__global__ void __launch_bounds__(256)
bal_swap_kernel(int64_t n, const float4 *__restrict__ posm, int32_t *__restrict__ owner,
                const int32_t *__restrict__ ptype, const int32_t *__restrict__ bal_hash, BalCtl *ctl, int A,
                int B, int T, const uint32_t *__restrict__ rankA, const uint32_t *__restrict__ rankB)
{
    // D = (coordinates leaving A) - (coordinates leaving B): sum[A] -= D, sum[B] += D.  Exact
    // integer sums, so the order of the block and grid reductions does not matter.
    __shared__ long long s_d[3];
    if (threadIdx.x < 3) s_d[threadIdx.x] = 0;
    __syncthreads();
    if (!ctl->valid) return;   // uniform over the grid
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    long long f[3] = {0, 0, 0};
    if (i < n) {
        const int o = owner[i];
        if ((o == A || o == B) && (!ptype || ptype[i] == T)) {
            const uint32_t hv = (uint32_t)bal_hash[i];
            const uint32_t thr = o == A ? ctl->thrA : ctl->thrB, quota = o == A ? ctl->quotaA : ctl->quotaB;
            const uint32_t rank = o == A ? rankA[i] : rankB[i];
            if (hv > 0 && (hv > thr || (hv == thr && rank < quota))) {
                owner[i] = o == A ? B : A;
                const float4 p = posm[i];
                const long long sgn = o == A ? 1 : -1;
                f[0] = sgn * fixed16(p.x); f[1] = sgn * fixed16(p.y); f[2] = sgn * fixed16(p.z);
            }
        }
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
    int32_t *bh = bal_hash ? bal_hash : reinterpret_cast<int32_t *>(c->s_hash);
    uint32_t *tieA = c->alt_keys, *tieB = c->alt_vals, *rankA = c->s_sorted_hash, *rankB = c->s_perm;
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
                    bal_pair_begin_kernel<<<1, 256, 0, c->stream>>>(ctl, A, B, T, typed, alpha);
                    SPH_CHECK_LAUNCH(c);
                    bal_hash_kernel<<<blocks, 256, 0, c->stream>>>(n, p4, owner, ptype, ctl, A, B, T, hmax, bh);
                    SPH_CHECK_LAUNCH(c);
                    bal_pair_select_kernel<<<1, kBalBins, 0, c->stream>>>(ctl, hmax);
                    SPH_CHECK_LAUNCH(c);
                    bal_ties_kernel<<<div_up(n, 256), 256, 0, c->stream>>>(n, owner, ptype, bh, ctl, A, B, T, tieA, tieB);
                    SPH_CHECK_LAUNCH(c);
                    int rc = launch_scan_exclusive(c, n, tieA, rankA, nullptr);
                    if (rc != SPH_OK) return rc;
                    rc = launch_scan_exclusive(c, n, tieB, rankB, nullptr);
                    if (rc != SPH_OK) return rc;
                    bal_swap_kernel<<<div_up(n, 256), 256, 0, c->stream>>>(n, p4, owner, ptype, bh, ctl, A, B, T,
                                                                          rankA, rankB);
                    SPH_CHECK_LAUNCH(c);
                }
    }
    bal_finish_kernel<<<1, 1, 0, c->stream>>>(ctl, swapped);
    SPH_CHECK_LAUNCH(c);
    return SPH_OK;
}

size_t balance_scratch_bytes() { return sizeof(BalCtl); }

}  // namespace sphb
