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
               float4 *__restrict__ recB, float4 *__restrict__ recC, float4 *__restrict__ recD)
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
        recC[k] = make_float4(s[0] * ir2, sxy, sxy, s[1] * ir2);
        recD[k] = make_float4(s[4] * ir2, s[5] * ir2, p.w, p.w * inv_rho);
    }
}

int launch_reorder(sph_ctx *c, int64_t n, const uint32_t *perm, const sph_state *in,
                   const sph_state *out)
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
        reorder_kernel<true><<<div_up(n, 256), 256, 0, c->stream>>>(n, perm, a, b, c->rec_B, c->rec_C, c->rec_D);
    else
        reorder_kernel<false><<<div_up(n, 256), 256, 0, c->stream>>>(n, perm, a, b, nullptr, nullptr, nullptr);
    SPH_CHECK_LAUNCH(c);
    c->rec_fresh = pack;
    return SPH_OK;
}

}  // namespace sphb
