// Stage 4b: explicit integration, symplectic Euler (step g; reading S18).
// rho += dt drho; v += dt a; sigma += dt dsig; x += dt v(new).  HBM-bound streaming kernel behind
// the sph_integrate entry point.  sph_step does not launch it: there the epilogue of the
// interaction kernel integrates and scatters to id order (interact_math.cuh, finish_particle).
#include "sph_internal.cuh"

namespace sphb {

struct IntegrateArgs {
    const float4 *posm, *velr, *acc;
    const float *sig[6], *dsig[6], *drho;
    const int32_t *owner;
    float4 *o_posm, *o_velr;
    float *o_sig[6];
    int32_t *o_owner;
    const uint32_t *perm;  // NULL: elementwise
};

__global__ void __launch_bounds__(256) integrate_kernel(int64_t n, float dt, IntegrateArgs a)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const float4 p = a.posm[k];
    const float4 v = a.velr[k];
    const float4 ac = __ldcs(a.acc + k);
    const float dr = __ldcs(a.drho + k);
    float s[6], ds[6];
#pragma unroll
    for (int c = 0; c < 6; ++c) { s[c] = a.sig[c][k]; ds[c] = __ldcs(a.dsig[c] + k); }
    const int64_t dst = a.perm ? (int64_t)__ldcs(a.perm + k) : k;
    float4 vn, pn;
    vn.x = fmaf(dt, ac.x, v.x);
    vn.y = fmaf(dt, ac.y, v.y);
    vn.z = fmaf(dt, ac.z, v.z);
    vn.w = fmaf(dt, dr, v.w);
    pn.x = fmaf(dt, vn.x, p.x);
    pn.y = fmaf(dt, vn.y, p.y);
    pn.z = fmaf(dt, vn.z, p.z);
    pn.w = p.w;
    a.o_posm[dst] = pn;
    a.o_velr[dst] = vn;
#pragma unroll
    for (int c = 0; c < 6; ++c) a.o_sig[c][dst] = fmaf(dt, ds[c], s[c]);
    if (a.o_owner) a.o_owner[dst] = a.owner[k];  // labels never change; copied only out of place
}

int launch_integrate(sph_ctx *c, int64_t n, float dt, const sph_state *in, const float *drho,
                     const float *acc, const float *const dsig[6], const sph_state *out,
                     const uint32_t *scatter_perm)
{
    if (n == 0) return SPH_OK;
    IntegrateArgs a;
    a.posm = reinterpret_cast<const float4 *>(in->posm);
    a.velr = reinterpret_cast<const float4 *>(in->velr);
    a.acc = reinterpret_cast<const float4 *>(acc);
    a.drho = drho;
    a.owner = in->owner;
    a.o_posm = reinterpret_cast<float4 *>(out->posm);
    a.o_velr = reinterpret_cast<float4 *>(out->velr);
    a.o_owner = (scatter_perm || out->owner == in->owner) ? nullptr : out->owner;
    a.perm = scatter_perm;
    for (int i = 0; i < 6; ++i) { a.sig[i] = in->sig[i]; a.dsig[i] = dsig[i]; a.o_sig[i] = out->sig[i]; }
    integrate_kernel<<<div_up(n, 256), 256, 0, c->stream>>>(n, dt, a);
    SPH_CHECK_LAUNCH(c);
    return SPH_OK;
}

}  // namespace sphb
