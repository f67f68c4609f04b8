// Stage 4a dispatcher: picks the shared-memory tiled kernel, or the direct global-memory kernel
// when forced (SPH_FLAG_INTERACT_DIRECT).  pair_count accumulates (callers zero it).
#include "sph_internal.cuh"
#include "interact_math.cuh"

namespace sphb {

int launch_interact(sph_ctx *c, int64_t n, const sph_state *sorted, const uint32_t *sorted_hash,
                    const uint32_t *cs, const uint32_t *ce, float *drho, float *acc,
                    float *const dsig[6], unsigned long long *pair_count, const sph_state *fuse_out,
                    const uint32_t *perm, float dt, int mode, const float *sorted_h, float *drho_f, float *acc_f,
                    float *const dsig_f[6])
{
    if (n == 0) return SPH_OK;
    InteractIn in;
    InteractOut out;
    in.posm = reinterpret_cast<const float4 *>(sorted->posm);
    in.velr = reinterpret_cast<const float4 *>(sorted->velr);
    in.owner = sorted->owner;
    in.h = sorted_h;
    out.drho = drho;   // NULL (with fuse_out set): the rates are not stored
    out.acc = reinterpret_cast<float4 *>(acc);
    for (int i = 0; i < 6; ++i) { in.sig[i] = sorted->sig[i]; out.dsig[i] = dsig ? dsig[i] : nullptr; }
    out.perm = nullptr;
    out.dt = dt;
    out.o_posm = out.o_velr = nullptr;
    for (int i = 0; i < 6; ++i) out.o_sig[i] = nullptr;
    if (fuse_out) {    // step g in the epilogue, scattered to id order through perm
        out.perm = perm;
        out.o_posm = reinterpret_cast<float4 *>(fuse_out->posm);
        out.o_velr = reinterpret_cast<float4 *>(fuse_out->velr);
        for (int i = 0; i < 6; ++i) out.o_sig[i] = fuse_out->sig[i];
    }
    if (mode == kPassBoth) {
        // steps e and f from one neighbour search: a second set of rate arrays (step f)
        InteractOut of = out;
        of.drho = drho_f;
        of.acc = reinterpret_cast<float4 *>(acc_f);
        for (int i = 0; i < 6; ++i) of.dsig[i] = dsig_f[i];
        if (c->params.flags & SPH_FLAG_INTERACT_DIRECT) {
            int rc = launch_interact_direct(c, n, in, sorted_hash, cs, ce, out, pair_count, kPassLocal);
            if (rc != SPH_OK) return rc;
            return launch_interact_direct(c, n, in, sorted_hash, cs, ce, of, pair_count + 1, kPassRemote);
        }
        return launch_interact_tiled(c, n, in, sorted_hash, cs, ce, out, pair_count, mode, &of);
    }
    if (c->params.flags & SPH_FLAG_INTERACT_DIRECT)
        return launch_interact_direct(c, n, in, sorted_hash, cs, ce, out, pair_count, mode);
    return launch_interact_tiled(c, n, in, sorted_hash, cs, ce, out, pair_count, mode);
}

}  // namespace sphb
