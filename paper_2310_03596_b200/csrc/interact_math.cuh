// Pair arithmetic shared by the two interaction kernels (O6-O8, fp32).
//
// Wendland C2, support 2h: grad_i W_ij = F(r) x_ij, F(r) = cF (1 - r/2h)^3, cF = -5 alpha / h^2.
// The constant cF is applied once per particle; per pair only t^3 is formed.
//   drho_i = sum_j m_j (v_i - v_j).gradW        = -cF sum (m_j t^3 x_ij) . dv,  dv = v_j - v_i
//   L_ab   = sum_j V_j dv_a gradW_b             =  cF sum dv_a (V_j t^3 x_ij)_b
//   acc_i  = sum_j m_j (S_i + S_j) gradW        =  cF [ S_i g + sum S_j (m_j t^3 x_ij) ],
//            g = sum m_j t^3 x_ij,  S = sigma / rho^2,  V = m / rho.
#pragma once
#include "sph_internal.cuh"

namespace sphb {

struct InteractIn {
    const float4 *posm, *velr;
    const float *sig[6];
    const int32_t *owner;   // sorted owner labels; only read by the split passes (NEXT-3)
    const float *h;         // sorted per-particle smoothing lengths (NEXT-4), NULL = uniform
};

// Which neighbours a pass takes: 0 = all (steps e and f as one loop),
// 1 = step e alone (same owner label), 2 = step f alone (other owner labels).
constexpr int kPassAll = 0, kPassLocal = 1, kPassRemote = 2;
// 3 = both split passes from ONE neighbour search (two rate sets; sph_interact_ef)
constexpr int kPassBoth = 3;
struct InteractOut {
    float *drho;          // rates, indexed by sorted position; all three NULL = not wanted
    float4 *acc;
    float *dsig[6];
    // optional fused integration (step g, O9): the epilogue advances the particle and scatters
    // it to id order through perm -- inside sph_step this removes the integrate pass (156 B per
    // particle) and, when the caller does not ask for the rates, their 44 B store as well
    const uint32_t *perm;  // NULL = no fused integration
    float dt;
    float4 *o_posm, *o_velr;
    float *o_sig[6];
};

// MUFU.SQRT: one instruction, sqrt(0) = 0 so coincident particles need no clamp (S15)
__device__ __forceinline__ float sqrt_approx(float x)
{
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// NEXT-4 (per-particle smoothing lengths, reading H2): pair length h_ij = (h_i + h_j) / 2.
// Returns 1 / (h_i + h_j) = 1 / (2 h_ij) (MUFU.RCP + one Newton step) and h_ij^-5 in *ih5:
// grad W = -(105 / 16 pi) h_ij^-5 (1 - r / 2 h_ij)^3 x_ij, the constant is applied per particle.
__device__ __forceinline__ float pair_inv_2h(float hi, float hj, float *ih5)
{
    const float hs = hi + hj;
    float inv;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(inv) : "f"(hs));
    inv = inv * fmaf(-hs, inv, 2.0f);
    const float ih = 2.0f * inv, ih2 = ih * ih;
    *ih5 = ih2 * ih2 * ih;
    return inv;
}

struct PairAccum {
    float dr;          // sum dv . mx
    float L[9];        // sum dv_a * wx_b
    float g[3];        // sum mx
    float a[3];        // sum S_j mx
    __device__ __forceinline__ void clear()
    {
        dr = 0.f;
#pragma unroll
        for (int i = 0; i < 9; ++i) L[i] = 0.f;
#pragma unroll
        for (int i = 0; i < 3; ++i) { g[i] = 0.f; a[i] = 0.f; }
    }
    // S = (xx, yy, zz, xy, xz, yz) of sigma_j / rho_j^2
    // scale = 1 (uniform h: the constant cF is applied once per particle) or h_ij^-5 (NEXT-4)
    __device__ __forceinline__ void add(float dx, float dy, float dz, float r2, float mj, float Vj,
                                        float dvx, float dvy, float dvz, const float (&S)[6],
                                        float half_inv_h, float scale = 1.0f)
    {
        const float r = sqrt_approx(r2);              // coincident particles: r = 0, gradW = 0 (S15)
        const float t = fmaxf(fmaf(r, -half_inv_h, 1.0f), 0.0f);  // W = 0 beyond the support
        const float F = t * t * t * scale;
        const float wm = mj * F, wV = Vj * F;
        const float mx = wm * dx, my = wm * dy, mz = wm * dz;
        const float wx = wV * dx, wy = wV * dy, wz = wV * dz;
        dr = fmaf(dvx, mx, dr); dr = fmaf(dvy, my, dr); dr = fmaf(dvz, mz, dr);
        L[0] = fmaf(dvx, wx, L[0]); L[1] = fmaf(dvx, wy, L[1]); L[2] = fmaf(dvx, wz, L[2]);
        L[3] = fmaf(dvy, wx, L[3]); L[4] = fmaf(dvy, wy, L[4]); L[5] = fmaf(dvy, wz, L[5]);
        L[6] = fmaf(dvz, wx, L[6]); L[7] = fmaf(dvz, wy, L[7]); L[8] = fmaf(dvz, wz, L[8]);
        g[0] += mx; g[1] += my; g[2] += mz;
        a[0] = fmaf(S[0], mx, a[0]); a[0] = fmaf(S[3], my, a[0]); a[0] = fmaf(S[4], mz, a[0]);
        a[1] = fmaf(S[3], mx, a[1]); a[1] = fmaf(S[1], my, a[1]); a[1] = fmaf(S[5], mz, a[1]);
        a[2] = fmaf(S[4], mx, a[2]); a[2] = fmaf(S[5], my, a[2]); a[2] = fmaf(S[2], mz, a[2]);
    }
};

// ---- packed fp32 pairs (sm_100a: FFMA2 / FADD2 / FMUL2, one issue slot for two lanes' worth of
// fp32 work; a scalar operand is broadcast by the hardware, SASS `R.F32`) ------------------------
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk(float lo, float hi)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ f32x2 bc(float s) { return pk(s, s); }
__device__ __forceinline__ float lo_of(f32x2 v)
{
    float a, b;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v));
    return a;
}
__device__ __forceinline__ float hi_of(f32x2 v)
{
    float a, b;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v));
    return b;
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
// in-place accumulate forms (acc += a * b, acc += a): the read-modify-write of one PTX register
// keeps ptxas from ping-ponging the accumulators between two register sets (it closed the loop
// of phase 2 with 14 moves per round before)
__device__ __forceinline__ void fma2_acc(f32x2 &acc, f32x2 a, f32x2 b)
{
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(a), "l"(b));
}
__device__ __forceinline__ void add2_acc(f32x2 &acc, f32x2 a)
{
    asm("add.rn.f32x2 %0, %0, %1;" : "+l"(acc) : "l"(a));
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

// The same sums as PairAccum, held as fp32 pairs so that one pair costs 30 issue slots instead
// of 46 (the FMA pipe does the same work; the freed slots go to the loads and the bookkeeping).
// Neighbour record (tiled kernel): A = x, y, z, |p|^2;  B = vx, vy, vz, Szz;
// C = Sxx, Sxy, Sxy, Syy;  D = Sxz, Syz, m, V   with S = sigma / rho^2, V = m / rho.
struct PairAccum2 {
    f32x2 dr2;            // (sum dvx mx, sum dvy my)
    float drz;            // sum dvz mz
    f32x2 Lx, Ly, Lz;     // rows a = x, y, z of L, columns (x, y):  sum dv_a (wx, wy)
    f32x2 Lc;             // column z of rows x, y:                 sum (dvx, dvy) wz
    float Lzz;
    f32x2 g2;             // (sum mx, sum my)
    float gz;
    f32x2 a2;             // (sum (S m)_x, sum (S m)_y)
    f32x2 az2;            // (sum Sxz mx, sum Syz my)
    float azz;            // sum Szz mz
    __device__ __forceinline__ void clear()
    {
        dr2 = Lx = Ly = Lz = Lc = g2 = a2 = az2 = 0ull;
        drz = Lzz = gz = azz = 0.f;
    }
    // tp = target position (tile-local), tv = target velocity; pa..pd = the neighbour record.
    // VH (NEXT-4): C.z carries h_j instead of the second copy of Sxy, hi = the target's length;
    // returns r^2 - (h_i + h_j)^2 + support2-free form: see the caller (pair counting).
    template <bool VH = false>
    __device__ __forceinline__ float add(f32x2 tpxy, float tpz, f32x2 tvxy, float tvz, const float4 &pa,
                                         const float4 &pb, const float4 &pc, const float4 &pd,
                                         float neg_half_inv_h, float hi = 0.f)
    {
        const f32x2 dxy = sub2(tpxy, pk(pa.x, pa.y));
        const float dz = tpz - pa.z;
        const f32x2 sq = mul2(dxy, dxy);
        const float r2 = fmaf(dz, dz, lo_of(sq)) + hi_of(sq);
        const float r = sqrt_approx(r2);              // coincident particles: r = 0, gradW = 0 (S15)
        float F;
        if (VH) {
            float ih5;
            const float inv = pair_inv_2h(hi, pc.z, &ih5);
            const float t = fmaxf(fmaf(r, -inv, 1.0f), 0.0f);     // W = 0 beyond 2 h_ij
            F = t * t * t * ih5;
        } else {
            const float t = fmaxf(fmaf(r, neg_half_inv_h, 1.0f), 0.0f);  // W = 0 beyond the support
            F = t * t * t;
        }
        const f32x2 wmV = mul2(bc(F), pk(pd.z, pd.w));            // (m F, V F)
        const f32x2 mxy = mul2(bc(lo_of(wmV)), dxy);              // m F (dx, dy)
        const f32x2 wxy = mul2(bc(hi_of(wmV)), dxy);              // V F (dx, dy)
        const f32x2 mwz = mul2(bc(dz), wmV);                      // (m F dz, V F dz)
        const float mz = lo_of(mwz), wz = hi_of(mwz);
        const f32x2 dvxy = sub2(pk(pb.x, pb.y), tvxy);
        const float dvz = pb.z - tvz;
        fma2_acc(dr2, dvxy, mxy);
        drz = fmaf(dvz, mz, drz);
        fma2_acc(Lx, bc(lo_of(dvxy)), wxy);
        fma2_acc(Ly, bc(hi_of(dvxy)), wxy);
        fma2_acc(Lz, bc(dvz), wxy);
        fma2_acc(Lc, bc(wz), dvxy);
        Lzz = fmaf(dvz, wz, Lzz);
        add2_acc(g2, mxy);
        gz += mz;
        fma2_acc(a2, bc(lo_of(mxy)), pk(pc.x, pc.y));
        fma2_acc(a2, bc(hi_of(mxy)), pk(VH ? pc.y : pc.z, pc.w));
        fma2_acc(a2, bc(mz), pk(pd.x, pd.y));
        fma2_acc(az2, pk(pd.x, pd.y), mxy);
        azz = fmaf(pb.w, mz, azz);
        return r2;
    }
    // unpack into the 16 sums of PairAccum (same order: dr, L[9] row-major, g[3], a[3])
    __device__ __forceinline__ void unpack(float (&v)[16]) const
    {
        v[0] = lo_of(dr2) + hi_of(dr2) + drz;
        v[1] = lo_of(Lx); v[2] = hi_of(Lx); v[3] = lo_of(Lc);
        v[4] = lo_of(Ly); v[5] = hi_of(Ly); v[6] = hi_of(Lc);
        v[7] = lo_of(Lz); v[8] = hi_of(Lz); v[9] = Lzz;
        v[10] = lo_of(g2); v[11] = hi_of(g2); v[12] = gz;
        v[13] = lo_of(a2); v[14] = hi_of(a2); v[15] = lo_of(az2) + hi_of(az2) + azz;
    }
};

// Per-particle epilogue: scale by cF, add the S_i term, form the stress rate (O8) and store.
// pos_i (x, y, z, m in the caller's coordinates) and vel_i are only read by the fused integration.
__device__ __forceinline__ void finish_particle(const PairAccum &A, const float (&sig_i)[6],
                                                float rho_i, const Consts &k, const InteractOut &out,
                                                int64_t i, const float4 &pos_i, float vx_i, float vy_i,
                                                float vz_i)
{
    const float cF = k.cF;
    const float ir = 1.0f / rho_i;
    const float ir2 = ir * ir;
    const float Sxx = sig_i[0] * ir2, Syy = sig_i[1] * ir2, Szz = sig_i[2] * ir2;
    const float Sxy = sig_i[3] * ir2, Sxz = sig_i[4] * ir2, Syz = sig_i[5] * ir2;
    float4 acc;
    acc.x = cF * (A.a[0] + Sxx * A.g[0] + Sxy * A.g[1] + Sxz * A.g[2]);
    acc.y = cF * (A.a[1] + Sxy * A.g[0] + Syy * A.g[1] + Syz * A.g[2]);
    acc.z = cF * (A.a[2] + Sxz * A.g[0] + Syz * A.g[1] + Szz * A.g[2]);
    acc.w = 0.f;
    const float drho = -cF * A.dr;
    if (out.drho) {
        out.drho[i] = drho;
        out.acc[i] = acc;
    }
    float L[9];
#pragma unroll
    for (int q = 0; q < 9; ++q) L[q] = cF * A.L[q];
    // D = sym(L), Om = skew(L);  dsig = K trD I + 2G (D - trD/3 I) + Om sig - sig Om
    const float Dxx = L[0], Dyy = L[4], Dzz = L[8];
    const float Dxy = 0.5f * (L[1] + L[3]), Dxz = 0.5f * (L[2] + L[6]), Dyz = 0.5f * (L[5] + L[7]);
    const float Oxy = 0.5f * (L[1] - L[3]), Oxz = 0.5f * (L[2] - L[6]), Oyz = 0.5f * (L[5] - L[7]);
    const float trD = Dxx + Dyy + Dzz;
    const float vol = (k.K - (2.0f / 3.0f) * k.G) * trD;
    const float G2 = 2.0f * k.G;
    const float sxx = sig_i[0], syy = sig_i[1], szz = sig_i[2], sxy = sig_i[3], sxz = sig_i[4],
                syz = sig_i[5];
    // (Om s - s Om) for skew Om = [[0,Oxy,Oxz],[-Oxy,0,Oyz],[-Oxz,-Oyz,0]] and symmetric s
    const float Jxx = 2.0f * (Oxy * sxy + Oxz * sxz);
    const float Jyy = 2.0f * (-Oxy * sxy + Oyz * syz);
    const float Jzz = -2.0f * (Oxz * sxz + Oyz * syz);
    const float Jxy = Oxy * (syy - sxx) + Oxz * syz + Oyz * sxz;
    const float Jxz = Oxz * (szz - sxx) + Oxy * syz - Oyz * sxy;
    const float Jyz = Oyz * (szz - syy) - Oxy * sxz - Oxz * sxy;
    float ds[6];
    ds[0] = vol + G2 * Dxx + Jxx;
    ds[1] = vol + G2 * Dyy + Jyy;
    ds[2] = vol + G2 * Dzz + Jzz;
    ds[3] = G2 * Dxy + Jxy;
    ds[4] = G2 * Dxz + Jxz;
    ds[5] = G2 * Dyz + Jyz;
    if (out.drho) {
#pragma unroll
        for (int c = 0; c < 6; ++c) out.dsig[c][i] = ds[c];
    }
    if (out.perm) {  // symplectic Euler (O9), result scattered to id order
        const float dt = out.dt;
        const int64_t dst = (int64_t)__ldg(out.perm + i);
        float4 vn, pn;
        vn.x = fmaf(dt, acc.x, vx_i);
        vn.y = fmaf(dt, acc.y, vy_i);
        vn.z = fmaf(dt, acc.z, vz_i);
        vn.w = fmaf(dt, drho, rho_i);
        pn.x = fmaf(dt, vn.x, pos_i.x);
        pn.y = fmaf(dt, vn.y, pos_i.y);
        pn.z = fmaf(dt, vn.z, pos_i.z);
        pn.w = pos_i.w;
        out.o_posm[dst] = pn;
        out.o_velr[dst] = vn;
#pragma unroll
        for (int c = 0; c < 6; ++c) out.o_sig[c][dst] = fmaf(dt, ds[c], sig_i[c]);
    }
}

// One particle of the plain global-memory walk over its 27-bucket stencil (9 contiguous runs).
// Used by the direct kernel and as the fallback of the tiled kernel.  Returns the number of
// accepted ordered pairs (j != i).
__device__ __forceinline__ uint32_t direct_particle(int64_t i, int cx, int cy, int cz,
                                                    const InteractIn &in, const uint32_t *__restrict__ cs,
                                                    const uint32_t *__restrict__ ce, const Grid &g,
                                                    const Consts &k, const InteractOut &out,
                                                    int mode = kPassAll)
{
    const int32_t oi = mode != kPassAll ? in.owner[i] : 0;
    const float hi = in.h ? in.h[i] : 0.f;   // NEXT-4: per-particle smoothing length
    const float4 pi = in.posm[i];
    const float4 vi = in.velr[i];
    PairAccum A;
    A.clear();
    uint32_t pairs = 0;
    const int x0 = max(cx - 1, 0), x1 = min(cx + 1, g.nx - 1);
    for (int dz = -1; dz <= 1; ++dz) {
        const int z = cz + dz;
        if (z < 0 || z >= g.nz) continue;
        for (int dy = -1; dy <= 1; ++dy) {
            const int y = cy + dy;
            if (y < 0 || y >= g.ny) continue;
            const uint32_t row = (uint32_t)g.nx * ((uint32_t)y + (uint32_t)g.ny * (uint32_t)z);
            const uint32_t jb = cs[row + x0], je = ce[row + x1];
            for (uint32_t j = jb; j < je; ++j) {
                const float4 pj = in.posm[j];
                const float dx = pi.x - pj.x, dy_ = pi.y - pj.y, dz_ = pi.z - pj.z;
                const float r2 = dx * dx + dy_ * dy_ + dz_ * dz_;
                if (mode != kPassAll && ((in.owner[j] == oi) != (mode == kPassLocal))) continue;
                float sup2 = k.support2, hinv = k.half_inv_h, scale = 1.0f;
                if (in.h) {   // pair length h_ij = (h_i + h_j) / 2, support 2 h_ij (reading H2)
                    const float hs = hi + in.h[j];
                    sup2 = hs * hs;
                    hinv = pair_inv_2h(hi, in.h[j], &scale);
                }
                if (r2 < sup2 && j != (uint32_t)i) {
                    const float4 vj = in.velr[j];
                    const float inv_rho = 1.0f / vj.w;
                    const float Vj = pj.w * inv_rho;
                    const float ir2 = inv_rho * inv_rho;
                    float Sj[6];
#pragma unroll
                    for (int c = 0; c < 6; ++c) Sj[c] = in.sig[c][j] * ir2;
                    A.add(dx, dy_, dz_, r2, pj.w, Vj, vj.x - vi.x, vj.y - vi.y, vj.z - vi.z, Sj,
                          hinv, scale);
                    ++pairs;
                }
            }
        }
    }
    float si[6];
#pragma unroll
    for (int c = 0; c < 6; ++c) si[c] = in.sig[c][i];
    finish_particle(A, si, vi.w, k, out, i, pi, vi.x, vi.y, vi.z);
    return pairs;
}

int launch_interact_direct(sph_ctx *c, int64_t n, const InteractIn &in, const uint32_t *sorted_hash,
                           const uint32_t *cs, const uint32_t *ce, const InteractOut &out,
                           unsigned long long *pair_count, int mode);
int launch_interact_tiled(sph_ctx *c, int64_t n, const InteractIn &in, const uint32_t *sorted_hash,
                          const uint32_t *cs, const uint32_t *ce, const InteractOut &out,
                          unsigned long long *pair_count, int mode, const InteractOut *out_f = nullptr);

}  // namespace sphb
