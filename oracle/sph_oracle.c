/*
 * sph_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded CPU restatement of the per-iteration hot path of the
 * particle-decomposition SPH scheme of Unfer, Colle & Limido (arxiv 2310.03596,
 * /root/reference/PAPER.md).  Every real quantity is fp64 (fp32 inputs are widened), except the
 * bucket hash, whose operation sequence is pinned in fp32 (reading S2) so that the
 * integer outputs have exactly one correct value.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this file.  It shares no code, header, table or constant with the CUDA path under
 * paper_2310_03596_b200/csrc/ and includes nothing from include/.
 *
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math -shared -fPIC (see oracle/build.py).
 *
 * Citations: "PAPER.md:N" = line N of /root/reference/PAPER.md; "S#"/"O#"/"I#" = the readings,
 * oracle steps and invariants listed in DESIGN.md section 3 (taken from SURVEY.md section 8(c)).
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): brute-force O(N^2) neighbour / owner
 * enumeration, kernel normalisation integral and dW/dr by finite differences, exact momentum
 * conservation, zero rates for uniform translation, continuum limits of the gradient operators
 * (sign and index conventions), Hooke / Jaumann textbook cases, expm() finite rotation,
 * cell-table identities, sort vs numpy.lexsort, hash at bucket faces, per-owner send buffers vs a
 * stable numpy argsort.  No function is unpinned.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_GARBAGE 0xFFFFFFFFu /* S8: "some garbage collector hash" := 2^32-1 */

/* ------------------------------------------------------------------------------------------
 * O1  Bucket hash ("cubic buckets of size 2h ... Each particle is given a hash
 * number corresponding to the bucket in which it is located"; PAPER.md:19 step a).
 * Reading S1: linear index, x fastest.  Reading S2: the fp32 sequence sub, mul, floor, clamp.
 * posm is [n][4] = x,y,z,m.
 * ---------------------------------------------------------------------------------------- */
void orc_hash(int64_t n, const float *posm, const float *origin, const int32_t *dims, float h,
              uint32_t *hash)
{
    const float edge = 2.0f * h;    /* bucket edge 2h */
    const float inv = 1.0f / edge;  /* rounded once, fp32 (S2)      */
    for (int64_t i = 0; i < n; ++i) {
        uint32_t c[3];
        for (int a = 0; a < 3; ++a) {
            float t = posm[4 * i + a] - origin[a];
            float u = t * inv;
            float f = floorf(u);
            float top = (float)(dims[a] - 1);
            if (f < 0.0f) f = 0.0f;      /* S3: out-of-grid particles are clamped */
            if (f > top) f = top;
            c[a] = (uint32_t)(int32_t)f;
        }
        hash[i] = c[0] + (uint32_t)dims[0] * (c[1] + (uint32_t)dims[1] * c[2]);
    }
}

/* ------------------------------------------------------------------------------------------
 * O2  Sort ("The particles are then sorted with respect to this hash number by
 * the radix sort algorithm").  Reading S5: the key is (hash, particle id), ids are 0..n-1.
 * The oracle is the definition: a comparison sort on the pairs.
 * ---------------------------------------------------------------------------------------- */
typedef struct { uint32_t hash, id; } orc_pair;

static int orc_pair_cmp(const void *a, const void *b)
{
    const orc_pair *p = (const orc_pair *)a, *q = (const orc_pair *)b;
    if (p->hash != q->hash) return p->hash < q->hash ? -1 : 1;
    if (p->id != q->id) return p->id < q->id ? -1 : 1;
    return 0;
}

int orc_sort(int64_t n, const uint32_t *hash, uint32_t *sorted_hash, uint32_t *perm)
{
    orc_pair *p = (orc_pair *)malloc((size_t)(n > 0 ? n : 1) * sizeof(orc_pair));
    if (!p) return -1;
    for (int64_t i = 0; i < n; ++i) { p[i].hash = hash[i]; p[i].id = (uint32_t)i; }
    qsort(p, (size_t)n, sizeof(orc_pair), orc_pair_cmp);
    for (int64_t k = 0; k < n; ++k) { sorted_hash[k] = p[k].hash; perm[k] = p[k].id; }
    free(p);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * O3  Cell start/end tables (BASELINE.json north_star: "with cell start/end tables"; implied by
 * PAPER.md:13 "restricted to its bucket and to the surrounding buckets").  Reading S7:
 * cell_start[c] = #{k : sorted_hash[k] <  c},  cell_end[c] = #{k : sorted_hash[k] <= c}.
 * ---------------------------------------------------------------------------------------- */
void orc_cell_ranges(int64_t n, const uint32_t *sorted_hash, int64_t n_cells, uint32_t *cell_start,
                     uint32_t *cell_end)
{
    for (int64_t c = 0; c < n_cells; ++c) {
        int64_t lo = 0, hi = n; /* first k with sorted_hash[k] >= c */
        while (lo < hi) {
            int64_t mid = lo + (hi - lo) / 2;
            if ((int64_t)sorted_hash[mid] < c) lo = mid + 1; else hi = mid;
        }
        cell_start[c] = (uint32_t)lo;
        hi = n;                 /* first k with sorted_hash[k] > c */
        while (lo < hi) {
            int64_t mid = lo + (hi - lo) / 2;
            if ((int64_t)sorted_hash[mid] <= c) lo = mid + 1; else hi = mid;
        }
        cell_end[c] = (uint32_t)lo;
    }
}

/* ------------------------------------------------------------------------------------------
 * O4  Communication hash ("If particles from other GPUs are present in the
 * particle's bucket or in the surrounding buckets, the communication hash number is equal to
 * the hash number, otherwise it is equal to some garbage collector hash"; PAPER.md:22 step c).
 * Plain per-particle definition.  Readings S9 (out-of-grid buckets skipped, no wrap), S10
 * (bucket-level presence, not distance), S12 (every particle carries a label).
 * All arrays are in sorted order (index k).
 * ---------------------------------------------------------------------------------------- */
void orc_comm_hash(int64_t n, const uint32_t *sorted_hash, const int32_t *sorted_owner,
                   const int32_t *dims, const uint32_t *cell_start, const uint32_t *cell_end,
                   uint32_t *comm_hash)
{
    const int64_t nx = dims[0], ny = dims[1], nz = dims[2];
    for (int64_t k = 0; k < n; ++k) {
        const int64_t hsh = sorted_hash[k];
        const int64_t cx = hsh % nx, cy = (hsh / nx) % ny, cz = hsh / (nx * ny);
        const int32_t o = sorted_owner[k];
        int found = 0;
        for (int64_t dz = -1; dz <= 1 && !found; ++dz)
            for (int64_t dy = -1; dy <= 1 && !found; ++dy)
                for (int64_t dx = -1; dx <= 1 && !found; ++dx) {
                    const int64_t x = cx + dx, y = cy + dy, z = cz + dz;
                    if (x < 0 || x >= nx || y < 0 || y >= ny || z < 0 || z >= nz) continue;
                    const int64_t c = x + nx * (y + ny * z);
                    for (uint32_t j = cell_start[c]; j < cell_end[c]; ++j)
                        if (sorted_owner[j] != o) { found = 1; break; }
                }
        comm_hash[k] = found ? (uint32_t)hsh : ORC_GARBAGE;
    }
}

/* ------------------------------------------------------------------------------------------
 * O5  MGPU boundary particle set ("Then the particles can be sorted according to
 * this communication hash, so that the data that shall be broadcasted to the other GPUs can be
 * isolated").  The paper's algorithm is followed literally: a comparison sort of the particles
 * on the key (comm_hash, id); the boundary list is the head of that order (everything before
 * the first garbage key).  Reading S11: one global list plus per-owner counts.
 * Returns the count M; boundary_ids has room for n entries.
 * ---------------------------------------------------------------------------------------- */
int64_t orc_boundary(int64_t n, const uint32_t *comm_hash, const uint32_t *perm,
                     const int32_t *sorted_owner, int32_t n_owners, uint32_t *boundary_ids,
                     uint32_t *owner_counts)
{
    orc_pair *p = (orc_pair *)malloc((size_t)(n > 0 ? n : 1) * sizeof(orc_pair));
    int32_t *owner_of_id = (int32_t *)malloc((size_t)(n > 0 ? n : 1) * sizeof(int32_t));
    if (!p || !owner_of_id) { free(p); free(owner_of_id); return -1; }
    for (int64_t k = 0; k < n; ++k) {
        p[k].hash = comm_hash[k];
        p[k].id = perm[k];
        owner_of_id[perm[k]] = sorted_owner[k];
    }
    qsort(p, (size_t)n, sizeof(orc_pair), orc_pair_cmp);
    for (int32_t g = 0; g < n_owners; ++g) owner_counts[g] = 0;
    int64_t m = 0;
    while (m < n && p[m].hash != ORC_GARBAGE) {
        boundary_ids[m] = p[m].id;
        owner_counts[owner_of_id[p[m].id]] += 1;
        ++m;
    }
    free(p);
    free(owner_of_id);
    return m;
}

/* ------------------------------------------------------------------------------------------
 * O5b  Per-owner send buffers ("each GPU ... the data that
 * shall be broadcasted to the other GPUs can be isolated", PAPER.md:23 step d "Each GPU
 * broadcasts its MGPU boundary particle data").  In the paper every GPU isolates ITS OWN boundary
 * particles; with owner labels that is the boundary list cut into one segment per owner.
 * Definition written out: segment g = the entries of the boundary list (already in (hash, id)
 * order) whose owner is g, in list order; offsets[g] = number of entries in segments < g,
 * offsets[n_owners] = M; the packed records are the id-ordered state read at packed_ids.
 * posm / velr are [n][4], sig is [6][n] (SoA); packed sig is [6][M].
 * ---------------------------------------------------------------------------------------- */
void orc_pack_boundary(int64_t n, int64_t m, const uint32_t *boundary_ids, const int32_t *owner,
                       int32_t n_owners, const float *posm, const float *velr, const float *sig,
                       uint32_t *offsets, uint32_t *packed_ids, float *p_posm, float *p_velr,
                       float *p_sig, int32_t *p_owner)
{
    int64_t j = 0;
    for (int32_t g = 0; g < n_owners; ++g) {
        offsets[g] = (uint32_t)j;
        for (int64_t k = 0; k < m; ++k) {
            const uint32_t id = boundary_ids[k];
            if (owner[id] != g) continue;
            packed_ids[j] = id;
            for (int a = 0; a < 4; ++a) {
                p_posm[4 * j + a] = posm[4 * (int64_t)id + a];
                p_velr[4 * j + a] = velr[4 * (int64_t)id + a];
            }
            for (int c = 0; c < 6; ++c) p_sig[(int64_t)c * m + j] = sig[(int64_t)c * n + id];
            p_owner[j] = owner[id];
            ++j;
        }
    }
    offsets[n_owners] = (uint32_t)j;
}

/* ------------------------------------------------------------------------------------------
 * O5c  Per-DESTINATION send lists (second half; PAPER.md:23 step d "Each
 * GPU broadcasts its MGPU boundary particle data to the other GPUs").  The paper sends every
 * boundary particle to every other GPU; GPU g only ever uses a foreign particle that lies in the
 * own or a surrounding bucket of one of ITS particles (PAPER.md:25 step f searches the same 27
 * buckets).  Reading D1: particle k is on the list of destination g iff its owner
 * is not g and a particle owned by g lies in the 27-bucket stencil of k's bucket (bucket-level
 * test as for the communication hash, readings S9 / S10).  Each list holds particle ids in the
 * (hash, id) order of the sorted array; lists are stored back to back by ascending g,
 * dest_offsets[g] = entries of the lists before g, dest_offsets[n_owners] = total.
 * Plain per-destination, per-particle definition; all arrays in sorted order (index k).
 * dest_ids may be NULL (count only); entries beyond `cap` are counted but not stored.
 * Returns the total number of entries.
 * ---------------------------------------------------------------------------------------- */
int64_t orc_pack_destinations(int64_t n, const uint32_t *sorted_hash, const int32_t *sorted_owner,
                              const uint32_t *perm, const int32_t *dims, const uint32_t *cell_start,
                              const uint32_t *cell_end, int32_t n_owners, uint32_t *dest_offsets,
                              uint32_t *dest_ids, int64_t cap)
{
    const int64_t nx = dims[0], ny = dims[1], nz = dims[2];
    int64_t total = 0;
    for (int32_t g = 0; g < n_owners; ++g) {
        dest_offsets[g] = (uint32_t)total;
        for (int64_t k = 0; k < n; ++k) {
            if (sorted_owner[k] == g) continue; /* a GPU does not send to itself */
            const int64_t hsh = sorted_hash[k];
            const int64_t cx = hsh % nx, cy = (hsh / nx) % ny, cz = hsh / (nx * ny);
            int found = 0;
            for (int64_t dz = -1; dz <= 1 && !found; ++dz)
                for (int64_t dy = -1; dy <= 1 && !found; ++dy)
                    for (int64_t dx = -1; dx <= 1 && !found; ++dx) {
                        const int64_t x = cx + dx, y = cy + dy, z = cz + dz;
                        if (x < 0 || x >= nx || y < 0 || y >= ny || z < 0 || z >= nz) continue;
                        const int64_t c = x + nx * (y + ny * z);
                        for (uint32_t j = cell_start[c]; j < cell_end[c]; ++j)
                            if (sorted_owner[j] == g) { found = 1; break; }
                    }
            if (!found) continue;
            if (dest_ids && total < cap) dest_ids[total] = perm[k];
            ++total;
        }
    }
    dest_offsets[n_owners] = (uint32_t)total;
    return total;
}

/* ------------------------------------------------------------------------------------------
 * O6  Kernel (BASELINE.json configs[0]: "Wendland C2 kernel with support 2h"; reading S14).
 * q = r/h;  W = alpha (1 - q/2)^4 (1 + 2q),  alpha = 21 / (16 pi h^3)   for q < 2, else 0.
 * grad_i W_ij = F(r) x_ij with F(r) = (dW/dr)/r = -(5 alpha / h^2) (1 - q/2)^3.
 * ---------------------------------------------------------------------------------------- */
double orc_kernel_W(double r, double h)
{
    const double q = r / h;
    if (q >= 2.0) return 0.0;
    const double alpha = 21.0 / (16.0 * M_PI * h * h * h);
    const double t = 1.0 - 0.5 * q;
    return alpha * t * t * t * t * (1.0 + 2.0 * q);
}

double orc_kernel_F(double r, double h)
{
    const double q = r / h;
    if (q >= 2.0) return 0.0;
    const double alpha = 21.0 / (16.0 * M_PI * h * h * h);
    const double t = 1.0 - 0.5 * q;
    return -(5.0 * alpha / (h * h)) * t * t * t;
}

/* ------------------------------------------------------------------------------------------
 * O7 + O8  Interaction loops and stress rate (PAPER.md:13 neighbour search in own + surrounding
 * buckets; PAPER.md:24-25 steps e, f; "several interaction loops for one iteration";
 * BASELINE.json north_star: "density rate and momentum/stress divergence").  Readings S13-S19.
 *
 * Neighbours of i: every j != i in the 27-bucket stencil of i's bucket (out-of-grid buckets
 * skipped) with r_ij^2 < (2h)^2, compared in fp64 on the widened fp32 positions.
 *   loop 1:  Drho_i   = sum_j m_j (v_i - v_j) . grad_i W_ij
 *            L_i[a][b] = sum_j (m_j / rho_j) (v_j - v_i)_a (grad_i W_ij)_b
 *   loop 2:  a_i      = sum_j m_j (sigma_i/rho_i^2 + sigma_j/rho_j^2) . grad_i W_ij
 *   O8:      D = (L + L^T)/2, Om = (L - L^T)/2,
 *            dsig = K tr(D) I + 2G (D - tr(D)/3 I) + Om sigma - sigma Om
 *
 * All arrays are in sorted order.  posm [n][4] = x,y,z,m; velr [n][4] = vx,vy,vz,rho;
 * sig [6][n] = xx,yy,zz,xy,xz,yz.  If idx != NULL only the n_idx particles idx[] are computed
 * and outputs are indexed by position in idx (used for sampled parity at full size).
 * Outputs: drho[m], L[m][9] (row major a,b), acc[m][3], dsig[m][6]; *pair_count = number of
 * ordered accepted pairs (S25).
 * ---------------------------------------------------------------------------------------- */
static void orc_sym_load(const float *sig, int64_t n, int64_t k, double s[3][3])
{
    const double xx = sig[0 * n + k], yy = sig[1 * n + k], zz = sig[2 * n + k];
    const double xy = sig[3 * n + k], xz = sig[4 * n + k], yz = sig[5 * n + k];
    s[0][0] = xx; s[1][1] = yy; s[2][2] = zz;
    s[0][1] = s[1][0] = xy;
    s[0][2] = s[2][0] = xz;
    s[1][2] = s[2][1] = yz;
}

/* which = 0: every neighbour (steps e and f together, the one-GPU loop);
 * which = 1: step e alone, "local particle interaction routines" -- only neighbours
 *            carrying the particle's own owner label;
 * which = 2: step f alone, "local particle interaction with the MGPU boundary
 *            particles" -- only neighbours carrying another label.
 * The sums are linear in the pair contributions, so pass 1 + pass 2 = pass 0 up to rounding. */
static void orc_interact_impl(int64_t n, const float *posm, const float *velr, const float *sig,
                  const uint32_t *sorted_hash, const int32_t *dims, const uint32_t *cell_start,
                  const uint32_t *cell_end, float h_f32, float K_f32, float G_f32,
                  int64_t n_idx, const int64_t *idx, const int32_t *owner, int which,
                  const float *hp,
                  double *drho, double *L, double *acc, double *dsig, int64_t *pair_count)
{
    const double h = (double)h_f32, K = (double)K_f32, G = (double)G_f32;
    const double support2 = (2.0 * h) * (2.0 * h);
    const int64_t nx = dims[0], ny = dims[1], nz = dims[2];
    const int64_t m_out = idx ? n_idx : n;
    int64_t pairs = 0;

    for (int64_t out = 0; out < m_out; ++out) {
        const int64_t i = idx ? idx[out] : out;
        const int64_t hsh = sorted_hash[i];
        const int64_t cx = hsh % nx, cy = (hsh / nx) % ny, cz = hsh / (nx * ny);
        const double xi[3] = { posm[4 * i + 0], posm[4 * i + 1], posm[4 * i + 2] };
        const double vi[3] = { velr[4 * i + 0], velr[4 * i + 1], velr[4 * i + 2] };
        const double rhoi = velr[4 * i + 3];
        double si[3][3];
        orc_sym_load(sig, n, i, si);

        /* ---- loop 1: density rate and velocity gradient ---- */
        double dr = 0.0, Li[3][3] = { { 0 } };
        for (int64_t dz = -1; dz <= 1; ++dz)
            for (int64_t dy = -1; dy <= 1; ++dy)
                for (int64_t dx = -1; dx <= 1; ++dx) {
                    const int64_t x = cx + dx, y = cy + dy, z = cz + dz;
                    if (x < 0 || x >= nx || y < 0 || y >= ny || z < 0 || z >= nz) continue;
                    const int64_t c = x + nx * (y + ny * z);
                    for (int64_t j = cell_start[c]; j < (int64_t)cell_end[c]; ++j) {
                        if (j == i) continue; /* S15 */
                        if (which == 1 && owner[j] != owner[i]) continue; /* step e */
                        if (which == 2 && owner[j] == owner[i]) continue; /* step f */
                        const double xij[3] = { xi[0] - posm[4 * j + 0], xi[1] - posm[4 * j + 1],
                                                xi[2] - posm[4 * j + 2] };
                        const double r2 = xij[0] * xij[0] + xij[1] * xij[1] + xij[2] * xij[2];
                        /* O7h (reading H2): per-particle smoothing lengths enter through the
                         * symmetrised pair length h_ij = (h_i + h_j) / 2, support 2 h_ij */
                        const double hij = hp ? 0.5 * ((double)hp[i] + (double)hp[j]) : h;
                        const double sup2 = hp ? (2.0 * hij) * (2.0 * hij) : support2;
                        if (!(r2 < sup2)) continue;
                        ++pairs;
                        const double F = orc_kernel_F(sqrt(r2), hij);
                        const double mj = posm[4 * j + 3], rhoj = velr[4 * j + 3];
                        const double gW[3] = { F * xij[0], F * xij[1], F * xij[2] };
                        const double vij[3] = { vi[0] - velr[4 * j + 0], vi[1] - velr[4 * j + 1],
                                                vi[2] - velr[4 * j + 2] };
                        dr += mj * (vij[0] * gW[0] + vij[1] * gW[1] + vij[2] * gW[2]);
                        for (int a = 0; a < 3; ++a)
                            for (int b = 0; b < 3; ++b)
                                Li[a][b] += (mj / rhoj) * (-vij[a]) * gW[b];
                    }
                }

        /* ---- loop 2: momentum (stress divergence) ---- */
        double ai[3] = { 0, 0, 0 };
        for (int64_t dz = -1; dz <= 1; ++dz)
            for (int64_t dy = -1; dy <= 1; ++dy)
                for (int64_t dx = -1; dx <= 1; ++dx) {
                    const int64_t x = cx + dx, y = cy + dy, z = cz + dz;
                    if (x < 0 || x >= nx || y < 0 || y >= ny || z < 0 || z >= nz) continue;
                    const int64_t c = x + nx * (y + ny * z);
                    for (int64_t j = cell_start[c]; j < (int64_t)cell_end[c]; ++j) {
                        if (j == i) continue;
                        if (which == 1 && owner[j] != owner[i]) continue;
                        if (which == 2 && owner[j] == owner[i]) continue;
                        const double xij[3] = { xi[0] - posm[4 * j + 0], xi[1] - posm[4 * j + 1],
                                                xi[2] - posm[4 * j + 2] };
                        const double r2 = xij[0] * xij[0] + xij[1] * xij[1] + xij[2] * xij[2];
                        const double hij = hp ? 0.5 * ((double)hp[i] + (double)hp[j]) : h;
                        const double sup2 = hp ? (2.0 * hij) * (2.0 * hij) : support2;
                        if (!(r2 < sup2)) continue;
                        const double F = orc_kernel_F(sqrt(r2), hij);
                        const double mj = posm[4 * j + 3], rhoj = velr[4 * j + 3];
                        double sj[3][3];
                        orc_sym_load(sig, n, j, sj);
                        for (int a = 0; a < 3; ++a) {
                            double t = 0.0;
                            for (int b = 0; b < 3; ++b)
                                t += (si[a][b] / (rhoi * rhoi) + sj[a][b] / (rhoj * rhoj)) *
                                     (F * xij[b]);
                            ai[a] += mj * t;
                        }
                    }
                }

        /* ---- O8: Hooke's law in rate form with the Jaumann rate ---- */
        double D[3][3], Om[3][3];
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) {
                D[a][b] = 0.5 * (Li[a][b] + Li[b][a]);
                Om[a][b] = 0.5 * (Li[a][b] - Li[b][a]);
            }
        const double trD = D[0][0] + D[1][1] + D[2][2];
        double sd[3][3];
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) {
                double v = 2.0 * G * (D[a][b] - (a == b ? trD / 3.0 : 0.0)) +
                           (a == b ? K * trD : 0.0);
                for (int c = 0; c < 3; ++c) v += Om[a][c] * si[c][b] - si[a][c] * Om[c][b];
                sd[a][b] = v;
            }

        drho[out] = dr;
        for (int a = 0; a < 3; ++a) {
            acc[3 * out + a] = ai[a];
            for (int b = 0; b < 3; ++b) L[9 * out + 3 * a + b] = Li[a][b];
        }
        dsig[6 * out + 0] = sd[0][0]; dsig[6 * out + 1] = sd[1][1]; dsig[6 * out + 2] = sd[2][2];
        dsig[6 * out + 3] = sd[0][1]; dsig[6 * out + 4] = sd[0][2]; dsig[6 * out + 5] = sd[1][2];
    }
    if (pair_count) *pair_count = pairs;
}

void orc_interact(int64_t n, const float *posm, const float *velr, const float *sig,
                  const uint32_t *sorted_hash, const int32_t *dims, const uint32_t *cell_start,
                  const uint32_t *cell_end, float h_f32, float K_f32, float G_f32,
                  int64_t n_idx, const int64_t *idx,
                  double *drho, double *L, double *acc, double *dsig, int64_t *pair_count)
{
    orc_interact_impl(n, posm, velr, sig, sorted_hash, dims, cell_start, cell_end, h_f32, K_f32, G_f32,
                      n_idx, idx, NULL, 0, NULL, drho, L, acc, dsig, pair_count);
}

/* NEXT-3: steps e (which = 1) and f (which = 2) as separate passes; owner is in sorted order.
 * idx != NULL: only the n_idx sorted positions idx[] are computed (sampled parity at full size). */
void orc_interact_split(int64_t n, const float *posm, const float *velr, const float *sig,
                        const uint32_t *sorted_hash, const int32_t *dims, const uint32_t *cell_start,
                        const uint32_t *cell_end, float h_f32, float K_f32, float G_f32,
                        const int32_t *owner, int which, int64_t n_idx, const int64_t *idx,
                        double *drho, double *L, double *acc, double *dsig, int64_t *pair_count)
{
    orc_interact_impl(n, posm, velr, sig, sorted_hash, dims, cell_start, cell_end, h_f32, K_f32, G_f32,
                      n_idx, idx, owner, which, NULL, drho, L, acc, dsig, pair_count);
}

/* NEXT-4, second half ("cubic buckets of size 2h with h the maximum
 * smoothing length of the particles"; "multiple particle types with different
 * smoothing lengths"): O7 with a smoothing length per particle.  Readings:
 *   H1  the bucket grid is built on h_max (the h of orc_hash / cell tables), every hp[i] <= h_max;
 *   H2  a pair uses the symmetrised length h_ij = (h_i + h_j) / 2 in fp64: W(r, h_ij), neighbours
 *       are the stencil particles with r < 2 h_ij (inside the 27 buckets because h_ij <= h_max);
 *       the pair force stays antisymmetric, so momentum is still conserved exactly;
 *   H3  everything else (sums, O8) as in orc_interact; uniform hp == h reproduces it bit for bit.
 * hp [n] in sorted order; owner / which as in orc_interact_split (owner may be NULL with which = 0). */
void orc_interact_varh(int64_t n, const float *posm, const float *velr, const float *sig,
                       const float *hp, const uint32_t *sorted_hash, const int32_t *dims,
                       const uint32_t *cell_start, const uint32_t *cell_end, float hmax_f32, float K_f32,
                       float G_f32, const int32_t *owner, int which, int64_t n_idx, const int64_t *idx,
                       double *drho, double *L, double *acc, double *dsig, int64_t *pair_count)
{
    orc_interact_impl(n, posm, velr, sig, sorted_hash, dims, cell_start, cell_end, hmax_f32, K_f32, G_f32,
                      n_idx, idx, owner, which, hp, drho, L, acc, dsig, pair_count);
}

/* ------------------------------------------------------------------------------------------
 * O9  Explicit integration (PAPER.md:26 step g: "Each GPU can integrate its equations").
 * Reading S18: symplectic Euler.  rho+ = rho + dt Drho; v+ = v + dt a; sigma+ = sigma + dt dsig;
 * x+ = x + dt v+.  Mass unchanged.  Inputs fp32 state + fp64 rates (layouts as orc_interact's
 * outputs); outputs fp64: posm_out [n][4], velr_out [n][4], sig_out [6][n].
 * ---------------------------------------------------------------------------------------- */
void orc_integrate(int64_t n, double dt, const float *posm, const float *velr, const float *sig,
                   const double *drho, const double *acc, const double *dsig, double *posm_out,
                   double *velr_out, double *sig_out)
{
    for (int64_t i = 0; i < n; ++i) {
        double vp[3];
        for (int a = 0; a < 3; ++a) {
            vp[a] = (double)velr[4 * i + a] + dt * acc[3 * i + a];
            velr_out[4 * i + a] = vp[a];
            posm_out[4 * i + a] = (double)posm[4 * i + a] + dt * vp[a];
        }
        posm_out[4 * i + 3] = (double)posm[4 * i + 3];
        velr_out[4 * i + 3] = (double)velr[4 * i + 3] + dt * drho[i];
        for (int c = 0; c < 6; ++c)
            sig_out[(int64_t)c * n + i] = (double)sig[(int64_t)c * n + i] + dt * dsig[6 * i + c];
    }
}

/* ------------------------------------------------------------------------------------------
 * O10  Communication-load balancing, single particle type (
 * PAPER.md:36, section III.A), followed step by step, one sweep over all owner pairs:
 *   "Every GPU computes its own particle cloud centre of gravity (Cg).  A balancing hash number
 *    is defined based on the projection of the particle position on the line from one GPU Cg
 *    to the other.  If the projection is located on the own GPU side of the middle of the
 *    segment of the two Cgs, the particle is disregarded for swapping (hash number 0).  If the
 *    projection is located beyond the other Cg, the particle is given the maximum swapping hash
 *    number (typically 1000).  In between the balancing hash number is proportional to the
 *    distance between the middle of the Cgs and the other Cg up to the maximum swapping hash
 *    number.  If both GPUs have particles with positive hash numbers, some particle swapping
 *    occurs.  The number of particles to be swapped is determined by the minimum number of
 *    particles with a positive hash number on each GPU.  The particle data can be sorted by the
 *    balancing hash number and the corresponding particles can be swapped between the two GPUs.
 *    The algorithm is then repeated for each GPU pair."
 * Readings: B1 pairs (A, B), A < B, in lexicographic order, labels
 * updated after every pair, Cgs recomputed before every pair; B2 Cg = unweighted mean position,
 * summed EXACTLY in 2^-16 fixed point (int64), so that the result does not depend on the order of
 * the reduction; B3 s = ((x - CgA) . d) / (d . d), d = CgB - CgA, fp64, sums left to right, no
 * contraction; B4 hash = 0 if !(s > 1/2), hmax if s >= 1, else ceil(hmax (2 s - 1)) clipped to
 * [1, hmax]; B5 a pair with an empty owner or coincident Cgs is skipped; B6 n = min(nA, nB), the
 * n particles of each side that come first in the order (hash descending, id ascending) swap
 * labels; B7 hmax = 1000 by default.
 * owner [n] is updated in place; bal_hash (may be NULL) receives, for the LAST pair processed
 * that involved the particle, its balancing hash (diagnostic).  Returns the number of swapped
 * particle pairs.
 * ---------------------------------------------------------------------------------------- */
typedef struct { int32_t hash; uint32_t id; } orc_bal;

static int orc_bal_cmp(const void *a, const void *b)
{
    const orc_bal *x = (const orc_bal *)a, *y = (const orc_bal *)b;
    if (x->hash != y->hash) return x->hash > y->hash ? -1 : 1; /* hash descending */
    if (x->id != y->id) return x->id < y->id ? -1 : 1;         /* id ascending (B6) */
    return 0;
}

static int32_t orc_balance_hash(const float *posm, int64_t i, const double cg_own[3],
                                const double cg_other[3], int32_t hmax)
{
    const double d0 = cg_other[0] - cg_own[0], d1 = cg_other[1] - cg_own[1], d2 = cg_other[2] - cg_own[2];
    const double dd = d0 * d0 + d1 * d1 + d2 * d2;
    const double e0 = (double)posm[4 * i + 0] - cg_own[0], e1 = (double)posm[4 * i + 1] - cg_own[1],
                 e2 = (double)posm[4 * i + 2] - cg_own[2];
    const double s = (e0 * d0 + e1 * d1 + e2 * d2) / dd;
    if (!(s > 0.5)) return 0;
    if (s >= 1.0) return hmax;
    double hv = ceil((double)hmax * (2.0 * s - 1.0));
    if (hv < 1.0) hv = 1.0;
    if (hv > (double)hmax) hv = (double)hmax;
    return (int32_t)hv;
}

int64_t orc_balance(int64_t n, const float *posm, int32_t *owner, int32_t n_owners, int32_t hmax,
                    int32_t *bal_hash)
{
    orc_bal *la = (orc_bal *)malloc((size_t)(n > 0 ? n : 1) * sizeof(orc_bal));
    orc_bal *lb = (orc_bal *)malloc((size_t)(n > 0 ? n : 1) * sizeof(orc_bal));
    if (!la || !lb) { free(la); free(lb); return -1; }
    int64_t swapped = 0;
    for (int32_t A = 0; A < n_owners; ++A)
        for (int32_t B = A + 1; B < n_owners; ++B) {
            int64_t sum[2][3] = { { 0, 0, 0 }, { 0, 0, 0 } }, cnt[2] = { 0, 0 };
            for (int64_t i = 0; i < n; ++i) {
                const int side = owner[i] == A ? 0 : (owner[i] == B ? 1 : -1);
                if (side < 0) continue;
                for (int a = 0; a < 3; ++a) sum[side][a] += (int64_t)llrint((double)posm[4 * i + a] * 65536.0);
                cnt[side] += 1;
            }
            if (cnt[0] == 0 || cnt[1] == 0) continue; /* B5 */
            double cg[2][3];
            for (int side = 0; side < 2; ++side)
                for (int a = 0; a < 3; ++a)
                    cg[side][a] = ((double)sum[side][a] / (double)cnt[side]) * (1.0 / 65536.0);
            if (cg[0][0] == cg[1][0] && cg[0][1] == cg[1][1] && cg[0][2] == cg[1][2]) continue; /* B5 */
            int64_t na = 0, nb = 0;
            for (int64_t i = 0; i < n; ++i) {
                if (owner[i] == A) {
                    const int32_t hv = orc_balance_hash(posm, i, cg[0], cg[1], hmax);
                    if (bal_hash) bal_hash[i] = hv;
                    if (hv > 0) { la[na].hash = hv; la[na].id = (uint32_t)i; ++na; }
                } else if (owner[i] == B) {
                    const int32_t hv = orc_balance_hash(posm, i, cg[1], cg[0], hmax);
                    if (bal_hash) bal_hash[i] = hv;
                    if (hv > 0) { lb[nb].hash = hv; lb[nb].id = (uint32_t)i; ++nb; }
                }
            }
            const int64_t m = na < nb ? na : nb;
            if (m == 0) continue;
            qsort(la, (size_t)na, sizeof(orc_bal), orc_bal_cmp);
            qsort(lb, (size_t)nb, sizeof(orc_bal), orc_bal_cmp);
            for (int64_t k = 0; k < m; ++k) {
                owner[la[k].id] = B;
                owner[lb[k].id] = A;
            }
            swapped += m;
        }
    free(la);
    free(lb);
    return swapped;
}

/* ------------------------------------------------------------------------------------------
 * O11  Balancing with multiple particle types (section
 * III.B): "all particle types shall be balanced over each GPU ...  The swapping algorithm of
 * section III.A can then be applied for each particle type.  However, this may lead to an
 * independent decomposition from particle type to particle type.  To overcome this to a certain
 * extent, a biased Cg' can be used ... shift the Cg used for balancing from the actual Cg of the
 * particles of the desired type towards the global Cg of the particles:
 *     Cg'_typeA = alpha Cg_alltypes + (1 - alpha) Cg_typeA   with alpha = 0.1".
 * Readings: B8 types are processed in ascending order, each with the full pair sweep of O10
 * restricted to the particles of that type (only they get a hash, only they swap); B9 Cg_alltypes
 * of an owner is the unweighted mean over ALL its particles (current labels), Cg_type over its
 * particles of the type, both from exact fixed-point sums; Cg' = alpha * Cg_all + (1 - alpha) *
 * Cg_type evaluated in fp64 as written (two products, one sum, no contraction); B10 a pair is
 * skipped when either owner holds no particle of the type or the two Cg' coincide.
 * ---------------------------------------------------------------------------------------- */
int64_t orc_balance_types(int64_t n, const float *posm, int32_t *owner, const int32_t *ptype,
                          int32_t n_owners, int32_t n_types, int32_t hmax, double alpha, int32_t *bal_hash)
{
    orc_bal *la = (orc_bal *)malloc((size_t)(n > 0 ? n : 1) * sizeof(orc_bal));
    orc_bal *lb = (orc_bal *)malloc((size_t)(n > 0 ? n : 1) * sizeof(orc_bal));
    if (!la || !lb) { free(la); free(lb); return -1; }
    int64_t swapped = 0;
    for (int32_t T = 0; T < n_types; ++T)
        for (int32_t A = 0; A < n_owners; ++A)
            for (int32_t B = A + 1; B < n_owners; ++B) {
                int64_t st[2][3] = { { 0 } }, sa[2][3] = { { 0 } }, ct[2] = { 0, 0 }, ca[2] = { 0, 0 };
                for (int64_t i = 0; i < n; ++i) {
                    const int side = owner[i] == A ? 0 : (owner[i] == B ? 1 : -1);
                    if (side < 0) continue;
                    for (int a = 0; a < 3; ++a) {
                        const int64_t f = (int64_t)llrint((double)posm[4 * i + a] * 65536.0);
                        sa[side][a] += f;
                        if (ptype[i] == T) st[side][a] += f;
                    }
                    ca[side] += 1;
                    if (ptype[i] == T) ct[side] += 1;
                }
                if (ct[0] == 0 || ct[1] == 0) continue; /* B10 */
                double cg[2][3];
                for (int side = 0; side < 2; ++side)
                    for (int a = 0; a < 3; ++a) {
                        const double call = ((double)sa[side][a] / (double)ca[side]) * (1.0 / 65536.0);
                        const double ctyp = ((double)st[side][a] / (double)ct[side]) * (1.0 / 65536.0);
                        cg[side][a] = alpha * call + (1.0 - alpha) * ctyp;
                    }
                if (cg[0][0] == cg[1][0] && cg[0][1] == cg[1][1] && cg[0][2] == cg[1][2]) continue;
                int64_t na = 0, nb = 0;
                for (int64_t i = 0; i < n; ++i) {
                    if (ptype[i] != T) continue;
                    if (owner[i] == A) {
                        const int32_t hv = orc_balance_hash(posm, i, cg[0], cg[1], hmax);
                        if (bal_hash) bal_hash[i] = hv;
                        if (hv > 0) { la[na].hash = hv; la[na].id = (uint32_t)i; ++na; }
                    } else if (owner[i] == B) {
                        const int32_t hv = orc_balance_hash(posm, i, cg[1], cg[0], hmax);
                        if (bal_hash) bal_hash[i] = hv;
                        if (hv > 0) { lb[nb].hash = hv; lb[nb].id = (uint32_t)i; ++nb; }
                    }
                }
                const int64_t m = na < nb ? na : nb;
                if (m == 0) continue;
                qsort(la, (size_t)na, sizeof(orc_bal), orc_bal_cmp);
                qsort(lb, (size_t)nb, sizeof(orc_bal), orc_bal_cmp);
                for (int64_t k = 0; k < m; ++k) {
                    owner[la[k].id] = B;
                    owner[lb[k].id] = A;
                }
                swapped += m;
            }
    free(la);
    free(lb);
    return swapped;
}

