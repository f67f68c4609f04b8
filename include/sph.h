/*
 * sph.h -- C-ABI boundary of the B200-native SPH hot path (libsph_b200.so).
 *
 * One iteration of the particle-decomposition SPH scheme of Unfer, Colle & Limido
 * (arxiv 2310.03596; cited below as PAPER.md:<line> = /root/reference/PAPER.md), restricted to
 * one GPU: owner labels stand in for the paper's GPUs, the "MGPU boundary
 * particle" set is the product of stage 3, the multi-GPU broadcasts (steps b, d)
 * are out of scope.  Readings of everything the paper leaves open (S1..S28) are in DESIGN.md
 * section 3.
 *
 * Conventions
 *  - "dev"  = CUDA device pointer, owned by the CALLER (e.g. a torch tensor); the library never
 *    allocates, frees or retains it beyond the call's enqueued work.
 *    "host" = ordinary host pointer (only sph_params, sph_state structs themselves, and the
 *    buffers of sph_step_host).
 *  - sph_ctx owns only scratch (radix-sort ping-pong buffers, histograms, tile status words,
 *    per-bucket owner masks, scan space, the sorted copy of the state used by sph_step).  It is
 *    sized for max_n particles and the grid of the sph_params given at creation.
 *  - Every entry point except sph_create / sph_destroy / sph_step_host / sph_balance[_types] only ENQUEUES work on the
 *    ctx's stream and returns; outputs are valid once the caller synchronises that stream.
 *    No allocation and no host synchronisation happens on the hot path.  One ctx per host thread.
 *  - Return value: 0 = SPH_OK, negative = error (below).  No exception crosses this boundary.
 *  - Per-particle arrays: posm [n][4] = x, y, z, m;  velr [n][4] = vx, vy, vz, rho;
 *    sig[c] [n], c = xx, yy, zz, xy, xz, yz (SoA);  owner [n] in [0, n_owners).
 *    The labels are the caller's contract and are NOT validated on the device (a check would
 *    cost a pass and a host synchronisation): the kernels use label & 31 (bucket masks) and
 *    label & 255 (partition passes), so an out-of-range label gives wrong boundary sets, never a fault.
 *    All real data fp32, all hashes / indices uint32.  posm / velr / acc must be 16-byte aligned,
 *    everything else 4-byte aligned.
 *  - "sorted position k": index in the (hash, id) order produced by sph_sort; perm[k] is the
 *    persistent particle id (= index in the caller's id-ordered arrays) of the k-th particle.
 */
#ifndef SPH_B200_H
#define SPH_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SPH_OK        0
#define SPH_EINVAL   -1   /* null pointer, n < 0, n > max_n, bad params                         */
#define SPH_ECUDA    -2   /* a CUDA runtime call or launch failed (see sph_last_cuda_error)     */
#define SPH_ENOMEM   -3   /* scratch allocation failed                                           */
#define SPH_ELIMIT   -4   /* size beyond a fixed capacity stated at the entry point's declaration */

#define SPH_GARBAGE_HASH 0xFFFFFFFFu  /* PAPER.md:17 "some garbage collector hash" (reading S8) */
#define SPH_MAX_OWNERS   32           /* paper's envelope is <= 16 GPUs           */
#define SPH_NOALLOC_MAX_CELLS (1 << 22) /* buckets sph_comm_hash_noalloc's built-in scratch holds  */

/* sph_params.flags */
#define SPH_FLAG_INTERACT_DIRECT 1u   /* force the simple global-memory interaction kernel      */

typedef struct sph_ctx sph_ctx;      /* opaque */

typedef struct {
    float    origin[3];  /* lower corner of the bucket grid (reading S3)                        */
    int32_t  dims[3];    /* nx, ny, nz buckets; each 1 .. 2^24, nx*ny*nz < 2^32 - 1              */
    float    h;          /* smoothing length (the MAXIMUM one with sph_*_varh); bucket edge = 2h   */
    float    K, G;       /* bulk / shear modulus of the linear-elastic law (BASELINE.json cfgs)  */
    int32_t  n_owners;   /* 1 .. SPH_MAX_OWNERS                                                  */
    uint32_t flags;      /* SPH_FLAG_* or 0                                                      */
} sph_params;

typedef struct {          /* SoA particle state; every pointer dev, length n                     */
    float   *posm;        /* [n][4] x, y, z, m                                                   */
    float   *velr;        /* [n][4] vx, vy, vz, rho                                              */
    float   *sig[6];      /* xx, yy, zz, xy, xz, yz                                              */
    int32_t *owner;       /* [n]                                                                 */
} sph_state;

/* Create a context: validates params, allocates scratch for max_n particles on the current
 * device.  cuda_stream is a cudaStream_t (borrowed; NULL = legacy default stream).
 * Errors: SPH_EINVAL (null, max_n < 0 or >= 2^30, a dim <= 0 or > 2^24, product >= 2^32-1, h <= 0 or not
 * finite, n_owners outside 1..32), SPH_ENOMEM, SPH_ECUDA. */
int sph_create(sph_ctx **ctx, const sph_params *params, int64_t max_n, void *cuda_stream);
int sph_destroy(sph_ctx *ctx);

/* Stage 1 -- bucket hash ("Each particle is given a hash number corresponding to the
 * bucket in which it is located"; step a).  For each axis a, in fp32 and in this
 * order (reading S2): t = x_a - origin_a; u = t * inv (inv = 1.0f / (2.0f * h), rounded once);
 * f = floorf(u) clamped to [0, dims_a - 1] (out-of-grid particles are clamped, never an error);
 * hash = cx + nx * (cy + ny * cz) (reading S1).  Non-finite positions give an unspecified hash.
 * posm: dev [n][4] in id order.  hash: dev [n] out. */
int sph_hash(sph_ctx *ctx, int64_t n, const float *posm, uint32_t *hash);

/* Stage 2a -- stable LSD radix sort (hand-written onesweep) on the key (hash, id)
 * ("sorted with respect to this hash number by the radix sort algorithm"; reading
 * S5).  hash: dev [n] in id order (index = particle id), every value < nx*ny*nz.
 * sorted_hash, perm: dev [n] out; perm[k] = id of the k-th particle, sorted_hash[k] =
 * hash[perm[k]].  Only the ceil(log2(nx*ny*nz)) live key bits are sorted. */
int sph_sort(sph_ctx *ctx, int64_t n, const uint32_t *hash, uint32_t *sorted_hash, uint32_t *perm);

/* Stage 2b -- gather the state into sorted order: out.X[k] = in.X[perm[k]] for every field
 * ("The particles are then sorted").  in and out must not alias. */
int sph_reorder(sph_ctx *ctx, int64_t n, const uint32_t *perm, const sph_state *in,
                const sph_state *out);

/* Stage 2c -- cell start/end tables (BASELINE.json north_star; reading S7):
 * cell_start[c] = #{k : sorted_hash[k] < c}, cell_end[c] = #{k : sorted_hash[k] <= c};
 * both dev [nx*ny*nz] out.  Empty bucket => start == end. */
int sph_cell_ranges(sph_ctx *ctx, int64_t n, const uint32_t *sorted_hash, uint32_t *cell_start,
                    uint32_t *cell_end);

/* Stage 3 -- communication hash and MGPU boundary particles (step c PAPER.md:22).
 * comm_hash[k] = sorted_hash[k] if a particle with a different owner lies in the 27-bucket
 * stencil of k's bucket (out-of-grid buckets skipped, reading S9; bucket-level test, S10), else
 * SPH_GARBAGE_HASH.  boundary_ids = ids (perm values) of the particles with comm_hash !=
 * garbage in ascending (comm_hash, id) order, i.e. the head of the paper's sort on that key
 * (I6: identical to a stable compaction of the sorted array); *boundary_count = M;
 * owner_counts[g] = how many of them carry owner g.
 * In: sorted_hash, sorted_owner, perm dev [n]; cell_start, cell_end dev [cells].
 * Out: comm_hash dev [n]; boundary_ids dev, capacity n; boundary_count dev scalar;
 * owner_counts dev [n_owners]. */
int sph_comm_hash(sph_ctx *ctx, int64_t n, const uint32_t *sorted_hash, const int32_t *sorted_owner,
                  const uint32_t *perm, const uint32_t *cell_start, const uint32_t *cell_end,
                  uint32_t *comm_hash, uint32_t *boundary_ids, uint32_t *boundary_count,
                  uint32_t *owner_counts);

/* Stage 4a -- SPH interaction loops over the 27-bucket stencil (steps e/f
 * PAPER.md:24-25, "several interaction loops" PAPER.md:28; equations: DESIGN.md O6-O8).
 * Neighbours of i: every j != i in the stencil of i's bucket with r_ij^2 < (2h)^2.
 *   drho_i = sum_j m_j (v_i - v_j) . gradW_ij            (density rate)
 *   L_i    = sum_j (m_j / rho_j) (v_j - v_i) (x) gradW_ij (velocity gradient)
 *   acc_i  = sum_j m_j (sigma_i / rho_i^2 + sigma_j / rho_j^2) . gradW_ij
 *   dsig_i = K tr(D) I + 2G dev(D) + Om sigma - sigma Om,  D, Om = sym / skew part of L
 * with the Wendland C2 kernel, gradW_ij = F(r) x_ij.  All rates use the state at the start of
 * the step.  `sorted` is the state in sorted order (sorted_hash gives each particle's bucket).
 * Out (dev, indexed by sorted position): drho [n], acc [n][4] (w = 0), dsig[c] [n].
 * pair_count: dev scalar or NULL; receives the number of ordered accepted pairs (reading S25). */
int sph_interact(sph_ctx *ctx, int64_t n, const sph_state *sorted, const uint32_t *sorted_hash,
                 const uint32_t *cell_start, const uint32_t *cell_end, float *drho, float *acc,
                 float *const dsig[6], unsigned long long *pair_count);

/* NEXT-3 -- steps e and f of the paper as SEPARATE passes ("local
 * particle interaction routines", overlapped with the broadcast; "local particle
 * interaction with the MGPU boundary particles"): which = 1 takes only the neighbours that carry
 * the particle's own owner label (step e), which = 2 only those with another label (step f).
 * Same arguments and outputs as sph_interact; the rates are linear in the pair contributions, so
 * pass 1 + pass 2 equals sph_interact up to rounding, and the pair counts add up exactly
 * (pair_count accumulates; zero it first).  sorted->owner is read. */
int sph_interact_split(sph_ctx *ctx, int64_t n, const sph_state *sorted, const uint32_t *sorted_hash,
                       const uint32_t *cell_start, const uint32_t *cell_end, int32_t which,
                       float *drho, float *acc, float *const dsig[6], unsigned long long *pair_count);

/* Stage 4b -- explicit integration, symplectic Euler (step g; reading S18):
 * rho += dt drho; v += dt acc; sigma += dt dsig; x += dt v(new).  m and owner are copied.
 * Elementwise: in, rates and out use the same index order; out may alias in. */
int sph_integrate(sph_ctx *ctx, int64_t n, float dt, const sph_state *in, const float *drho,
                  const float *acc, const float *const dsig[6], const sph_state *out);

/* The whole iteration on one stream, no host synchronisation (PAPER.md:19-26 with steps b, d
 * removed): hash -> sort -> reorder -> cell ranges -> comm hash + compaction -> interact ->
 * integrate.  `state` is in ID ORDER on entry and on exit (so the (hash, id) tie-break stays
 * exact when every step re-sorts, reading S5).  Every output pointer below is optional (NULL =
 * keep it in ctx scratch); when given it receives exactly what the stage call of the same name
 * would produce (rates indexed by sorted position).  Two stage boundaries are fused inside this
 * call: the reorder pass also writes the interaction kernel's packed records, and the
 * interaction epilogue integrates and scatters to id order.  The rates drho / acc / dsig are
 * intermediates of that epilogue: if all three are NULL they are not stored anywhere; if any is
 * given all of them are computed as usual (missing ones go to ctx scratch).  The integrated
 * state agrees with sph_integrate of the same rates to 3 ulp (sigma and rho re-enter the
 * epilogue as sigma / rho^2 * rho^2 and m / (m / rho)). */
int sph_step(sph_ctx *ctx, int64_t n, float dt, const sph_state *state,
             uint32_t *hash, uint32_t *sorted_hash, uint32_t *perm,
             uint32_t *cell_start, uint32_t *cell_end, uint32_t *comm_hash,
             uint32_t *boundary_ids, uint32_t *boundary_count, uint32_t *owner_counts,
             float *drho, float *acc, float *const dsig[6], unsigned long long *pair_count);

/* NEXT-1 -- per-owner send buffers: the product of step d ("the data
 * that shall be broadcasted to the other GPUs can be isolated"; "Each GPU broadcasts
 * its MGPU boundary particle data").  In the paper every GPU isolates its OWN boundary particles;
 * with owner labels that is the boundary list cut into one segment per owner:
 *   segment g = the entries of boundary_ids (already in (hash, id) order) whose owner is g, in
 *   list order;  owner_offsets[g] = size of the segments before g, owner_offsets[n_owners] = m;
 *   packed_ids = the segments back to back;  packed->X[j] = state->X[packed_ids[j]] for posm,
 *   velr, sig[0..5], owner -- contiguous per owner, ready to be handed to a collective.
 * m = number of boundary particles, a HOST value (read boundary_count after synchronising the
 * stream: the exchange needs the size on the host anyway); 0 <= m <= n.
 * In: state dev, id order, length n; boundary_ids dev [m].
 * Out: owner_offsets dev [n_owners + 1]; packed_ids dev [m]; packed dev arrays of capacity m
 * (packed->sig[c] are six separate planes).  Not part of sph_step. */
int sph_pack_boundary(sph_ctx *ctx, int64_t n, int64_t m, const sph_state *state,
                      const uint32_t *boundary_ids, uint32_t *owner_offsets, uint32_t *packed_ids,
                      const sph_state *packed);

/* NEXT-1, second half -- per-DESTINATION send lists.  Step d of the paper ships every
 * MGPU boundary particle to every other GPU ("Each GPU broadcasts its MGPU boundary
 * particle data to the other GPUs"); GPU g, however, only uses a foreign particle that lies in the
 * own or a surrounding bucket of one of its particles (step f searches those 27 buckets,
 * PAPER.md:25).  Reading D1: particle k is on the list of destination g iff
 * owner_k != g and a particle owned by g lies in the 27-bucket stencil of k's bucket (bucket-level
 * test, out-of-grid buckets skipped, as for the communication hash).  The union of the lists is the
 * boundary set; their total length is at most M (n_owners - 1), the size of the broadcast, and far
 * less for compact decompositions (three wide slabs: half).
 * In: sorted_hash, sorted_owner, perm dev [n] (sorted order, as for sph_comm_hash; no cell tables).
 * Out: dest_offsets dev [n_owners + 1]: list g = dest_ids[dest_offsets[g] .. dest_offsets[g + 1]),
 * dest_offsets[n_owners] = total number of entries; dest_ids dev, capacity `cap` entries, or NULL to
 * get the offsets only (size the buffer, then call again): particle ids (perm values), each list
 * in (hash, id) order.  Entries beyond cap are not written (compare the total with cap after
 * synchronising).  Limit: n (n_owners - 1) must be below 2^30 (SPH_ELIMIT otherwise: the scan
 * carries 30-bit prefixes).  Enqueues only; not part of sph_step. */
int sph_pack_destinations(sph_ctx *ctx, int64_t n, const uint32_t *sorted_hash, const int32_t *sorted_owner,
                          const uint32_t *perm, uint32_t *dest_offsets, uint32_t *dest_ids, int64_t cap);

/* NEXT-2 -- one sweep of the communication-load balancing heuristic on the owner
 * labels, single particle type (section III.A; the paper runs it every 20 integration
 * loops, PAPER.md:32 -- the cadence is the caller's).  For every owner pair (A, B), A < B, in
 * lexicographic order (labels and centres of gravity are updated after every pair): Cg = unweighted
 * mean position of an owner's particles; balancing hash of a particle = 0 if its projection s on
 * the line Cg_own -> Cg_other (s = 0 at Cg_own, 1 at Cg_other) is not beyond the middle (s <= 1/2),
 * hmax if s >= 1, else ceil(hmax (2 s - 1)); n = min over the two owners of the number of particles
 * with a positive hash; the n first particles of each side in the order (hash descending, id
 * ascending) swap labels.  Every owner keeps its particle count.  Exact arithmetic contract (so
 * that the labels have one correct value): Cg from 2^-16 fixed-point int64 coordinate sums, s in
 * fp64 without contraction.
 * Unlike the stage calls this one SYNCHRONISES the ctx's stream once (the ids are first grouped by
 * owner, and the sizes of the groups, read back once per sweep, size the launches of the pairs).
 * In: posm dev [n][4] in id order; hmax in 1 .. 1023 (the paper's typical value: 1000).
 * In/out: owner dev [n].  Out (optional, may be NULL): bal_hash dev [n] = the hash each particle
 * got in the last pair that involved it (0 if none); swapped dev scalar = particle pairs swapped. */
int sph_balance(sph_ctx *ctx, int64_t n, const float *posm, int32_t *owner, int32_t hmax,
                int32_t *bal_hash, unsigned long long *swapped);

/* NEXT-4 -- the balancing sweep for multiple particle types (PAPER.md:54-57,
 * section III.B): the pair sweep of sph_balance is applied to each particle type in ascending
 * order (only particles of the type get a hash and swap, so every (owner, type) count is kept),
 * with the biased centre of gravity of PAPER.md:56
 *     Cg'_type = alpha Cg_alltypes + (1 - alpha) Cg_type        (the paper: alpha = 0.1)
 * where Cg_alltypes is the mean over ALL particles of the owner and Cg_type over its particles of
 * the type (exact fixed-point sums; the blend in fp64 as written, no contraction).
 * ptype dev [n], values in [0, n_types), n_types <= 8; 0 <= alpha <= 1; the rest as sph_balance. */
int sph_balance_types(sph_ctx *ctx, int64_t n, const float *posm, int32_t *owner, const int32_t *ptype,
                      int32_t n_types, double alpha, int32_t hmax, int32_t *bal_hash,
                      unsigned long long *swapped);

/* NEXT-3, both passes from ONE neighbour search: the stencil is searched once per particle, the
 * accepted neighbours are split by owner label, and the sums of step e (same label)
 * and of step f (other labels) are accumulated one after the other into two sets of
 * rate arrays.  Equal to sph_interact_split(which = 1) and (which = 2) up to rounding, at the cost
 * of one search instead of two.  (On one GPU the two steps have no exchange between them to wait
 * for; a multi-GPU run that overlaps step e with the broadcast would call the split passes.)
 * sorted_h: per-particle smoothing lengths in sorted order as in sph_interact_varh, or NULL for the
 * uniform sph_params.h.  pair_counts dev [2] out: accepted ordered pairs of step e and of step f
 * (zeroed by the call).  All arrays dev, indexed by sorted position, as in sph_interact. */
int sph_interact_ef(sph_ctx *ctx, int64_t n, const sph_state *sorted, const float *sorted_h,
                    const uint32_t *sorted_hash, const uint32_t *cell_start, const uint32_t *cell_end,
                    float *drho_e, float *acc_e, float *const dsig_e[6], float *drho_f, float *acc_f,
                    float *const dsig_f[6], unsigned long long *pair_counts);

/* NEXT-4, second half -- per-particle smoothing lengths ("cubic
 * buckets of size 2h with h the maximum smoothing length of the particles"; PAPER.md:54 particle
 * types "with different smoothing lengths").  Readings H1-H3: the bucket grid
 * stays the one of sph_params.h, which is now h_max (every h[i] must be in (0, h_max]; larger
 * values lose neighbours outside the 27 buckets, not checked); a pair uses the symmetrised length
 * h_ij = (h_i + h_j) / 2: W(r, h_ij), neighbours = stencil particles with r < 2 h_ij; all sums and
 * the stress rate as in sph_interact.  Every h[i] == sph_params.h gives sph_interact's result up
 * to rounding.  Stages 1-3 do not depend on h.
 * sph_interact_varh: sorted_h dev [n] in sorted order; which = 0 all neighbours, 1 / 2 = the split
 * passes of sph_interact_split; the rest as sph_interact (pair_count is zeroed by the call).
 * sph_step_varh: h dev [n] in ID order (read only; smoothing lengths do not evolve); the rest as
 * sph_step. */
int sph_interact_varh(sph_ctx *ctx, int64_t n, const sph_state *sorted, const float *sorted_h,
                      const uint32_t *sorted_hash, const uint32_t *cell_start, const uint32_t *cell_end,
                      int32_t which, float *drho, float *acc, float *const dsig[6],
                      unsigned long long *pair_count);
int sph_step_varh(sph_ctx *ctx, int64_t n, float dt, const sph_state *state, const float *h, uint32_t *hash,
                  uint32_t *sorted_hash, uint32_t *perm, uint32_t *cell_start, uint32_t *cell_end,
                  uint32_t *comm_hash, uint32_t *boundary_ids, uint32_t *boundary_count,
                  uint32_t *owner_counts, float *drho, float *acc, float *const dsig[6],
                  unsigned long long *pair_count);

/* End-to-end variant with HOST buffers (pinned memory recommended): uploads the id-ordered state,
 * runs `steps` iterations, downloads the state, the boundary list of the last step and the
 * counters, and synchronises the stream before returning.  Device staging lives in the ctx
 * (allocated on first use).  posm goes up first on the ctx's stream, the rest of the state on a
 * second stream owned by the ctx while hash + sort already run; the download follows the last
 * step (its epilogue writes the whole state, so nothing of it can leave earlier).  host_state pointers are host; boundary_ids host capacity n (may be
 * NULL); boundary_count / pair_count host scalars (may be NULL; pair_count accumulates over the
 * steps). */
int sph_step_host(sph_ctx *ctx, int64_t n, float dt, int32_t steps, const sph_state *host_state,
                  uint32_t *boundary_ids, uint32_t *boundary_count, unsigned long long *pair_count);

/* Stage 3 for callers that cannot allocate device memory (step c).
 *
 * Every other entry point works on an sph_ctx, and sph_create obtains the ctx's scratch with
 * cudaMalloc.  Some callers cannot do that: a solver that gave all device memory to its own pool at
 * start-up, a plug-in whose host application forbids allocations (and the device-wide stall of a
 * cudaFree) inside the time loop, a thread feeding a latency-critical stream that must stay clear of
 * the allocator's locks.  For them this call needs NO ctx and calls no cudaMalloc, cudaFree or any
 * allocating routine: its only scratch, one owner bitmask per bucket, is an array of
 * SPH_NOALLOC_MAX_CELLS 32-bit words (16 MiB) built into the library image.  Every GPU that loads
 * the library holds those 16 MiB until the process exits, used or not.
 *
 * Computes, for the same inputs, exactly sph_comm_hash's comm_hash and *boundary_count:
 * comm_hash[k] = sorted_hash[k] if a particle with another owner lies in the 27-bucket stencil of
 * k's bucket, else SPH_GARBAGE_HASH; *boundary_count = number of particles with comm_hash !=
 * garbage.  The boundary list and the owner counts are not produced (they need tables this call has
 * no room for); no cell_start / cell_end are needed.
 * params: host; only dims and n_owners are read (dims > 0, n_owners in 1..SPH_MAX_OWNERS).
 * In: sorted_hash, sorted_owner dev [n], n <= 2^30, sorted by hash, every hash < nx*ny*nz (a larger
 * one gets the garbage hash and marks nothing, never a fault).  Out: comm_hash dev [n],
 * boundary_count dev scalar -- caller-owned like everywhere else.  cuda_stream: a cudaStream_t
 * (NULL = legacy default stream); the call only enqueues on it (two memsets, two kernels).
 * The device is the CURRENT one; all pointers must belong to it.
 *
 * What the shared built-in array implies:
 *  - Limit: nx*ny*nz > SPH_NOALLOC_MAX_CELLS is refused with SPH_ELIMIT before any CUDA call
 *    (BASELINE.json's largest grid, 156^3 = 3.8 M buckets for 64 M particles, fits).
 *  - It keeps the previous call's masks; each call first clears the words of its own grid.
 *  - All calls on one GPU use the same array: calls whose work can overlap on the GPU (different
 *    streams, or host threads that do not order their streams) race and give wrong flags.  Keep
 *    them on one stream or order them with events.
 *  - Set-up: the first call made while a given device is current looks up the array's address on
 *    that device (cudaGetSymbolAddress, once per device, kept for the process).  Make that first
 *    call before starting any stream capture.
 * Errors: SPH_EINVAL (null pointer, n out of range, bad dims / n_owners, device ordinal >= 64),
 * SPH_ELIMIT, SPH_ECUDA (the CUDA error is left pending: read it with cudaGetLastError). */
int sph_comm_hash_noalloc(const sph_params *params, int64_t n, const uint32_t *sorted_hash,
                          const int32_t *sorted_owner, uint32_t *comm_hash, uint32_t *boundary_count,
                          void *cuda_stream);

/* Per-stage device time of sph_step, measured with CUDA events recorded on the ctx's stream
 * (enabled by sph_enable_timing(ctx, 1); adds no host sync to sph_step itself -- sph_get_timing
 * synchronises).  ms[0..7] = hash, sort, reorder, cell_ranges, comm_hash, interact, integrate,
 * total, each the AVERAGE over the steps enqueued since the last sph_get_timing / enable call (at
 * most the 32 most recent: the events live in a ring).  SPH_EINVAL if no step was recorded. */
int sph_enable_timing(sph_ctx *ctx, int32_t on);
int sph_get_timing(sph_ctx *ctx, float ms[8]);

/* How many kernels the library has launched through this ctx since creation. */
int64_t sph_launch_count(const sph_ctx *ctx);

const char *sph_strerror(int code);
const char *sph_last_cuda_error(const sph_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* SPH_B200_H */
