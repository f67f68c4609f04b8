// C-ABI entry points of libsph_b200.so (include/sph.h): argument checks, scratch management and
// the per-iteration sequence of PAPER.md:19-26 on one stream.
#include <math.h>
#include <new>
#include <string.h>

#include "sph_internal.cuh"

using namespace sphb;

namespace {

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Carver {
    char *base;
    size_t off;
    template <typename T> T *take(size_t count)
    {
        off = align_up(off, 256);
        T *p = base ? reinterpret_cast<T *>(base + off) : nullptr;
        off += count * sizeof(T);
        return p;
    }
};

int ceil_log2_u64(uint64_t v)
{
    int b = 0;
    while ((1ull << b) < v) ++b;
    return b;
}

void carve(sph_ctx *c, char *base, size_t *total)
{
    Carver k{base, 0};
    const size_t n = (size_t)(c->max_n > 0 ? c->max_n : 1);
    const size_t cells = c->grid.n_cells;
    const size_t tiles = (n + kSortTile - 1) / kSortTile;
    const size_t scan_n = cells > n ? cells : n;
    const size_t scan_tiles = (scan_n + kScanTile - 1) / kScanTile;
    c->alt_keys = k.take<uint32_t>(n);
    c->alt_vals = k.take<uint32_t>(n);
    c->hist = k.take<uint32_t>(kMaxPasses * kRadix);
    c->tile_status = k.take<uint32_t>((size_t)(c->n_passes > 0 ? c->n_passes : 1) * tiles * kRadix);
    c->tile_counter = k.take<uint32_t>(kMaxPasses + 2);
    c->cell_mask = k.take<uint32_t>(cells);
    c->cell_flag_count = k.take<uint32_t>(cells);
    c->cell_offset = k.take<uint32_t>(cells);
    c->scan_status = k.take<uint32_t>(scan_tiles);
    c->dest_counts = k.take<uint32_t>(2 * (size_t)c->params.n_owners * ((n + 255) / 256));
    c->s_hash = k.take<uint32_t>(n);
    c->s_sorted_hash = k.take<uint32_t>(n);
    c->s_perm = k.take<uint32_t>(n);
    c->s_cell_start = k.take<uint32_t>(cells);
    c->s_cell_end = k.take<uint32_t>(cells);
    c->s_comm_hash = k.take<uint32_t>(n);
    c->s_boundary_ids = k.take<uint32_t>(n);
    c->s_boundary_count = k.take<uint32_t>(4);
    c->s_owner_counts = k.take<uint32_t>(SPH_MAX_OWNERS);
    c->s_drho = k.take<float>(n);
    c->s_acc = k.take<float>(4 * n);
    for (int i = 0; i < 6; ++i) c->s_dsig[i] = k.take<float>(n);
    c->s_pair_count = k.take<unsigned long long>(2);
    c->sorted.posm = k.take<float>(4 * n);
    c->sorted.velr = k.take<float>(4 * n);
    for (int i = 0; i < 6; ++i) c->sorted.sig[i] = k.take<float>(n);
    c->sorted.owner = k.take<int32_t>(n);
    c->sorted_h = k.take<float>(n);
    c->rec_B = k.take<float4>(n + 2);
    c->rec_C = k.take<float4>(n + 2);
    c->rec_D = k.take<float4>(n + 2);
    c->bal = k.take<unsigned long long>((balance_scratch_bytes() + 7) / 8);
    *total = align_up(k.off, 256);
}

bool state_ok(const sph_state *s)
{
    if (!s || !s->posm || !s->velr || !s->owner) return false;
    for (int i = 0; i < 6; ++i)
        if (!s->sig[i]) return false;
    return true;
}

bool n_ok(const sph_ctx *c, int64_t n) { return c && n >= 0 && n <= c->max_n; }

struct StageTimer {
    sph_ctx *c;
    int idx = 0, slot = 0;
    explicit StageTimer(sph_ctx *ctx) : c(ctx)
    {
        // the slot is claimed here but only counted by commit(), after the last mark of a step
        // that enqueued completely: a step that fails midway leaves no half-recorded slot behind
        if (c->timing.on) slot = (int)(c->timing.count % kTimingSlots);
        mark();
    }
    void commit()
    {
        if (c->timing.on) c->timing.count++;
    }
    void mark()
    {
        if (c->timing.on) cudaEventRecord(c->timing.ev[slot][idx], c->stream);
        ++idx;
    }
};

}  // namespace

extern "C" {

static int step_impl(sph_ctx *c, int64_t n, float dt, const sph_state *state, uint32_t *hash,
                     uint32_t *sorted_hash, uint32_t *perm, uint32_t *cell_start, uint32_t *cell_end,
                     uint32_t *comm_hash, uint32_t *boundary_ids, uint32_t *boundary_count,
                     uint32_t *owner_counts, float *drho, float *acc, float *const dsig[6],
                     unsigned long long *pair_count, bool zero_pairs, const float *hp = nullptr);

int sph_create(sph_ctx **out, const sph_params *p, int64_t max_n, void *cuda_stream)
{
    if (!out || !p) return SPH_EINVAL;
    *out = nullptr;
    if (max_n < 0 || max_n >= (1ll << 30)) return SPH_EINVAL;
    if (!(p->h > 0.0f) || !isfinite(p->h)) return SPH_EINVAL;
    if (p->n_owners < 1 || p->n_owners > SPH_MAX_OWNERS) return SPH_EINVAL;
    uint64_t cells = 1;
    for (int a = 0; a < 3; ++a) {
        // above 2^24 a bucket coordinate is no longer exact in fp32 (clamping to (float)(n - 1)
        // and clamping the converted integer to n - 1 would differ): such grids are refused
        if (p->dims[a] <= 0 || p->dims[a] > (1 << 24)) return SPH_EINVAL;
        cells *= (uint64_t)p->dims[a];
        if (cells >= 0xFFFFFFFFull) return SPH_EINVAL;
    }
    if (!isfinite(p->origin[0]) || !isfinite(p->origin[1]) || !isfinite(p->origin[2])) return SPH_EINVAL;

    sph_ctx *c = new (std::nothrow) sph_ctx();
    if (!c) return SPH_ENOMEM;
    c->params = *p;
    c->max_n = max_n;
    c->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    c->launches = 0;
    c->last_err = cudaSuccess;
    c->staging_ready = false;
    c->host_streams_ready = false;
    c->h_count = nullptr;
    c->wait_before_reorder = nullptr;
    c->rec_fresh = false;
    c->hist_for = nullptr;
    c->attr_sort = c->attr_interact = false;
    memset(&c->staging, 0, sizeof(c->staging));

    // grid constants: inv_edge rounded once in fp32 (reading S2)
    const float edge = 2.0f * p->h;
    c->grid.ox = p->origin[0]; c->grid.oy = p->origin[1]; c->grid.oz = p->origin[2];
    c->grid.inv_edge = 1.0f / edge;
    c->grid.nx = p->dims[0]; c->grid.ny = p->dims[1]; c->grid.nz = p->dims[2];
    c->grid.n_cells = (uint32_t)cells;
    // kernel constants (computed in double, rounded once)
    const double h = (double)p->h;
    const double alpha = 21.0 / (16.0 * 3.14159265358979323846 * h * h * h);
    c->consts.support2 = edge * edge;
    c->consts.half_inv_h = (float)(0.5 / h);
    c->consts.cF = (float)(-5.0 * alpha / (h * h));
    c->consts.cF_varh = (float)(-105.0 / (16.0 * 3.14159265358979323846));
    c->consts.K = p->K;
    c->consts.G = p->G;
    c->key_bits = ceil_log2_u64(cells);
    c->n_passes = (c->key_bits + kRadixBits - 1) / kRadixBits;

    cudaError_t e = cudaGetDevice(&c->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, c->device);
    if (e != cudaSuccess) { delete c; return SPH_ECUDA; }

    size_t total = 0;
    carve(c, nullptr, &total);
    c->arena_bytes = total;
    e = cudaMalloc(&c->arena, total);
    if (e != cudaSuccess) { cudaGetLastError(); delete c; return SPH_ENOMEM; }
    carve(c, static_cast<char *>(c->arena), &total);
    *out = c;
    return SPH_OK;
}

int sph_destroy(sph_ctx *c)
{
    if (!c) return SPH_EINVAL;
    cudaStreamSynchronize(c->stream);
    if (c->timing.created)
        for (int s = 0; s < kTimingSlots; ++s)
            for (int i = 0; i < 9; ++i) cudaEventDestroy(c->timing.ev[s][i]);
    if (c->staging_ready) {
        cudaFree(c->staging.posm);
    }
    if (c->host_streams_ready) {
        cudaStreamSynchronize(c->copy_stream);
        cudaEventDestroy(c->ev_posm);
        cudaEventDestroy(c->ev_rest);
        cudaStreamDestroy(c->copy_stream);
        cudaFreeHost(c->h_count);
    }
    cudaFree(c->arena);
    delete c;
    return SPH_OK;
}

int sph_hash(sph_ctx *c, int64_t n, const float *posm, uint32_t *hash)
{
    if (!n_ok(c, n) || !posm || !hash) return SPH_EINVAL;
    return launch_hash(c, n, posm, hash);
}

int sph_sort(sph_ctx *c, int64_t n, const uint32_t *hash, uint32_t *sorted_hash, uint32_t *perm)
{
    if (!n_ok(c, n) || !hash || !sorted_hash || !perm) return SPH_EINVAL;
    return launch_sort(c, n, hash, sorted_hash, perm);
}

int sph_reorder(sph_ctx *c, int64_t n, const uint32_t *perm, const sph_state *in, const sph_state *out)
{
    if (!n_ok(c, n) || !perm || !state_ok(in) || !state_ok(out)) return SPH_EINVAL;
    return launch_reorder(c, n, perm, in, out);
}

int sph_pack_boundary(sph_ctx *c, int64_t n, int64_t m, const sph_state *state, const uint32_t *boundary_ids,
                      uint32_t *owner_offsets, uint32_t *packed_ids, const sph_state *packed)
{
    if (!n_ok(c, n) || m < 0 || m > n || !state_ok(state) || !owner_offsets) return SPH_EINVAL;
    if (m > 0 && (!boundary_ids || !packed_ids || !state_ok(packed))) return SPH_EINVAL;
    uint32_t *dest = c->s_boundary_ids;   // scratch: destination of every list entry
    if (boundary_ids == dest) return SPH_EINVAL;
    int rc = launch_partition_by_label(c, m, boundary_ids, state->owner, c->params.n_owners, owner_offsets, dest);
    if (rc != SPH_OK || m == 0) return rc;
    return launch_scatter_records(c, m, boundary_ids, dest, state, packed, packed_ids);
}

int sph_balance(sph_ctx *c, int64_t n, const float *posm, int32_t *owner, int32_t hmax, int32_t *bal_hash,
                unsigned long long *swapped)
{
    if (!n_ok(c, n) || !posm || !owner || hmax < 1 || hmax > 1023) return SPH_EINVAL;
    return launch_balance(c, n, posm, owner, nullptr, 1, 0.0, hmax, bal_hash, swapped);
}

int sph_balance_types(sph_ctx *c, int64_t n, const float *posm, int32_t *owner, const int32_t *ptype,
                      int32_t n_types, double alpha, int32_t hmax, int32_t *bal_hash, unsigned long long *swapped)
{
    if (!n_ok(c, n) || !posm || !owner || !ptype || hmax < 1 || hmax > 1023 || n_types < 1 || n_types > 8 ||
        !(alpha >= 0.0 && alpha <= 1.0))
        return SPH_EINVAL;
    return launch_balance(c, n, posm, owner, ptype, n_types, alpha, hmax, bal_hash, swapped);
}

int sph_cell_ranges(sph_ctx *c, int64_t n, const uint32_t *sorted_hash, uint32_t *cs, uint32_t *ce)
{
    if (!n_ok(c, n) || !sorted_hash || !cs || !ce) return SPH_EINVAL;
    return launch_cell_ranges(c, n, sorted_hash, cs, ce);
}

int sph_comm_hash(sph_ctx *c, int64_t n, const uint32_t *sorted_hash, const int32_t *sorted_owner,
                  const uint32_t *perm, const uint32_t *cs, const uint32_t *ce, uint32_t *comm_hash,
                  uint32_t *boundary_ids, uint32_t *boundary_count, uint32_t *owner_counts)
{
    if (!n_ok(c, n) || !sorted_hash || !sorted_owner || !perm || !cs || !ce || !comm_hash ||
        !boundary_ids || !boundary_count || !owner_counts)
        return SPH_EINVAL;
    return launch_comm_hash(c, n, sorted_hash, sorted_owner, perm, cs, ce, comm_hash, boundary_ids,
                            boundary_count, owner_counts);
}

int sph_interact(sph_ctx *c, int64_t n, const sph_state *sorted, const uint32_t *sorted_hash,
                 const uint32_t *cs, const uint32_t *ce, float *drho, float *acc,
                 float *const dsig[6], unsigned long long *pair_count)
{
    if (!n_ok(c, n) || !state_ok(sorted) || !sorted_hash || !cs || !ce || !drho || !acc || !dsig)
        return SPH_EINVAL;
    for (int i = 0; i < 6; ++i)
        if (!dsig[i]) return SPH_EINVAL;
    if (pair_count)
        SPH_CUDA_TRY(c, cudaMemsetAsync(pair_count, 0, sizeof(unsigned long long), c->stream));
    return launch_interact(c, n, sorted, sorted_hash, cs, ce, drho, acc, dsig, pair_count, nullptr, nullptr, 0.f);
}

int sph_interact_split(sph_ctx *c, int64_t n, const sph_state *sorted, const uint32_t *sorted_hash,
                       const uint32_t *cs, const uint32_t *ce, int32_t which, float *drho, float *acc,
                       float *const dsig[6], unsigned long long *pair_count)
{
    if (!n_ok(c, n) || !state_ok(sorted) || !sorted_hash || !cs || !ce || !drho || !acc || !dsig) return SPH_EINVAL;
    if (which != 1 && which != 2) return SPH_EINVAL;
    for (int i = 0; i < 6; ++i)
        if (!dsig[i]) return SPH_EINVAL;
    return launch_interact(c, n, sorted, sorted_hash, cs, ce, drho, acc, dsig, pair_count, nullptr, nullptr, 0.f,
                           which);
}

int sph_interact_ef(sph_ctx *c, int64_t n, const sph_state *sorted, const float *sorted_h,
                    const uint32_t *sorted_hash, const uint32_t *cs, const uint32_t *ce, float *drho_e,
                    float *acc_e, float *const dsig_e[6], float *drho_f, float *acc_f, float *const dsig_f[6],
                    unsigned long long *pair_counts)
{
    if (!n_ok(c, n) || !state_ok(sorted) || !sorted_hash || !cs || !ce || !drho_e || !acc_e || !dsig_e || !drho_f ||
        !acc_f || !dsig_f || !pair_counts)
        return SPH_EINVAL;
    for (int i = 0; i < 6; ++i)
        if (!dsig_e[i] || !dsig_f[i]) return SPH_EINVAL;
    SPH_CUDA_TRY(c, cudaMemsetAsync(pair_counts, 0, 2 * sizeof(unsigned long long), c->stream));
    return launch_interact(c, n, sorted, sorted_hash, cs, ce, drho_e, acc_e, dsig_e, pair_counts, nullptr, nullptr,
                           0.f, 3, sorted_h, drho_f, acc_f, dsig_f);
}

int sph_pack_destinations(sph_ctx *c, int64_t n, const uint32_t *sorted_hash, const int32_t *sorted_owner,
                          const uint32_t *perm, uint32_t *dest_offsets, uint32_t *dest_ids, int64_t cap)
{
    if (!n_ok(c, n) || !dest_offsets || cap < 0) return SPH_EINVAL;
    if (n > 0 && (!sorted_hash || !sorted_owner || !perm)) return SPH_EINVAL;
    if (n * (int64_t)(c->params.n_owners - 1) >= (1ll << 30)) return SPH_ELIMIT;   // 30-bit scan prefixes
    return launch_pack_destinations(c, n, sorted_hash, sorted_owner, perm, dest_offsets, dest_ids, cap);
}

int sph_integrate(sph_ctx *c, int64_t n, float dt, const sph_state *in, const float *drho,
                  const float *acc, const float *const dsig[6], const sph_state *out)
{
    if (!n_ok(c, n) || !state_ok(in) || !state_ok(out) || !drho || !acc || !dsig) return SPH_EINVAL;
    for (int i = 0; i < 6; ++i)
        if (!dsig[i]) return SPH_EINVAL;
    return launch_integrate(c, n, dt, in, drho, acc, dsig, out, nullptr);
}

static int step_impl(sph_ctx *c, int64_t n, float dt, const sph_state *state, uint32_t *hash,
                     uint32_t *sorted_hash, uint32_t *perm, uint32_t *cell_start, uint32_t *cell_end,
                     uint32_t *comm_hash, uint32_t *boundary_ids, uint32_t *boundary_count,
                     uint32_t *owner_counts, float *drho, float *acc, float *const dsig[6],
                     unsigned long long *pair_count, bool zero_pairs, const float *hp)
{
    if (!n_ok(c, n) || !state || (n > 0 && !state_ok(state))) return SPH_EINVAL;
    if (pair_count && zero_pairs)
        SPH_CUDA_TRY(c, cudaMemsetAsync(pair_count, 0, sizeof(unsigned long long), c->stream));
    if (!hash) hash = c->s_hash;
    if (!sorted_hash) sorted_hash = c->s_sorted_hash;
    if (!perm) perm = c->s_perm;
    if (!cell_start) cell_start = c->s_cell_start;
    if (!cell_end) cell_end = c->s_cell_end;
    if (!comm_hash) comm_hash = c->s_comm_hash;
    if (!boundary_ids) boundary_ids = c->s_boundary_ids;
    if (!boundary_count) boundary_count = c->s_boundary_count;
    if (!owner_counts) owner_counts = c->s_owner_counts;
    // the rates are an optional product: when the caller wants none of them the fused epilogue
    // does not store them at all
    const bool want_rates = drho || acc || (dsig && (dsig[0] || dsig[1] || dsig[2] || dsig[3] || dsig[4] || dsig[5]));
    float *ds[6];
    for (int i = 0; i < 6; ++i) ds[i] = (dsig && dsig[i]) ? dsig[i] : c->s_dsig[i];
    if (want_rates) {
        if (!drho) drho = c->s_drho;
        if (!acc) acc = c->s_acc;
    }

    int rc;
    StageTimer t(c);
    if ((rc = launch_hash_hist(c, n, state->posm, hash)) != SPH_OK) return rc;             // step a (+ the sort's histograms)
    t.mark();
    if ((rc = launch_sort(c, n, hash, sorted_hash, perm)) != SPH_OK) return rc;
    t.mark();
    if (c->wait_before_reorder) {   // sph_step_host: the rest of the state arrives on the copy stream
        SPH_CUDA_TRY(c, cudaStreamWaitEvent(c->stream, c->wait_before_reorder, 0));
        c->wait_before_reorder = nullptr;
    }
    if ((rc = launch_reorder(c, n, perm, state, &c->sorted, hp, c->sorted_h)) != SPH_OK) return rc;
    t.mark();
    if ((rc = launch_cell_ranges(c, n, sorted_hash, cell_start, cell_end)) != SPH_OK) return rc;
    t.mark();
    if ((rc = launch_comm_hash(c, n, sorted_hash, c->sorted.owner, perm, cell_start, cell_end,   // step c
                               comm_hash, boundary_ids, boundary_count, owner_counts)) != SPH_OK)
        return rc;
    t.mark();
    // steps e, f and g: the interaction epilogue integrates (O9) and scatters the result back to
    // id order through perm; `state` is only written, the loops read the sorted copy
    if ((rc = launch_interact(c, n, &c->sorted, sorted_hash, cell_start, cell_end, want_rates ? drho : nullptr,
                              want_rates ? acc : nullptr, want_rates ? ds : nullptr, pair_count, state, perm,
                              dt, 0, hp ? c->sorted_h : nullptr)) != SPH_OK)
        return rc;
    t.mark();
    t.mark();
    t.commit();
    return SPH_OK;
}

int sph_step(sph_ctx *c, int64_t n, float dt, const sph_state *state, uint32_t *hash,
             uint32_t *sorted_hash, uint32_t *perm, uint32_t *cell_start, uint32_t *cell_end,
             uint32_t *comm_hash, uint32_t *boundary_ids, uint32_t *boundary_count,
             uint32_t *owner_counts, float *drho, float *acc, float *const dsig[6],
             unsigned long long *pair_count)
{
    return step_impl(c, n, dt, state, hash, sorted_hash, perm, cell_start, cell_end, comm_hash,
                     boundary_ids, boundary_count, owner_counts, drho, acc, dsig, pair_count, true);
}

int sph_step_varh(sph_ctx *c, int64_t n, float dt, const sph_state *state, const float *h, uint32_t *hash,
                  uint32_t *sorted_hash, uint32_t *perm, uint32_t *cell_start, uint32_t *cell_end,
                  uint32_t *comm_hash, uint32_t *boundary_ids, uint32_t *boundary_count,
                  uint32_t *owner_counts, float *drho, float *acc, float *const dsig[6],
                  unsigned long long *pair_count)
{
    if (!h && n > 0) return SPH_EINVAL;
    return step_impl(c, n, dt, state, hash, sorted_hash, perm, cell_start, cell_end, comm_hash,
                     boundary_ids, boundary_count, owner_counts, drho, acc, dsig, pair_count, true, h);
}

int sph_interact_varh(sph_ctx *c, int64_t n, const sph_state *sorted, const float *sorted_h,
                      const uint32_t *sorted_hash, const uint32_t *cs, const uint32_t *ce, int32_t which,
                      float *drho, float *acc, float *const dsig[6], unsigned long long *pair_count)
{
    if (!n_ok(c, n) || !state_ok(sorted) || !sorted_h || !sorted_hash || !cs || !ce || !drho || !acc || !dsig)
        return SPH_EINVAL;
    if (which < 0 || which > 2) return SPH_EINVAL;
    for (int i = 0; i < 6; ++i)
        if (!dsig[i]) return SPH_EINVAL;
    if (pair_count)
        SPH_CUDA_TRY(c, cudaMemsetAsync(pair_count, 0, sizeof(unsigned long long), c->stream));
    return launch_interact(c, n, sorted, sorted_hash, cs, ce, drho, acc, dsig, pair_count, nullptr, nullptr, 0.f,
                           which, sorted_h);
}

static int step_host_impl(sph_ctx *c, int64_t n, float dt, int32_t steps, const sph_state *hs,
                          uint32_t *boundary_ids, uint32_t *boundary_count, unsigned long long *pair_count)
{
    if (!c->staging_ready) {
        const size_t m = (size_t)(c->max_n > 0 ? c->max_n : 1);
        char *base = nullptr;
        // posm 16, velr 16, sig 24, owner 4 bytes per particle, each block 256-aligned
        const size_t bytes = align_up(16 * m, 256) * 2 + align_up(4 * m, 256) * 7;
        if (cudaMalloc(&base, bytes) != cudaSuccess) { cudaGetLastError(); return SPH_ENOMEM; }
        Carver k{base, 0};
        c->staging.posm = k.take<float>(4 * m);
        c->staging.velr = k.take<float>(4 * m);
        for (int i = 0; i < 6; ++i) c->staging.sig[i] = k.take<float>(m);
        c->staging.owner = k.take<int32_t>(m);
        c->staging_ready = true;
    }
    const sph_state &d = c->staging;
    cudaStream_t s = c->stream;
    const size_t nn = (size_t)n;
    if (!c->host_streams_ready) {
        SPH_CUDA_TRY(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
        SPH_CUDA_TRY(c, cudaEventCreateWithFlags(&c->ev_posm, cudaEventDisableTiming));
        SPH_CUDA_TRY(c, cudaEventCreateWithFlags(&c->ev_rest, cudaEventDisableTiming));
        // pinned landing word for the boundary count (an async D2H into pageable stack memory
        // would only be safe because of the synchronisation that follows it)
        SPH_CUDA_TRY(c, cudaHostAlloc(reinterpret_cast<void **>(&c->h_count), sizeof(uint32_t), cudaHostAllocDefault));
        c->host_streams_ready = true;
    }
    // posm first, on the ctx's stream: hash, sort and nothing else of the step can start on it.
    // The other 44 bytes per particle follow on the copy stream (behind posm, so that the two
    // uploads do not share the link), and the step waits for them in front of its reorder pass.
    cudaStream_t s2 = c->copy_stream;
    SPH_CUDA_TRY(c, cudaMemcpyAsync(d.posm, hs->posm, 16 * nn, cudaMemcpyHostToDevice, s));
    SPH_CUDA_TRY(c, cudaEventRecord(c->ev_posm, s));
    SPH_CUDA_TRY(c, cudaStreamWaitEvent(s2, c->ev_posm, 0));
    SPH_CUDA_TRY(c, cudaMemcpyAsync(d.velr, hs->velr, 16 * nn, cudaMemcpyHostToDevice, s2));
    for (int i = 0; i < 6; ++i)
        SPH_CUDA_TRY(c, cudaMemcpyAsync(d.sig[i], hs->sig[i], 4 * nn, cudaMemcpyHostToDevice, s2));
    SPH_CUDA_TRY(c, cudaMemcpyAsync(d.owner, hs->owner, 4 * nn, cudaMemcpyHostToDevice, s2));
    SPH_CUDA_TRY(c, cudaEventRecord(c->ev_rest, s2));
    c->wait_before_reorder = c->ev_rest;
    SPH_CUDA_TRY(c, cudaMemsetAsync(c->s_pair_count, 0, 2 * sizeof(unsigned long long), s));
    for (int32_t it = 0; it < steps; ++it) {
        int rc = step_impl(c, n, dt, &d, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr,
                           nullptr, nullptr, nullptr, nullptr, nullptr, c->s_pair_count, false);
        if (rc != SPH_OK) return rc;
    }
    if (c->wait_before_reorder) {   // steps == 0: nothing has waited for the second upload yet
        SPH_CUDA_TRY(c, cudaStreamWaitEvent(s, c->wait_before_reorder, 0));
        c->wait_before_reorder = nullptr;
    }
    SPH_CUDA_TRY(c, cudaMemcpyAsync(hs->posm, d.posm, 16 * nn, cudaMemcpyDeviceToHost, s));
    SPH_CUDA_TRY(c, cudaMemcpyAsync(hs->velr, d.velr, 16 * nn, cudaMemcpyDeviceToHost, s));
    for (int i = 0; i < 6; ++i)
        SPH_CUDA_TRY(c, cudaMemcpyAsync(hs->sig[i], d.sig[i], 4 * nn, cudaMemcpyDeviceToHost, s));
    uint32_t m_host = 0;
    if (steps > 0 && (boundary_ids || boundary_count)) {
        SPH_CUDA_TRY(c, cudaMemcpyAsync(c->h_count, c->s_boundary_count, sizeof(uint32_t),
                                        cudaMemcpyDeviceToHost, s));
        SPH_CUDA_TRY(c, cudaStreamSynchronize(s));
        m_host = *c->h_count;
        if (boundary_ids && m_host)
            SPH_CUDA_TRY(c, cudaMemcpyAsync(boundary_ids, c->s_boundary_ids, sizeof(uint32_t) * m_host,
                                            cudaMemcpyDeviceToHost, s));
    }
    if (boundary_count) *boundary_count = m_host;
    if (pair_count)
        SPH_CUDA_TRY(c, cudaMemcpyAsync(pair_count, c->s_pair_count, sizeof(unsigned long long),
                                        cudaMemcpyDeviceToHost, s));
    SPH_CUDA_TRY(c, cudaStreamSynchronize(s));
    return SPH_OK;
}

int sph_step_host(sph_ctx *c, int64_t n, float dt, int32_t steps, const sph_state *hs,
                  uint32_t *boundary_ids, uint32_t *boundary_count, unsigned long long *pair_count)
{
    if (!n_ok(c, n) || !state_ok(hs) || steps < 0) return SPH_EINVAL;
    const int rc = step_host_impl(c, n, dt, steps, hs, boundary_ids, boundary_count, pair_count);
    if (rc != SPH_OK) {
        // a failure after the copies were enqueued: do not return while either stream may still
        // read or write the caller's host buffers, and leave no pending wait for a later sph_step
        c->wait_before_reorder = nullptr;
        if (c->host_streams_ready) cudaStreamSynchronize(c->copy_stream);
        cudaStreamSynchronize(c->stream);
    }
    return rc;
}

int sph_enable_timing(sph_ctx *c, int32_t on)
{
    if (!c) return SPH_EINVAL;
    if (on && !c->timing.created) {
        for (int s = 0; s < kTimingSlots; ++s)
            for (int i = 0; i < 9; ++i) SPH_CUDA_TRY(c, cudaEventCreate(&c->timing.ev[s][i]));
        c->timing.created = true;
    }
    c->timing.on = on != 0;
    c->timing.count = 0;
    return SPH_OK;
}

int sph_get_timing(sph_ctx *c, float ms[8])
{
    if (!c || !ms) return SPH_EINVAL;
    if (!c->timing.created || c->timing.count == 0) return SPH_EINVAL;
    SPH_CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    const int m = (int)(c->timing.count < kTimingSlots ? c->timing.count : kTimingSlots);
    for (int i = 0; i < 8; ++i) ms[i] = 0.f;
    for (int k = 0; k < m; ++k) {   // the m most recent steps
        const int s = (int)((c->timing.count - 1 - k) % kTimingSlots);
        float t;
        for (int i = 0; i < 7; ++i) {
            SPH_CUDA_TRY(c, cudaEventElapsedTime(&t, c->timing.ev[s][i], c->timing.ev[s][i + 1]));
            ms[i] += t / (float)m;
        }
        SPH_CUDA_TRY(c, cudaEventElapsedTime(&t, c->timing.ev[s][0], c->timing.ev[s][7]));
        ms[7] += t / (float)m;
    }
    c->timing.count = 0;
    return SPH_OK;
}

int64_t sph_launch_count(const sph_ctx *c) { return c ? c->launches : -1; }

const char *sph_strerror(int code)
{
    switch (code) {
    case SPH_OK: return "ok";
    case SPH_EINVAL: return "invalid argument";
    case SPH_ECUDA: return "CUDA error";
    case SPH_ENOMEM: return "out of device memory";
    case SPH_ELIMIT: return "size beyond a fixed capacity of the entry point (sph_comm_hash_noalloc: more than SPH_NOALLOC_MAX_CELLS buckets; sph_pack_destinations: n (n_owners - 1) >= 2^30)";
    default: return "unknown error";
    }
}

const char *sph_last_cuda_error(const sph_ctx *c)
{
    return c ? cudaGetErrorString(c->last_err) : "no context";
}

}  // extern "C"
