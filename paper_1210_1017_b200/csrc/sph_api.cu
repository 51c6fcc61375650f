// C-ABI entry points of libsph_b200.so (include/sph_b200.h): argument checks, workspace
// carving, call-order bookkeeping and stage timers.  All arithmetic of the method runs in the
// kernels of keys.cu / radix_sort.cu / gather_cells.cu / halo_migrate.cu / interact.cu / verlet.cu.
#include <math.h>
#include <new>
#include <stdio.h>
#include <string.h>
#include "sph_internal.cuh"

using namespace sph;

namespace {

constexpr size_t ALIGN = 256;
size_t align_up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

struct Layout {
    size_t pos4[2], velrho4[2], velrhoM1[2], idt[2], acc4, mumax, dt_red, kv[2], keyword, hist, tile_state, counters,
        cell_begin, cell_loc, gap_list, mig_tile, mig_grp, mig_off, scratch64, slab_begin, halo_range, halo_offset, halo_pos4, halo_velrho4, halo_idt,
        migrants, mig_total, mig_count, prev_init, flags, ia_tiles, total;
};

bool grid_of(const sph_params *p, int nc[3], uint64_t *ncells)
{
    if (!(p->h > 0.f) || !isfinite(p->h)) return false;
    uint64_t tot = 1;
    for (int k = 0; k < 3; ++k) {
        double ext = (double)p->dom_max[k] - (double)p->dom_min[k];
        if (!(ext > 0.0) || !isfinite(ext)) return false;
        double c = ceil(ext / (2.0 * (double)p->h));
        if (c < 1.0) c = 1.0;
        if (c > 268435456.0) return false;
        nc[k] = (int)c;
        tot *= (uint64_t)nc[k];
        if (tot > (1ull << 28)) return false;
    }
    *ncells = tot;
    return true;
}

// cells per z-block of a tile of the production interaction kernel: 2 x 2 columns x zm cells fill an
// item's target list
int mma_zblock(const sph_params *p)
{
    double ppc = pow(2.0 * (double)p->h / (double)p->dp, 3.0);
    int zm = (int)floor((double)interact_mma_targets() * 0.97 / (4.0 * (ppc > 0.05 ? ppc : 0.05)));
    if (zm < 1) zm = 1;
    if (zm > interact_mma_zmax()) zm = interact_mma_zmax();
    return zm;
}

bool make_layout(const sph_params *p, uint64_t n, int max_slabs, Layout *L)
{
    int nc[3];
    uint64_t ncells;
    if (!p || n > (1ull << 28) || max_slabs < 1 || max_slabs > SPH_MAX_SLABS) return false;
    if (!grid_of(p, nc, &ncells)) return false;
    size_t off = 0;
    size_t nn = n ? n : 1;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
    for (int b = 0; b < 2; ++b) {
        L->pos4[b] = take(16 * nn);
        L->velrho4[b] = take(16 * nn);
        L->velrhoM1[b] = take(16 * nn);
        L->idt[b] = take(4 * nn);
    }
    L->acc4 = take(16 * nn);
    L->mumax = take(4 * nn);
    L->dt_red = take(4 * 2 * SPH_MAX_SLABS);
    L->kv[0] = take(8 * nn);
    L->kv[1] = take(8 * nn);
    L->keyword = take(4 * nn);
    L->hist = take(4 * 256 * 4);
    uint32_t tiles = radix_tiles(nn);
    L->tile_state = take((size_t)4 * 256 * tiles * 4);
    L->counters = take(4 * 64);
    L->cell_begin = take(4 * (ncells + 1));
    L->cell_loc = take(max_slabs > 1 ? 4 * (ncells + 1) : 4);
    L->gap_list = take(16 * gap_list_entries(ncells));
    L->mig_tile = take(4 * ((size_t)gather_tiles(nn) + 1));
    L->mig_grp = take(4 * ((size_t)mig_groups(nn) + 1));
    L->mig_off = take(4 * ((size_t)mig_groups(nn) + 1));
    L->scratch64 = take(16);
    L->slab_begin = take(4 * (SPH_MAX_SLABS + 1));
    L->halo_range = take(4 * 4 * SPH_MAX_SLABS);
    L->halo_offset = take(4 * (2 * SPH_MAX_SLABS + 1));
    size_t hn = max_slabs > 1 ? nn : 1;        // every particle is in at most one halo list
    L->halo_pos4 = take(16 * hn);
    L->halo_velrho4 = take(16 * hn);
    L->halo_idt = take(4 * hn);
    L->migrants = take(16 * hn);
    L->mig_total = take(4);
    L->mig_count = take(4 * 2 * SPH_MAX_SLABS);
    L->prev_init = take(nn);
    L->flags = take(4);
    L->ia_tiles = take(4 * interact_mma_tile_capacity(nc, mma_zblock(p)));
    L->total = off;
    return true;
}

// The library never prints: the text of the last failed CUDA call is kept for sph_last_cuda_error
// (per context, and in a per-thread slot for failures before a context exists).
thread_local char g_last_cuda_error[160] = "";

int cuda_fail(sph_ctx *c, cudaError_t e)
{
    if (e == cudaSuccess) return SPH_OK;
    const char *msg = cudaGetErrorString(e);
    snprintf(g_last_cuda_error, sizeof(g_last_cuda_error), "%s", msg ? msg : "unknown CUDA error");
    if (c) {
        c->sticky = SPH_ERR_CUDA;
        snprintf(c->last_cuda_error, sizeof(c->last_cuda_error), "%s", g_last_cuda_error);
    }
    return SPH_ERR_CUDA;
}
#define CK(c, call)                                       \
    do {                                                  \
        cudaError_t e__ = (call);                         \
        if (e__ != cudaSuccess) return cuda_fail(c, e__); \
    } while (0)

bool planes_ok(const int32_t *planes, int S, int ncx, int max_slabs)
{
    if (!planes || S < 1 || S > max_slabs) return false;
    if (planes[0] != 0 || planes[S] != ncx) return false;
    for (int s = 0; s < S; ++s) {
        int w = planes[s + 1] - planes[s];
        if (w < 1 || (S > 1 && w < 2)) return false;
    }
    return true;
}

bool same_slabs(const SlabC &a, const SlabC &b)
{
    if (a.n_slabs != b.n_slabs) return false;
    for (int s = 0; s <= a.n_slabs; ++s)
        if (a.planes[s] != b.planes[s]) return false;
    return true;
}

void fill_phys(sph_ctx *c)
{
    const sph_params &P = c->P;
    PhysC &ph = c->phys;
    const double pi = 3.14159265358979323846;
    double h = P.h;
    ph.h = P.h;
    ph.inv_h_half = (float)(0.5 / h);
    ph.four_h2 = (float)(4.0 * h * h);
    ph.eta2 = (float)(0.01 * h * h);
    if (P.kernel == 0) ph.kF = (float)(-5.0 * 21.0 / (16.0 * pi * h * h * h) / (h * h));
    else ph.kF = (float)(1.0 / (pi * h * h * h) / (h * h));
    ph.alpha_h = (float)((double)P.alpha * h);
    ph.rho0 = P.rho0;
    ph.inv_rho0 = (float)(1.0 / (double)P.rho0);
    ph.c0 = P.c0;
    ph.B = (float)((double)P.c0 * P.c0 * P.rho0 / (double)P.gamma);
    ph.gamma = P.gamma;
    double binom = 1.0;
    for (int k = 0; k < 16; ++k) ph.tait[k] = 0.f;
    for (int k = 1; k <= P.gamma; ++k) {
        binom = binom * (double)(P.gamma - k + 1) / (double)k;
        ph.tait[k] = (float)binom;
    }
    for (int k = 0; k < 3; ++k) ph.g[k] = P.g[k];
    ph.mass_fluid = P.mass_fluid;
    ph.mass_bound = P.mass_bound;
    ph.uniform_mass = (P.mass_fluid == P.mass_bound) ? 1 : 0;
    ph.kernel = P.kernel;
}

// ---- stage timers ----------------------------------------------------------------------------
struct Timed {
    sph_ctx *c;
    int idx;
    Timed(sph_ctx *ctx, int stage) : c(ctx), idx(-1)
    {
        StageTimer &t = c->timer;
        if (!t.enabled || t.n_pairs >= StageTimer::MAX_PAIRS) return;
        idx = t.n_pairs++;
        while (t.n_created < 2 * (idx + 1)) {
            if (cudaEventCreate(&t.ev[t.n_created]) != cudaSuccess) { idx = -1; --t.n_pairs; return; }
            ++t.n_created;
        }
        t.stage[idx] = stage;
        cudaEventRecord(t.ev[2 * idx], c->stream);
    }
    ~Timed()
    {
        if (idx >= 0) cudaEventRecord(c->timer.ev[2 * idx + 1], c->stream);
    }
};

int upload_state(sph_ctx *c, const sph_particles *part)
{
    const uint64_t n = c->n;
    if (!part || part->n != n) return SPH_ERR_ARG;
    if (n && (!part->pos || !part->vel || !part->rho)) return SPH_ERR_ARG;
    c->cur = 0;
    const float *dpos = part->pos, *dvel = part->vel, *drho = part->rho;
    const uint8_t *dtype = part->type;
    if (n && !part->on_device) {
        // stage the host arrays in the idle half of the double buffers
        float *spos = (float *)c->pos4[1], *svel = (float *)c->velrho4[1];
        float *srho = (float *)c->velrhoM1[1];
        uint8_t *stype = (uint8_t *)c->idt[1];
        CK(c, cudaMemcpyAsync(spos, part->pos, 12 * n, cudaMemcpyHostToDevice, c->stream));
        CK(c, cudaMemcpyAsync(svel, part->vel, 12 * n, cudaMemcpyHostToDevice, c->stream));
        CK(c, cudaMemcpyAsync(srho, part->rho, 4 * n, cudaMemcpyHostToDevice, c->stream));
        if (part->type) CK(c, cudaMemcpyAsync(stype, part->type, n, cudaMemcpyHostToDevice, c->stream));
        dpos = spos; dvel = svel; drho = srho;
        dtype = part->type ? stype : nullptr;
    }
    if (n && part->prev_slab) {
        CK(c, cudaMemcpyAsync(c->prev_init, part->prev_slab, n,
                              part->on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, c->stream));
        c->have_prev_init = true;
    } else {
        c->have_prev_init = false;
    }
    CK(c, cudaMemsetAsync(c->flags, 0, 4, c->stream));
    CK(c, launch_init_state(c, dpos, dvel, drho, dtype));
    if (!part->on_device) CK(c, cudaStreamSynchronize(c->stream));   // host arrays may be reused
    c->have_prev_ranges = false;
    c->sort_had_prev = false;
    c->id_order = true;
    c->sorted_valid = c->halos_valid = c->rates_valid = c->mu_valid = false;
    c->step_index = 0;
    return SPH_OK;
}

}  // namespace

extern "C" {

size_t sph_workspace_bytes(const sph_params *p, uint64_t n_max, int max_slabs)
{
    Layout L;
    if (!make_layout(p, n_max, max_slabs, &L)) return 0;
    return L.total;
}

int sph_init(sph_ctx **out, const sph_params *p, const sph_particles *part, int max_slabs,
             void *workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (!out || !p || !part) return SPH_ERR_ARG;
    *out = nullptr;
    if (p->gamma < 1 || p->gamma > 15 || !(p->rho0 > 0.f) || !(p->c0 > 0.f) || !(p->h > 0.f) || !(p->dp > 0.f) ||
        (p->kernel != 0 && p->kernel != 1) || max_slabs < 1 || max_slabs > SPH_MAX_SLABS)
        return SPH_ERR_ARG;
    int nc[3];
    uint64_t ncells;
    if (part->n > (1ull << 28)) return SPH_ERR_GRID_TOO_LARGE;
    if (!grid_of(p, nc, &ncells)) {
        for (int k = 0; k < 3; ++k)
            if (!(p->dom_max[k] > p->dom_min[k])) return SPH_ERR_ARG;
        return SPH_ERR_GRID_TOO_LARGE;
    }
    Layout L;
    if (!make_layout(p, part->n, max_slabs, &L)) return SPH_ERR_ARG;
    if (!workspace || ((uintptr_t)workspace % ALIGN) != 0 || workspace_bytes < L.total) return SPH_ERR_WORKSPACE;

    sph_ctx *c = new (std::nothrow) sph_ctx();
    if (!c) return SPH_ERR_ARG;
    c->P = *p;
    c->n = part->n;
    c->max_slabs = max_slabs;
    c->stream = (cudaStream_t)cuda_stream;
    c->sticky = SPH_OK;
    for (int k = 0; k < 3; ++k) { c->grid.min[k] = p->dom_min[k]; c->grid.nc[k] = nc[k]; }
    c->grid.inv_cell = 1.0f / (2.0f * p->h);      // two separately rounded fp32 operations
    c->grid.nyz = nc[1] * nc[2];
    c->grid.ncells = (uint32_t)ncells;
    int bits = 1;
    while ((1ull << bits) < ncells) ++bits;
    c->cell_bits = bits;
    c->passes = (bits + 7) / 8;
    c->slabs.n_slabs = 1;
    for (int s = 0; s <= SPH_MAX_SLABS; ++s) c->slabs.planes[s] = 0;
    c->slabs.planes[1] = nc[0];
    c->tagged_slabs = c->slabs;
    fill_phys(c);

    char *w = (char *)workspace;
    for (int b = 0; b < 2; ++b) {
        c->pos4[b] = (float4 *)(w + L.pos4[b]);
        c->velrho4[b] = (float4 *)(w + L.velrho4[b]);
        c->velrhoM1[b] = (float4 *)(w + L.velrhoM1[b]);
        c->idt[b] = (uint32_t *)(w + L.idt[b]);
        c->kv[b] = (uint2 *)(w + L.kv[b]);
    }
    c->acc4 = (float4 *)(w + L.acc4);
    c->mumax = (float *)(w + L.mumax);
    c->dt_red = (uint32_t *)(w + L.dt_red);
    c->adaptive_dt = 0;
    c->mu_valid = false;
    c->keyword = (uint32_t *)(w + L.keyword);
    c->hist = (uint32_t *)(w + L.hist);
    c->tile_state = (uint32_t *)(w + L.tile_state);
    c->counters = (uint32_t *)(w + L.counters);
    c->rs_tiles = radix_tiles(c->n);
    c->cell_begin = (uint32_t *)(w + L.cell_begin);
    c->cell_loc = (uint32_t *)(w + L.cell_loc);
    c->ia_ov.on = false;
    c->gap_list = (uint4 *)(w + L.gap_list);
    c->mig_tile = (uint32_t *)(w + L.mig_tile);
    c->mig_grp = (uint32_t *)(w + L.mig_grp);
    c->mig_off = (uint32_t *)(w + L.mig_off);
    c->scratch64 = (unsigned long long *)(w + L.scratch64);
    c->slab_begin = (uint32_t *)(w + L.slab_begin);
    c->halo_range = (uint32_t *)(w + L.halo_range);
    c->halo_offset = (uint32_t *)(w + L.halo_offset);
    c->halo_pos4 = (float4 *)(w + L.halo_pos4);
    c->halo_velrho4 = (float4 *)(w + L.halo_velrho4);
    c->halo_idt = (uint32_t *)(w + L.halo_idt);
    c->migrants = (uint4 *)(w + L.migrants);
    c->mig_total = (uint32_t *)(w + L.mig_total);
    c->mig_count = (uint32_t *)(w + L.mig_count);
    c->prev_init = (uint8_t *)(w + L.prev_init);
    c->flags = (uint32_t *)(w + L.flags);
    c->interact_variant = 0;
    c->zblock_mma = mma_zblock(p);
    c->ia_tiles = (uint32_t *)(w + L.ia_tiles);

    c->last_cuda_error[0] = 0;
    c->id_order = true;
    c->sort_had_prev = false;
    // kernel attributes are per device: set them for the device this context lives on
    cudaError_t e = configure_interact();
    if (e == cudaSuccess) e = configure_sort();
    int dev = 0;
    c->num_sms = NUM_SMS;
    if (e == cudaSuccess) e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess && c->num_sms < 1) c->num_sms = NUM_SMS;
    if (e == cudaSuccess) e = configure_keys(c);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->acc4, 0, 16 * (c->n ? c->n : 1), c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->mig_total, 0, 4, c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->mig_count, 0, 4 * 2 * SPH_MAX_SLABS, c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->halo_offset, 0, 4 * (2 * SPH_MAX_SLABS + 1), c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->slab_begin, 0, 4 * (SPH_MAX_SLABS + 1), c->stream);
    if (e != cudaSuccess) { int rc = cuda_fail(c, e); delete c; return rc; }
    int rc = upload_state(c, part);
    if (rc != SPH_OK) { delete c; return rc; }
    *out = c;
    return SPH_OK;
}

int sph_set_state(sph_ctx *c, const sph_particles *part)
{
    if (!c) return SPH_ERR_ARG;
    if (c->sticky) return c->sticky;
    return upload_state(c, part);
}

int sph_set_slabs(sph_ctx *c, const int32_t *planes, int n_slabs)
{
    if (!c) return SPH_ERR_ARG;
    if (!planes_ok(planes, n_slabs, c->grid.nc[0], c->max_slabs)) return SPH_ERR_SLABS;
    c->slabs.n_slabs = n_slabs;
    for (int s = 0; s <= SPH_MAX_SLABS; ++s) c->slabs.planes[s] = s <= n_slabs ? planes[s] : 0;
    return SPH_OK;
}

int sph_slab_planes_from_x(const sph_ctx *c, const float *x_bounds, int n_slabs, int32_t *planes_out)
{
    if (!c || !x_bounds || !planes_out || n_slabs < 1 || n_slabs > c->max_slabs) return SPH_ERR_ARG;
    const int ncx = c->grid.nc[0];
    planes_out[0] = 0;
    planes_out[n_slabs] = ncx;
    for (int s = 1; s < n_slabs; ++s) {
        double t = ((double)x_bounds[s] - (double)c->grid.min[0]) / (2.0 * (double)c->P.h);
        int pl = (int)floor(t + 0.5);
        int lo = planes_out[s - 1] + 2, hi = ncx - 2 * (n_slabs - s);
        if (pl < lo) pl = lo;
        if (pl > hi) pl = hi;
        planes_out[s] = pl;
    }
    return planes_ok(planes_out, n_slabs, ncx, c->max_slabs) ? SPH_OK : SPH_ERR_SLABS;
}

int sph_sort_and_cells(sph_ctx *c)
{
    if (!c) return SPH_ERR_ARG;
    if (c->sticky) return c->sticky;
    c->sort_had_prev = c->have_prev_init || c->have_prev_ranges;
    {
        Timed t(c, SPH_T_KEYS);
        CK(c, launch_keys(c));
    }
    {
        Timed t(c, SPH_T_SORT);
        CK(c, launch_sort(c));
    }
    {
        Timed t(c, SPH_T_GATHER);
        CK(c, launch_gather_cells(c));
    }
    {
        Timed t(c, SPH_T_CELLS);
        CK(c, launch_cell_fill(c));
        c->tagged_slabs = c->slabs;
        CK(c, launch_slab_meta(c));
    }
    c->have_prev_init = false;
    c->have_prev_ranges = true;
    c->id_order = false;
    c->sorted_valid = true;
    c->halos_valid = false;
    c->rates_valid = false;
    c->mu_valid = false;
    return SPH_OK;
}

int sph_build_halos(sph_ctx *c, const int32_t *planes, int n_slabs)
{
    if (!c) return SPH_ERR_ARG;
    if (c->sticky) return c->sticky;
    if (!c->sorted_valid) return SPH_ERR_ORDER;
    if (planes) {
        int rc = sph_set_slabs(c, planes, n_slabs);
        if (rc != SPH_OK) return rc;
    }
    {
        Timed t(c, SPH_T_HALO);
        if (!same_slabs(c->slabs, c->tagged_slabs)) {
            // new planes without a new sort: owners, edge and migration labels, slab and halo ranges
            c->tagged_slabs = c->slabs;
            CK(c, launch_retag(c, c->sort_had_prev));
            CK(c, launch_slab_meta(c));
        }                                   // else: the ranges the sort left are current
        CK(c, launch_halo_gather(c));
    }
    {
        Timed t(c, SPH_T_MIGRATE);
        CK(c, launch_migrants(c));
    }
    c->halos_valid = true;
    return SPH_OK;
}

int sph_interact(sph_ctx *c)
{
    if (!c) return SPH_ERR_ARG;
    if (c->sticky) return c->sticky;
    if (!c->sorted_valid) return SPH_ERR_ORDER;
    Timed t(c, SPH_T_INTERACT);
    CK(c, launch_interact(c, c->adaptive_dt != 0));
    c->rates_valid = true;
    c->mu_valid = c->adaptive_dt != 0;
    return SPH_OK;
}

static int verlet_and_advance(sph_ctx *c, float dt)
{
    {
        Timed t(c, SPH_T_VERLET);
        int ns = c->P.verlet_ns;
        int corrective = ns <= 0 ? (c->step_index == 0) : (c->step_index % (uint64_t)ns == 0);
        CK(c, launch_verlet(c, dt, corrective));
    }
    c->step_index++;
    c->sorted_valid = false;      // positions moved: the cell table no longer matches them
    c->halos_valid = false;
    c->rates_valid = false;
    c->mu_valid = false;
    return SPH_OK;
}

int sph_step(sph_ctx *c, float dt)
{
    if (!c) return SPH_ERR_ARG;
    if (!(dt > 0.f) || !isfinite(dt)) return SPH_ERR_ARG;
    int rc = sph_sort_and_cells(c);
    if (rc != SPH_OK) return rc;
    rc = sph_build_halos(c, nullptr, 0);
    if (rc != SPH_OK) return rc;
    rc = sph_interact(c);
    if (rc != SPH_OK) return rc;
    return verlet_and_advance(c, dt);
}

int sph_interact_slab(sph_ctx *c, int slab)
{
    if (!c) return SPH_ERR_ARG;
    if (c->sticky) return c->sticky;
    if (!c->sorted_valid || !c->halos_valid) return SPH_ERR_ORDER;
    const int S = c->tagged_slabs.n_slabs;
    if (slab < 0 || slab >= S) return SPH_ERR_ARG;
    if (c->max_slabs < 2) return SPH_ERR_ARG;     // the local cell table exists only for max_slabs >= 2
    uint32_t h_begin[SPH_MAX_SLABS + 1], h_range[4 * SPH_MAX_SLABS], h_off[2 * SPH_MAX_SLABS + 1];
    memset(h_range, 0, sizeof(h_range));
    memset(h_off, 0, sizeof(h_off));
    CK(c, cudaMemcpyAsync(h_begin, c->slab_begin, 4 * (S + 1), cudaMemcpyDeviceToHost, c->stream));
    if (S > 1) {
        CK(c, cudaMemcpyAsync(h_range, c->halo_range, 4 * 4 * S, cudaMemcpyDeviceToHost, c->stream));
        CK(c, cudaMemcpyAsync(h_off, c->halo_offset, 4 * (2 * S + 1), cudaMemcpyDeviceToHost, c->stream));
    }
    CK(c, cudaStreamSynchronize(c->stream));
    Timed t(c, SPH_T_INTERACT);
    CK(c, launch_interact_slab(c, slab, h_begin, h_range, h_off));
    c->rates_valid = true;
    c->mu_valid = false;
    return SPH_OK;
}

int sph_time_step(sph_ctx *c, float cfl, float *dt, float *amax_slab, float *smax_slab)
{
    if (!c || !(cfl > 0.f) || !isfinite(cfl)) return SPH_ERR_ARG;
    if (c->sticky) return c->sticky;
    if (!c->sorted_valid || !c->rates_valid || !c->mu_valid) return SPH_ERR_ORDER;
    uint32_t h[2 * SPH_MAX_SLABS];
    {
        Timed t(c, SPH_T_DTREDUCE);
        CK(c, launch_dt_reduce(c));
    }
    CK(c, cudaMemcpyAsync(h, c->dt_red, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CK(c, cudaStreamSynchronize(c->stream));
    const int S = c->tagged_slabs.n_slabs;
    float amax = 0.f, smax = 0.f;
    for (int k = 0; k < S; ++k) {
        float a2, sg;
        memcpy(&a2, &h[2 * k], 4);
        memcpy(&sg, &h[2 * k + 1], 4);
        const float a = sqrtf(a2);
        if (amax_slab) amax_slab[k] = a;
        if (smax_slab) smax_slab[k] = sg;
        if (a > amax) amax = a;
        if (sg > smax) smax = sg;
    }
    if (dt) {
        const double hh = (double)c->P.h;
        const double dt_f = amax > 0.f ? sqrt(hh / (double)amax) : INFINITY;
        const double dt_cv = smax > 0.f ? hh / (double)smax : INFINITY;
        *dt = (float)((double)cfl * (dt_f < dt_cv ? dt_f : dt_cv));
    }
    return SPH_OK;
}

int sph_step_adaptive(sph_ctx *c, float cfl, float *dt_used)
{
    if (!c || !(cfl > 0.f) || !isfinite(cfl)) return SPH_ERR_ARG;
    c->adaptive_dt = 1;
    int rc = sph_sort_and_cells(c);
    if (rc != SPH_OK) return rc;
    rc = sph_build_halos(c, nullptr, 0);
    if (rc != SPH_OK) return rc;
    rc = sph_interact(c);
    if (rc != SPH_OK) return rc;
    float dt = 0.f;
    rc = sph_time_step(c, cfl, &dt, nullptr, nullptr);
    if (rc != SPH_OK) return rc;
    if (!(dt > 0.f) || !isfinite(dt)) return SPH_ERR_NONFINITE;
    if (dt_used) *dt_used = dt;
    return verlet_and_advance(c, dt);
}

int sph_get_view(sph_ctx *c, sph_view *v)
{
    if (!c || !v) return SPH_ERR_ARG;
    memset(v, 0, sizeof(*v));
    v->n = c->n;
    for (int k = 0; k < 3; ++k) v->nc[k] = c->grid.nc[k];
    v->ncells = c->grid.ncells;
    v->cell_bits = c->cell_bits;
    v->n_slabs = c->tagged_slabs.n_slabs;
    v->step_index = c->step_index;
    v->pos4 = (const float *)c->pos4[c->cur];
    v->velrho4 = (const float *)c->velrho4[c->cur];
    v->velrhoM1_4 = (const float *)c->velrhoM1[c->cur];
    v->acc4 = (const float *)c->acc4;
    v->idt = c->idt[c->cur];
    v->keyword = c->keyword;
    v->cell_begin = c->cell_begin;
    v->slab_begin = c->slab_begin;
    v->halo_offset = c->halo_offset;
    v->halo_pos4 = (const float *)c->halo_pos4;
    v->halo_velrho4 = (const float *)c->halo_velrho4;
    v->halo_idt = c->halo_idt;
    v->mig_total = c->mig_total;
    v->migrants = (const uint32_t *)c->migrants;
    v->mig_count = c->mig_count;
    v->mumax = c->mumax;
    return SPH_OK;
}

int sph_download(sph_ctx *c, float *pos, float *vel, float *rho, float *acc, float *drho)
{
    if (!c) return SPH_ERR_ARG;
    if (c->sticky) return c->sticky;
    const uint64_t n = c->n;
    if (n == 0) return SPH_OK;
    // packed id-order staging lives in the idle half of the double buffers
    int o = 1 - c->cur;
    float *spos = (float *)c->pos4[o], *svel = (float *)c->velrho4[o];
    float *srho = (float *)c->idt[o], *sacc = (float *)c->velrhoM1[o];
    float *sdrho = (float *)c->kv[1 - c->kv_sorted];
    CK(c, launch_download_pack(c, pos ? spos : nullptr, vel ? svel : nullptr, rho ? srho : nullptr,
                               acc ? sacc : nullptr, drho ? sdrho : nullptr));
    if (pos) CK(c, cudaMemcpyAsync(pos, spos, 12 * n, cudaMemcpyDeviceToHost, c->stream));
    if (vel) CK(c, cudaMemcpyAsync(vel, svel, 12 * n, cudaMemcpyDeviceToHost, c->stream));
    if (rho) CK(c, cudaMemcpyAsync(rho, srho, 4 * n, cudaMemcpyDeviceToHost, c->stream));
    if (acc) CK(c, cudaMemcpyAsync(acc, sacc, 12 * n, cudaMemcpyDeviceToHost, c->stream));
    if (drho) CK(c, cudaMemcpyAsync(drho, sdrho, 4 * n, cudaMemcpyDeviceToHost, c->stream));
    CK(c, cudaStreamSynchronize(c->stream));
    return SPH_OK;
}

int sph_status(sph_ctx *c)
{
    if (!c) return SPH_ERR_ARG;
    if (c->sticky) return c->sticky;
    uint32_t f = 0;
    CK(c, cudaMemcpyAsync(&f, c->flags, 4, cudaMemcpyDeviceToHost, c->stream));
    CK(c, cudaStreamSynchronize(c->stream));
    if (f & FLAG_NONFINITE) return SPH_ERR_NONFINITE;
    return SPH_OK;
}

int sph_set_option(sph_ctx *c, int option, int value)
{
    if (!c) return SPH_ERR_ARG;
    switch (option) {
    case SPH_OPT_INTERACT_VARIANT:
        if (value < 0 || value > 1) return SPH_ERR_ARG;
        c->interact_variant = value;
        return SPH_OK;
    case SPH_OPT_ADAPTIVE_DT:
        if (value != 0 && value != 1) return SPH_ERR_ARG;
        c->adaptive_dt = value;
        return SPH_OK;
    default:
        return SPH_ERR_ARG;
    }
}

int sph_profile_enable(sph_ctx *c, int enable)
{
    if (!c) return SPH_ERR_ARG;
    c->timer.enabled = enable != 0;
    return SPH_OK;
}

int sph_profile_read(sph_ctx *c, float *ms, int *launches)
{
    if (!c) return SPH_ERR_ARG;
    CK(c, cudaStreamSynchronize(c->stream));
    StageTimer &t = c->timer;
    for (int k = 0; k < t.n_pairs; ++k) {
        float e = 0.f;
        if (cudaEventElapsedTime(&e, t.ev[2 * k], t.ev[2 * k + 1]) == cudaSuccess) {
            if (ms) ms[t.stage[k]] += e;
            if (launches) launches[t.stage[k]] += 1;
        }
    }
    t.n_pairs = 0;
    return SPH_OK;
}

int sph_pair_stats(sph_ctx *c, uint64_t *out)
{
    if (!c || !out) return SPH_ERR_ARG;
    if (c->sticky) return c->sticky;
    if (!c->sorted_valid) return SPH_ERR_ORDER;
    unsigned long long *d = c->scratch64;
    CK(c, launch_pair_stats(c, d));
    unsigned long long h[2] = {0, 0};
    CK(c, cudaMemcpyAsync(h, d, 16, cudaMemcpyDeviceToHost, c->stream));
    CK(c, cudaStreamSynchronize(c->stream));
    out[0] = h[0];
    out[1] = h[1];
    return SPH_OK;
}

int sph_download_resume(sph_ctx *c, float *vel_m1, float *rho_m1, uint64_t *step_index)
{
    if (!c) return SPH_ERR_ARG;
    if (c->sticky) return c->sticky;
    const uint64_t n = c->n;
    if (step_index) *step_index = c->step_index;
    if (n == 0 || (!vel_m1 && !rho_m1)) return SPH_OK;
    int o = 1 - c->cur;                                   // idle halves as packed id-order staging
    float *svel = (float *)c->velrho4[o], *srho = (float *)c->idt[o];
    CK(c, launch_m1_pack(c, vel_m1 ? svel : nullptr, rho_m1 ? srho : nullptr));
    if (vel_m1) CK(c, cudaMemcpyAsync(vel_m1, svel, 12 * n, cudaMemcpyDeviceToHost, c->stream));
    if (rho_m1) CK(c, cudaMemcpyAsync(rho_m1, srho, 4 * n, cudaMemcpyDeviceToHost, c->stream));
    CK(c, cudaStreamSynchronize(c->stream));
    return SPH_OK;
}

int sph_set_resume(sph_ctx *c, const float *vel_m1, const float *rho_m1, uint64_t step_index, int on_device)
{
    if (!c || !vel_m1 || !rho_m1) return SPH_ERR_ARG;
    if (c->sticky) return c->sticky;
    if (!c->id_order) return SPH_ERR_ORDER;               // only right after sph_init / sph_set_state
    const uint64_t n = c->n;
    const float *dvel = vel_m1, *drho = rho_m1;
    if (n && !on_device) {
        float *svel = (float *)c->velrho4[1 - c->cur], *srho = (float *)c->idt[1 - c->cur];
        CK(c, cudaMemcpyAsync(svel, vel_m1, 12 * n, cudaMemcpyHostToDevice, c->stream));
        CK(c, cudaMemcpyAsync(srho, rho_m1, 4 * n, cudaMemcpyHostToDevice, c->stream));
        dvel = svel; drho = srho;
    }
    CK(c, launch_m1_unpack(c, dvel, drho));
    if (!on_device) CK(c, cudaStreamSynchronize(c->stream));
    c->step_index = step_index;
    return SPH_OK;
}

int sph_balance_slabs(sph_ctx *c, int n_slabs, int32_t *planes_out)
{
    if (!c || !planes_out || n_slabs < 1 || n_slabs > c->max_slabs) return SPH_ERR_ARG;
    if (c->sticky) return c->sticky;
    if (!c->sorted_valid) return SPH_ERR_ORDER;
    if (c->grid.nc[0] < 2 * n_slabs && n_slabs > 1) return SPH_ERR_SLABS;
    int32_t *d_planes = (int32_t *)c->dt_red;             // 32 words of scratch, dead outside sph_time_step
    CK(c, launch_balance(c, n_slabs, d_planes));
    CK(c, cudaMemcpyAsync(planes_out, d_planes, 4 * (n_slabs + 1), cudaMemcpyDeviceToHost, c->stream));
    CK(c, cudaStreamSynchronize(c->stream));
    return planes_ok(planes_out, n_slabs, c->grid.nc[0], c->max_slabs) ? SPH_OK : SPH_ERR_SLABS;
}

int sph_fma_peak(sph_ctx *c, int variant, int iters, double *tflops)
{
    if (!c || !tflops || iters < 1 || (variant != 0 && variant != 1)) return SPH_ERR_ARG;
    if (c->sticky) return c->sticky;
    const int blocks = c->num_sms * 8;
    cudaEvent_t e0, e1;
    CK(c, cudaEventCreate(&e0));
    {
        cudaError_t ec = cudaEventCreate(&e1);
        if (ec != cudaSuccess) { cudaEventDestroy(e0); return cuda_fail(c, ec); }
    }
    float *sink = (float *)c->scratch64;
    int rc = SPH_OK;
    cudaError_t e = launch_fma_peak(c, variant, iters / 8 + 1, blocks, sink);      // warm-up
    if (e == cudaSuccess) e = cudaEventRecord(e0, c->stream);
    if (e == cudaSuccess) e = launch_fma_peak(c, variant, iters, blocks, sink);
    if (e == cudaSuccess) e = cudaEventRecord(e1, c->stream);
    if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    if (e != cudaSuccess) rc = cuda_fail(c, e);
    else *tflops = 2.0 * 8.0 * 8.0 * (double)iters * 256.0 * (double)blocks / ((double)ms * 1e-3) / 1e12;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return rc;
}

const char *sph_last_cuda_error(const sph_ctx *c)
{
    return c ? c->last_cuda_error : g_last_cuda_error;
}

int sph_launch_count(const sph_ctx *c, uint64_t *out)
{
    if (!c || !out) return SPH_ERR_ARG;
    *out = c->n_launches;
    return SPH_OK;
}

void sph_destroy(sph_ctx *c)
{
    if (!c) return;
    for (int k = 0; k < c->timer.n_created; ++k) cudaEventDestroy(c->timer.ev[k]);
    delete c;
}

const char *sph_strerror(int code)
{
    switch (code) {
    case SPH_OK: return "ok";
    case SPH_ERR_ARG: return "bad argument";
    case SPH_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
    case SPH_ERR_GRID_TOO_LARGE: return "grid has more than 2^28 cells or n > 2^28";
    case SPH_ERR_SLABS: return "bad slab planes";
    case SPH_ERR_CUDA: return "CUDA runtime error";
    case SPH_ERR_NONFINITE: return "non-finite particle state on the device";
    case SPH_ERR_ORDER: return "call order violated (sort first)";
    case SPH_ERR_STATIC_LIMIT: return "size beyond the built-in scratch of sph_cell_table_static";
    default: return "unknown error";
    }
}

}  // extern "C"
