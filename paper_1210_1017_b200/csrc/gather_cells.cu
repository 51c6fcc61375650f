// a3 + a4 - apply the sort permutation to the state arrays and build the cell table
// ("all arrays containing data information (position, velocity, etc.) are
// ordered according to the newly ordered ID array.  Last, an extra array is generated with the
// index of the first particle of each cell"; L276 "first and last particle in a given region").
//
// gather_kernel: one thread per sorted slot j; reads the sorted (keyword, source) pair, gathers
// pos4 / velrho4 / velrhoM1 / idt from the previous order (the source index is close to j in a
// running simulation, so the gather is L2-friendly), writes them contiguously and writes the
// sorted keyword array.  The cell table is written by the same threads: where a run of cell c
// starts at slot j, every cell in (previous cell, c] gets cell_begin = j (lower_bound semantics
// for empty cells, reading A11).  Gaps of up to GAP_INLINE cells are filled by the
// thread itself; longer ones (the empty part of the tank) go on a work list that
// gap_fill_kernel fills one CTA per chunk.  No memset and no scan over the table: every entry is
// written exactly once.  The kernel also counts the migrants of its 256 slots (a6).
// HBM-bound: 8 + 52 B read, 56 B written per particle; 4 B written per cell.
#include "sph_internal.cuh"

namespace sph {

__global__ void __launch_bounds__(GATHER_THREADS)
gather_kernel(uint32_t n, uint32_t ncells, const uint2 *__restrict__ kv,
              const float4 *__restrict__ pos_in, const float4 *__restrict__ vr_in,
              const float4 *__restrict__ vm_in, const uint32_t *__restrict__ idt_in,
              float4 *__restrict__ pos_out, float4 *__restrict__ vr_out, float4 *__restrict__ vm_out,
              uint32_t *__restrict__ idt_out, uint32_t *__restrict__ keyword,
              uint32_t *__restrict__ cell_begin, uint4 *__restrict__ gap_list, uint32_t *__restrict__ gap_count,
              uint32_t *__restrict__ mig_tile, uint32_t *__restrict__ mig_grp)
{
    const uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
    bool migrant = false;
    if (j < n) {
        const uint2 e = __ldcs(kv + j);
        const uint32_t src = e.y & 0x0FFFFFFFu;
        const uint32_t cell = e.x & CELL_MASK;
        const float4 p = pos_in[src];
        const float4 v = vr_in[src];
        const float4 m = vm_in[src];
        const uint32_t w = idt_in[src];
        __stcs(pos_out + j, p);       // streamed: re-read by later kernels but not by this one
        __stcs(vr_out + j, v);
        __stcs(vm_out + j, m);
        idt_out[j] = w;
        keyword[j] = e.x;
        migrant = (e.x >> 30) != 0;
        if (j == 0) {
            fill_cells(0u, cell, 0u, cell_begin, gap_list, gap_count);
        } else {
            const uint32_t prev_cell = kv[j - 1].x & CELL_MASK;
            if (cell != prev_cell) fill_cells(prev_cell + 1u, cell, j, cell_begin, gap_list, gap_count);
        }
        if (j == n - 1) fill_cells(cell + 1u, ncells, n, cell_begin, gap_list, gap_count);   // incl. the sentinel
    }
    const int cnt = __syncthreads_count(migrant);
    if (threadIdx.x == 0) {
        mig_tile[blockIdx.x] = (uint32_t)cnt;
        if (cnt) atomicAdd(&mig_grp[blockIdx.x / MG_SUB], (uint32_t)cnt);     // group of MG_SUB tiles
    }
}

// One CTA per work-list entry (grid-stride): cell_begin[lo..hi] = value.
__global__ void __launch_bounds__(256)
gap_fill_kernel(const uint4 *__restrict__ gap_list, const uint32_t *__restrict__ gap_count,
                uint32_t *__restrict__ cell_begin)
{
    const uint32_t count = *gap_count;
    for (uint32_t e = blockIdx.x; e < count; e += gridDim.x) {
        const uint4 g = gap_list[e];
        for (uint32_t cc = g.x + threadIdx.x; cc <= g.y; cc += blockDim.x) cell_begin[cc] = g.z;
    }
}

uint32_t mig_groups(uint64_t n) { return (gather_tiles(n) + MG_SUB - 1) / MG_SUB; }
uint32_t gather_tiles(uint64_t n) { return (uint32_t)((n + GATHER_THREADS - 1) / GATHER_THREADS); }
size_t gap_list_entries(uint64_t ncells) { return (size_t)(ncells / GAP_INLINE + ncells / GAP_CHUNK + 8); }

cudaError_t launch_gather_cells(sph_ctx *c)
{
    uint32_t n = (uint32_t)c->n;
    uint32_t *gap_count = c->counters + 8;
    cudaError_t e = cudaMemsetAsync(gap_count, 0, sizeof(uint32_t), c->stream);
    if (e != cudaSuccess) return e;
    if (n) {
        e = cudaMemsetAsync(c->mig_grp, 0, sizeof(uint32_t) * ((size_t)mig_groups(n) + 1), c->stream);
        if (e != cudaSuccess) return e;
        int o = 1 - c->cur;
        gather_kernel<<<gather_tiles(n), GATHER_THREADS, 0, c->stream>>>(
            n, c->grid.ncells, c->kv[c->kv_sorted], c->pos4[c->cur], c->velrho4[c->cur], c->velrhoM1[c->cur],
            c->idt[c->cur], c->pos4[o], c->velrho4[o], c->velrhoM1[o], c->idt[o], c->keyword, c->cell_begin,
            c->gap_list, gap_count, c->mig_tile, c->mig_grp);
        c->n_launches++;
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        c->cur = o;
    } else {
        // no particles: every entry, sentinel included, is 0
        e = cudaMemsetAsync(c->cell_begin, 0, sizeof(uint32_t) * ((size_t)c->grid.ncells + 1), c->stream);
    }
    return e;
}

// long gaps of the cell table (work list written by gather_kernel)
cudaError_t launch_gap_fill(sph_ctx *c, uint32_t *table)
{
    gap_fill_kernel<<<c->num_sms * 4, 256, 0, c->stream>>>(c->gap_list, c->counters + 8, table);
    c->n_launches++;
    return cudaGetLastError();
}

cudaError_t launch_cell_fill(sph_ctx *c)
{
    if (c->n == 0) return cudaSuccess;
    return launch_gap_fill(c, c->cell_begin);
}

// ---- slab ranges, halo ranges and offsets -------------------------------------------------------
// slab_begin[s] = cell_begin[planes[s]*nyz]; halo 2s = cell plane planes[s]-1 (s > 0),
// halo 2s+1 = cell plane planes[s+1] (s < S-1): each ONE contiguous sorted range (x-major keys).
__global__ void slab_meta_kernel(const uint32_t *__restrict__ cell_begin, SlabC sl, int nyz,
                                 uint32_t *__restrict__ slab_begin, uint32_t *__restrict__ halo_range,
                                 uint32_t *__restrict__ halo_offset, uint32_t *__restrict__ mig_total,
                                 uint32_t *__restrict__ mig_count)
{
    int t = threadIdx.x;
    __shared__ uint32_t cnt[2 * SPH_MAX_SLABS];
    if (t <= sl.n_slabs) slab_begin[t] = cell_begin[(size_t)sl.planes[t] * nyz];
    if (t < 2 * sl.n_slabs) {
        int s = t >> 1, side = t & 1;
        uint32_t b = 0, e = 0;
        if (side == 0 && s > 0) {
            b = cell_begin[(size_t)(sl.planes[s] - 1) * nyz];
            e = cell_begin[(size_t)sl.planes[s] * nyz];
        } else if (side == 1 && s < sl.n_slabs - 1) {
            b = cell_begin[(size_t)sl.planes[s + 1] * nyz];
            e = cell_begin[(size_t)(sl.planes[s + 1] + 1) * nyz];
        }
        halo_range[2 * t] = b;
        halo_range[2 * t + 1] = e - b;
        cnt[t] = e - b;
        mig_count[t] = 0;
    }
    if (t == 0) *mig_total = 0;
    __syncthreads();
    if (t == 0) {
        uint32_t acc = 0;
        for (int k = 0; k < 2 * sl.n_slabs; ++k) { halo_offset[k] = acc; acc += cnt[k]; }
        halo_offset[2 * sl.n_slabs] = acc;
    }
}

cudaError_t launch_slab_meta(sph_ctx *c)
{
    slab_meta_kernel<<<1, 64, 0, c->stream>>>(c->cell_begin, c->tagged_slabs, c->grid.nyz, c->slab_begin,
                                              c->halo_range, c->halo_offset, c->mig_total, c->mig_count);
    c->n_launches++;
    return cudaGetLastError();
}

// ---- edge and migration labels for new planes without re-sorting ----------------------------------
// Re-planing (sph_build_halos with planes that differ from the ones the sort tagged with; the
// load-balancing step of SURVEY 8(f) NEXT-4): owner, edge label (L240) and migration
// label (L264) of every particle are recomputed from its cell and the NEW planes; the previous owner
// is the one the sort recorded next to the pair (kv.y >> 28).  A particle whose owner changes only
// because a plane moved is a migrant like any other (reading A15).  The migrant counts per tile and
// per group that the compaction needs are rebuilt in the same pass (tile = GATHER_THREADS slots, as
// in gather_kernel).
__global__ void __launch_bounds__(GATHER_THREADS)
retag_kernel(uint32_t n, uint32_t *__restrict__ keyword, const uint2 *__restrict__ kv, SlabC sl, int nyz,
             int have_prev, uint32_t *__restrict__ mig_tile, uint32_t *__restrict__ mig_grp)
{
    const uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
    bool migrant = false;
    if (j < n) {
        const uint32_t w = keyword[j];
        const int cx = (int)((w & CELL_MASK) / (uint32_t)nyz);
        int slab = 0;
#pragma unroll
        for (int k = 1; k < SPH_MAX_SLABS; ++k) slab += (k < sl.n_slabs && cx >= sl.planes[k]) ? 1 : 0;
        uint32_t lab = 0;
        if (slab > 0 && cx == sl.planes[slab]) lab = 1;
        if (slab < sl.n_slabs - 1 && cx == sl.planes[slab + 1] - 1) lab = 2;
        uint32_t mig = 0;
        if (have_prev) {
            const int prev = (int)(kv[j].y >> 28);
            mig = slab < prev ? 1u : (slab > prev ? 2u : 0u);
        }
        migrant = mig != 0;
        keyword[j] = (w & CELL_MASK) | ((lab | (mig << 2)) << TAG_SHIFT);
    }
    const int cnt = __syncthreads_count(migrant);
    if (threadIdx.x == 0) {
        mig_tile[blockIdx.x] = (uint32_t)cnt;
        if (cnt) atomicAdd(&mig_grp[blockIdx.x / MG_SUB], (uint32_t)cnt);
    }
}

// have_prev: the last sort had previous owners (else nothing migrates: first sort, reading A15)
cudaError_t launch_retag(sph_ctx *c, bool have_prev)
{
    uint32_t n = (uint32_t)c->n;
    if (n == 0) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(c->mig_grp, 0, sizeof(uint32_t) * ((size_t)mig_groups(n) + 1), c->stream);
    if (e != cudaSuccess) return e;
    retag_kernel<<<gather_tiles(n), GATHER_THREADS, 0, c->stream>>>(n, c->keyword, c->kv[c->kv_sorted], c->tagged_slabs,
                                                                   c->grid.nyz, have_prev ? 1 : 0, c->mig_tile, c->mig_grp);
    c->n_launches++;
    return cudaGetLastError();
}

}  // namespace sph
