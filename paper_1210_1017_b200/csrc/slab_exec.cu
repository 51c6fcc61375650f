// Per-sub-domain execution of the interaction pass ("Data from the
// edge ... of domain n is used to construct the halo of the neighbouring domain n+1", L218-220: each
// GPU_k receives its halo, orders its arrays by cell, then "compute[s] particle interactions" for its
// own sub-domain, L226-228).
//
// sph_interact_slab(s) does on one device what GPU_s does in the paper: it assembles the arrays that
// GPU would hold - [halo received from s-1 | own particles | halo received from s+1], the halos taken
// from the HALO BUFFERS that a5 built, not from the global arrays -, rebuilds the cell table of that
// local set from the particles' positions, and runs the production interaction kernel on it for the
// cell planes the slab owns.  The rates land in the slab's own range of acc4.  Looping over all slabs
// must reproduce the global sph_interact result (tests/test_gpu_slabs.py) - value for value when every
// tile at a slab plane fits one candidate batch, to rounding otherwise (interact_mma.cu, DRAIN) -: that
// is the device-side proof that a halo of width 2h (one cell plane) is sufficient.
//
// Local storage: the idle halves of the double-buffered state (dead between the gather and the next
// sort) and one extra cell table.  With x-major keys the local set is a contiguous piece of the global
// sorted order, so local index = global index - base and the kernel is handed base-shifted pointers.
#include "sph_internal.cuh"

namespace sph {

// One thread per local slot q: copy the particle, recompute its cell from its position (a receiving
// GPU has nothing else for halo particles), write the local keyword, and - as the gather kernel does
// for the global table - every cell-table entry in (previous cell, own cell].
__global__ void __launch_bounds__(256)
slab_compose_kernel(uint32_t n_left, uint32_t n_own, uint32_t n_right, uint32_t base,
                    uint32_t cell_first, uint32_t cell_last /* entries [cell_first, cell_last] are written */,
                    const float4 *__restrict__ hpos_l, const float4 *__restrict__ hvr_l, const uint32_t *__restrict__ hid_l,
                    const float4 *__restrict__ pos_own, const float4 *__restrict__ vr_own, const uint32_t *__restrict__ id_own,
                    const float4 *__restrict__ hpos_r, const float4 *__restrict__ hvr_r, const uint32_t *__restrict__ hid_r,
                    float4 *__restrict__ pos_loc, float4 *__restrict__ vr_loc, uint32_t *__restrict__ id_loc,
                    uint32_t *__restrict__ kw_loc, uint32_t *__restrict__ cell_loc, uint4 *__restrict__ gap_list,
                    uint32_t *__restrict__ gap_count, GridC g)
{
    const uint32_t n_loc = n_left + n_own + n_right;
    const uint32_t q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= n_loc) return;
    auto fetch_pos = [&](uint32_t k) -> float4 {
        if (k < n_left) return hpos_l[k];
        if (k < n_left + n_own) return pos_own[k - n_left];
        return hpos_r[k - n_left - n_own];
    };
    auto cell_of = [&](const float4 &p) -> uint32_t {
        const int cx = cell_coord(p.x, g.min[0], g.inv_cell, g.nc[0]);
        const int cy = cell_coord(p.y, g.min[1], g.inv_cell, g.nc[1]);
        const int cz = cell_coord(p.z, g.min[2], g.inv_cell, g.nc[2]);
        return (uint32_t)((cx * g.nc[1] + cy) * g.nc[2] + cz);
    };
    const float4 p = fetch_pos(q);
    float4 v;
    uint32_t w;
    if (q < n_left) { v = hvr_l[q]; w = hid_l[q]; }
    else if (q < n_left + n_own) { v = vr_own[q - n_left]; w = id_own[q - n_left]; }
    else { v = hvr_r[q - n_left - n_own]; w = hid_r[q - n_left - n_own]; }
    pos_loc[q] = p;
    vr_loc[q] = v;
    id_loc[q] = w;
    const uint32_t cell = cell_of(p);
    kw_loc[q] = cell;
    if (q == 0) {
        fill_cells(cell_first, cell, base, cell_loc, gap_list, gap_count);
    } else {
        const uint32_t prev_cell = cell_of(fetch_pos(q - 1));
        if (cell != prev_cell) fill_cells(prev_cell + 1u, cell, base + q, cell_loc, gap_list, gap_count);
    }
    if (q == n_loc - 1 && cell < cell_last) fill_cells(cell + 1u, cell_last, base + n_loc, cell_loc, gap_list, gap_count);
}

// h_*: HOST copies of slab_begin (S + 1), halo_range (2 per halo: begin, count) and halo_offset.
cudaError_t launch_interact_slab(sph_ctx *c, int s, const uint32_t *h_slab_begin, const uint32_t *h_halo_range,
                                 const uint32_t *h_halo_offset)
{
    const int S = c->tagged_slabs.n_slabs;
    const uint32_t own_b = h_slab_begin[s], n_own = h_slab_begin[s + 1] - own_b;
    const uint32_t n_left = h_halo_range[2 * (2 * s) + 1], n_right = h_halo_range[2 * (2 * s + 1) + 1];
    const uint32_t off_l = h_halo_offset[2 * s], off_r = h_halo_offset[2 * s + 1];
    const uint32_t base = own_b - n_left;                     // plane P_s - 1 sits right before the slab
    const uint32_t n_loc = n_left + n_own + n_right;
    const int p_lo = s > 0 ? c->tagged_slabs.planes[s] - 1 : c->tagged_slabs.planes[s];
    const int p_hi = s < S - 1 ? c->tagged_slabs.planes[s + 1] : c->tagged_slabs.planes[s + 1] - 1;
    const uint32_t cell_first = (uint32_t)p_lo * (uint32_t)c->grid.nyz;
    const uint32_t cell_last = (uint32_t)(p_hi + 1) * (uint32_t)c->grid.nyz;      // inclusive: the end sentinel
    if (n_own == 0) return cudaSuccess;

    const int o = 1 - c->cur;                                  // idle halves of the double buffers
    float4 *pos_loc = c->pos4[o], *vr_loc = c->velrho4[o], *acc_loc = c->velrhoM1[o];
    uint32_t *id_loc = c->idt[o];
    uint32_t *kw_loc = reinterpret_cast<uint32_t *>(c->kv[1 - c->kv_sorted]);
    uint32_t *gap_count = c->counters + 8;
    cudaError_t e = cudaMemsetAsync(gap_count, 0, sizeof(uint32_t), c->stream);
    if (e != cudaSuccess) return e;
    slab_compose_kernel<<<(n_loc + 255) / 256, 256, 0, c->stream>>>(
        n_left, n_own, n_right, base, cell_first, cell_last,
        c->halo_pos4 + off_l, c->halo_velrho4 + off_l, c->halo_idt + off_l,
        c->pos4[c->cur] + own_b, c->velrho4[c->cur] + own_b, c->idt[c->cur] + own_b,
        c->halo_pos4 + off_r, c->halo_velrho4 + off_r, c->halo_idt + off_r,
        pos_loc, vr_loc, id_loc, kw_loc, c->cell_loc, c->gap_list, gap_count, c->grid);
    c->n_launches++;
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    e = launch_gap_fill(c, c->cell_loc);
    if (e != cudaSuccess) return e;

    // the production kernel on the local set: base-shifted pointers, own cell planes only
    c->ia_ov.on = true;
    c->ia_ov.pos4 = pos_loc - base;
    c->ia_ov.velrho4 = vr_loc - base;
    c->ia_ov.idt = id_loc - base;
    c->ia_ov.keyword = kw_loc - base;
    c->ia_ov.cell_begin = c->cell_loc;
    c->ia_ov.acc4 = acc_loc - base;
    c->ia_ov.cx_first = c->tagged_slabs.planes[s];
    c->ia_ov.cx_count = c->tagged_slabs.planes[s + 1] - c->tagged_slabs.planes[s];
    c->ia_ov.cand_lo = p_lo;
    c->ia_ov.cand_hi = p_hi;
    const int variant = c->interact_variant;
    c->interact_variant = 0;
    e = launch_interact(c, false);
    c->interact_variant = variant;
    c->ia_ov.on = false;
    if (e != cudaSuccess) return e;
    return cudaMemcpyAsync(c->acc4 + own_b, acc_loc + n_left, sizeof(float4) * (size_t)n_own, cudaMemcpyDeviceToDevice,
                           c->stream);
}

}  // namespace sph
