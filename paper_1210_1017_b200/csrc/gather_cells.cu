// a3 + a4 - apply the sort permutation to the state arrays and build the cell table
// ("all arrays containing data information (position, velocity, etc.) are
// ordered according to the newly ordered ID array.  Last, an extra array is generated with the
// index of the first particle of each cell"; L276 "first and last particle in a given region").
//
// gather_kernel: one thread per sorted slot j; reads the sorted (keyword, source) pair, gathers
// pos4 / velrho4 / velrhoM1 / idt from the previous order (the source index is close to j in a
// running simulation, so the gather is L2-friendly), writes them contiguously, writes the
// sorted keyword array and marks cell_begin[c] = j where a run of cell c starts.
// cell_fill_kernel: one chained suffix-min scan (decoupled look-back) gives every empty cell
// the begin of the next non-empty one, i.e. lower_bound semantics for all cells.
// HBM-bound: 8 + 52 B read, 56 B written per particle; 8 B per cell.
#include "sph_internal.cuh"

namespace sph {

__global__ void __launch_bounds__(256)
gather_kernel(uint32_t n, const uint2 *__restrict__ kv,
              const float4 *__restrict__ pos_in, const float4 *__restrict__ vr_in,
              const float4 *__restrict__ vm_in, const uint32_t *__restrict__ idt_in,
              float4 *__restrict__ pos_out, float4 *__restrict__ vr_out, float4 *__restrict__ vm_out,
              uint32_t *__restrict__ idt_out, uint32_t *__restrict__ keyword,
              uint32_t *__restrict__ cell_begin)
{
    uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    uint2 e = __ldcs(kv + j);
    uint32_t src = e.y & 0x0FFFFFFFu;
    uint32_t cell = e.x & CELL_MASK;
    uint32_t prev_cell = j ? (kv[j - 1].x & CELL_MASK) : 0xFFFFFFFFu;
    float4 p = pos_in[src];
    float4 v = vr_in[src];
    float4 m = vm_in[src];
    uint32_t w = idt_in[src];
    __stcs(pos_out + j, p);       // streamed: re-read by later kernels but not by this one
    __stcs(vr_out + j, v);
    __stcs(vm_out + j, m);
    idt_out[j] = w;
    keyword[j] = e.x;
    if (cell != prev_cell) cell_begin[cell] = j;
}

cudaError_t launch_gather_cells(sph_ctx *c)
{
    uint32_t n = (uint32_t)c->n;
    // unset cells = 0xFFFFFFFF; sentinel cell_begin[ncells] = n
    cudaError_t e = cudaMemsetAsync(c->cell_begin, 0xFF, sizeof(uint32_t) * ((size_t)c->grid.ncells + 1), c->stream);
    if (e != cudaSuccess) return e;
    if (n) {
        int o = 1 - c->cur;
        gather_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(
            n, c->kv[c->kv_sorted], c->pos4[c->cur], c->velrho4[c->cur], c->velrhoM1[c->cur], c->idt[c->cur],
            c->pos4[o], c->velrho4[o], c->velrhoM1[o], c->idt[o], c->keyword, c->cell_begin);
        c->n_launches++;
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        c->cur = o;
    }
    return cudaSuccess;
}

// ---- suffix-min scan over cell_begin[0..ncells] -----------------------------------------------
constexpr int CF_THREADS = 256;
constexpr int CF_IPT = 16;
constexpr int CF_TILE = CF_THREADS * CF_IPT;
uint32_t scan_tiles(uint64_t n) { return (uint32_t)((n + CF_TILE - 1) / CF_TILE); }

// Tiles are numbered from the END of the array (tile 0 holds the last elements), so that the
// suffix scan is a forward chained scan over tiles.  state word: flag<<32 | value.
__global__ void __launch_bounds__(CF_THREADS)
cell_fill_kernel(uint32_t m /* ncells+1 */, uint32_t n, uint32_t *__restrict__ cell_begin,
                 unsigned long long *state, uint32_t *ticket)
{
    __shared__ uint32_t s_tile, s_warp_min[CF_THREADS / 32], s_carry;
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    // element index of reversed position q: idx = m-1-q ; thread handles CF_IPT consecutive q
    const uint32_t q0 = tile * CF_TILE + tid * CF_IPT;
    uint32_t v[CF_IPT];
#pragma unroll
    for (int k = 0; k < CF_IPT; ++k) {
        uint32_t q = q0 + k;
        v[k] = 0xFFFFFFFFu;
        if (q < m) v[k] = (q == 0) ? n : cell_begin[m - 1 - q];
    }
    // inclusive running min in reversed order inside the thread
#pragma unroll
    for (int k = 1; k < CF_IPT; ++k) v[k] = min(v[k], v[k - 1]);
    uint32_t tmin = v[CF_IPT - 1];
    // exclusive scan (min) over threads
    uint32_t inc = tmin;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= (uint32_t)o) inc = min(inc, t);
    }
    uint32_t exc = __shfl_up_sync(0xffffffffu, inc, 1);
    if (lane == 0) exc = 0xFFFFFFFFu;
    if (lane == 31) s_warp_min[warp] = inc;
    __syncthreads();
    uint32_t wpre = 0xFFFFFFFFu, block_min = 0xFFFFFFFFu;
#pragma unroll
    for (int w = 0; w < CF_THREADS / 32; ++w) {
        uint32_t t = s_warp_min[w];
        if (w < (int)warp) wpre = min(wpre, t);
        block_min = min(block_min, t);
    }
    exc = min(exc, wpre);
    // chained look-back over earlier tiles (= later cells), warp 0, 32 tiles per round trip
    if (warp == 0) {
        if (lane == 0) st_relaxed_u64(state + tile, ((tile == 0 ? 2ull : 1ull) << 32) | block_min);
        uint32_t carry = 0xFFFFFFFFu;
        if (tile > 0) {
            carry = warp_lookback(state, tile, 0xFFFFFFFFu, [](uint32_t a, uint32_t b) { return min(a, b); });
            if (lane == 0) st_relaxed_u64(state + tile, (2ull << 32) | min(carry, block_min));
        }
        if (lane == 0) s_carry = carry;
    }
    __syncthreads();
    exc = min(exc, s_carry);
#pragma unroll
    for (int k = 0; k < CF_IPT; ++k) {
        uint32_t q = q0 + k;
        if (q < m) cell_begin[m - 1 - q] = min(v[k], exc);
    }
}

cudaError_t launch_cell_fill(sph_ctx *c)
{
    uint32_t m = c->grid.ncells + 1;
    uint32_t tiles = scan_tiles(m);
    cudaError_t e = cudaMemsetAsync(c->scan_state, 0, sizeof(unsigned long long) * tiles, c->stream);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(c->counters + 8, 0, sizeof(uint32_t), c->stream);
    if (e != cudaSuccess) return e;
    cell_fill_kernel<<<tiles, CF_THREADS, 0, c->stream>>>(m, (uint32_t)c->n, c->cell_begin, c->scan_state,
                                                        c->counters + 8);
    c->n_launches++;
    return cudaGetLastError();
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

// ---- edge labels for new planes without re-sorting ---------------------------------------------
__global__ void retag_kernel(uint32_t n, uint32_t *__restrict__ keyword, SlabC sl, int nyz)
{
    uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    uint32_t w = keyword[j];
    int cx = (int)((w & CELL_MASK) / (uint32_t)nyz);
    int slab = 0;
#pragma unroll
    for (int k = 1; k < SPH_MAX_SLABS; ++k) slab += (k < sl.n_slabs && cx >= sl.planes[k]) ? 1 : 0;
    uint32_t lab = 0;
    if (slab > 0 && cx == sl.planes[slab]) lab = 1;
    if (slab < sl.n_slabs - 1 && cx == sl.planes[slab + 1] - 1) lab = 2;
    keyword[j] = (w & ~(3u << TAG_SHIFT)) | (lab << TAG_SHIFT);
}

cudaError_t launch_retag(sph_ctx *c)
{
    uint32_t n = (uint32_t)c->n;
    if (n == 0) return cudaSuccess;
    retag_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(n, c->keyword, c->tagged_slabs, c->grid.nyz);
    c->n_launches++;
    return cudaGetLastError();
}

}  // namespace sph
