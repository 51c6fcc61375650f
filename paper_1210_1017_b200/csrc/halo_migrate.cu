// a5 + a6 - halo building and particle migration driven by the sorted keys
// ("Data from the edge (the portion of the sub-domain within a distance 2h to
// the sub-domain boundary) of domain n is used to construct the halo of the neighbouring domain
// n+1, and vice versa"; L198-219 the per-step migrate / edge steps; L240-264 packing by sort).
//
// The paper packs edges and migrants with two extra radix sorts and ships them through
// cudaMemcpy + MPI.  Here sub-domains are logical x-slabs of one device's arrays: with
// x-major cell keys an edge is ONE contiguous sorted range (a cell plane), so the halo of a
// slab is a bulk copy into its halo buffer, and migrants are a stream compaction of the
// migration label that the key kernel put in the keyword.
// HBM-bound: 72 B per halo particle; 4 B per particle + 16 B per migrant.
#include "sph_internal.cuh"

namespace sph {

__global__ void __launch_bounds__(256)
halo_gather_kernel(const uint32_t *__restrict__ halo_range, const uint32_t *__restrict__ halo_offset,
                   const float4 *__restrict__ pos4, const float4 *__restrict__ velrho4,
                   const uint32_t *__restrict__ idt, float4 *__restrict__ hpos, float4 *__restrict__ hvr,
                   uint32_t *__restrict__ hid)
{
    const uint32_t h = blockIdx.y;
    const uint32_t begin = halo_range[2 * h], count = halo_range[2 * h + 1];
    const uint32_t off = halo_offset[h];
    for (uint32_t k = blockIdx.x * blockDim.x + threadIdx.x; k < count; k += gridDim.x * blockDim.x) {
        hpos[off + k] = __ldg(pos4 + begin + k);
        hvr[off + k] = __ldg(velrho4 + begin + k);
        hid[off + k] = __ldg(idt + begin + k);
    }
}

cudaError_t launch_halo_gather(sph_ctx *c)
{
    int S = c->tagged_slabs.n_slabs;
    if (S <= 1 || c->n == 0) return cudaSuccess;
    // a cell plane holds about n/ncx particles; the grid-stride loop covers any count
    uint64_t per_plane = c->n / (uint64_t)c->grid.nc[0] + 1;
    uint32_t bx = (uint32_t)((per_plane + 1023) / 1024);
    if (bx < 1) bx = 1;
    if (bx > 2048) bx = 2048;
    dim3 grid(bx, 2 * S);
    halo_gather_kernel<<<grid, 256, 0, c->stream>>>(c->halo_range, c->halo_offset, c->pos4[c->cur],
                                                    c->velrho4[c->cur], c->idt[c->cur], c->halo_pos4,
                                                    c->halo_velrho4, c->halo_idt);
    c->n_launches++;
    return cudaGetLastError();
}

// ---- migrants: ordered stream compaction (chained scan with decoupled look-back) -----------------
constexpr int MG_THREADS = 256;
constexpr int MG_IPT = 16;
constexpr int MG_TILE = MG_THREADS * MG_IPT;

__global__ void __launch_bounds__(MG_THREADS)
migrants_kernel(uint32_t n, const uint32_t *__restrict__ keyword, const uint2 *__restrict__ kv,
                const uint32_t *__restrict__ idt, SlabC sl, int nyz, unsigned long long *state,
                uint32_t *ticket, uint4 *__restrict__ records, uint32_t *__restrict__ mig_total,
                uint32_t *__restrict__ mig_count)
{
    __shared__ uint32_t s_tile, s_warp[MG_THREADS / 32], s_carry;
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    // blocked arrangement keeps sorted order: thread owns MG_IPT consecutive slots
    const uint32_t j0 = tile * MG_TILE + tid * MG_IPT;
    uint32_t flags = 0, cnt = 0;
#pragma unroll
    for (int k = 0; k < MG_IPT; ++k) {
        uint32_t j = j0 + k;
        if (j < n && (keyword[j] >> 30) != 0) { flags |= 1u << k; ++cnt; }
    }
    uint32_t inc = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= (uint32_t)o) inc += t;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    uint32_t wpre = 0, total = 0;
#pragma unroll
    for (int w = 0; w < MG_THREADS / 32; ++w) {
        uint32_t t = s_warp[w];
        if (w < (int)warp) wpre += t;
        total += t;
    }
    if (warp == 0) {                     // look-back by warp 0, 32 tiles per round trip
        if (lane == 0) st_relaxed_u64(state + tile, ((tile == 0 ? 2ull : 1ull) << 32) | total);
        uint32_t carry = 0;
        if (tile > 0) {
            carry = warp_lookback(state, tile, 0u, [](uint32_t a, uint32_t b) { return a + b; });
            if (lane == 0) st_relaxed_u64(state + tile, (2ull << 32) | (carry + total));
        }
        if (lane == 0) {
            s_carry = carry;
            if (tile == gridDim.x - 1) *mig_total = carry + total;   // tiles are ticketed in order
        }
    }
    __syncthreads();
    uint32_t out = s_carry + wpre + inc - cnt;
    if (flags) {
#pragma unroll
        for (int k = 0; k < MG_IPT; ++k) {
            if (flags & (1u << k)) {
                uint32_t j = j0 + k;
                uint32_t w = keyword[j];
                int cx = (int)((w & CELL_MASK) / (uint32_t)nyz);
                int slab = 0;
                for (int q = 1; q < sl.n_slabs; ++q) slab += (cx >= sl.planes[q]) ? 1 : 0;
                uint32_t prev = kv[j].y >> 28;
                records[out++] = make_uint4(idt[j] & ID_MASK, j, prev, (uint32_t)slab);
                atomicAdd(&mig_count[2 * prev + ((w >> 30) == 2 ? 1 : 0)], 1u);
            }
        }
    }
}

cudaError_t launch_migrants(sph_ctx *c)
{
    uint32_t n = (uint32_t)c->n;
    if (n == 0) return cudaSuccess;
    uint32_t tiles = (n + MG_TILE - 1) / MG_TILE;
    cudaError_t e = cudaMemsetAsync(c->scan_state, 0, sizeof(unsigned long long) * tiles, c->stream);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(c->counters + 9, 0, sizeof(uint32_t), c->stream);
    if (e != cudaSuccess) return e;
    migrants_kernel<<<tiles, MG_THREADS, 0, c->stream>>>(
        n, c->keyword, c->kv[c->kv_sorted], c->idt[c->cur], c->tagged_slabs, c->grid.nyz, c->scan_state,
        c->counters + 9, c->migrants, c->mig_total, c->mig_count);
    c->n_launches++;
    return cudaGetLastError();
}

}  // namespace sph
