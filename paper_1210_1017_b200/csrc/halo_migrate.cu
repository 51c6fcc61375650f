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

// ---- migrants: ordered stream compaction in three steps without any inter-CTA wait ----------------
//  1. gather_kernel (gather_cells.cu) already counted the migrants of every 256-slot tile while it had
//     the sorted keywords in registers (mig_tile[t]) and of every group of MG_SUB tiles (mig_grp[g]);
//  2. mig_scan_kernel: exclusive scan of the group counts in place (one CTA; the array has n/4096
//     entries), total -> mig_total;
//  3. mig_compact_kernel: a CTA owns MG_SUB consecutive tiles, skips them when they hold no migrant
//     (in a running simulation migrants exist only next to the slab planes), otherwise re-reads the
//     keywords, ranks the flagged slots with ballots and writes the records in sorted order.
constexpr int MG_SCAN_THREADS = 1024;

__global__ void __launch_bounds__(MG_SCAN_THREADS)
mig_scan_kernel(uint32_t tiles, uint32_t *__restrict__ mig_tile /* tiles + 1 */, uint32_t *__restrict__ mig_total)
{
    __shared__ uint32_t s_warp[MG_SCAN_THREADS / 32];
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr uint32_t NW = MG_SCAN_THREADS / 32;
    // a warp owns a contiguous span; lanes read consecutive entries
    const uint32_t span = ((tiles + NW - 1) / NW + 31u) & ~31u;
    const uint32_t lo = warp * span, hi = min(tiles, lo + span);
    uint32_t sum = 0;
    for (uint32_t k = lo + lane; k < hi; k += 32) sum += mig_tile[k];
#pragma unroll
    for (int o = 16; o; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
    if (lane == 0) s_warp[warp] = sum;
    __syncthreads();
    if (warp == 0) {
        uint32_t v = s_warp[lane], inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= (uint32_t)o) inc += t;
        }
        s_warp[lane] = inc - v;
        if (lane == 31) { *mig_total = inc; mig_tile[tiles] = inc; }
    }
    __syncthreads();
    uint32_t carry = s_warp[warp];
    for (uint32_t k0 = lo; k0 < hi; k0 += 32) {
        const uint32_t k = k0 + lane;
        const uint32_t v = k < hi ? mig_tile[k] : 0u;
        uint32_t inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= (uint32_t)o) inc += t;
        }
        if (k < hi) mig_tile[k] = carry + inc - v;
        carry += __shfl_sync(0xffffffffu, inc, 31);
    }
}

__global__ void __launch_bounds__(GATHER_THREADS)
mig_compact_kernel(uint32_t n, uint32_t tiles, const uint32_t *__restrict__ mig_off,
                   const uint32_t *__restrict__ mig_tile, const uint32_t *__restrict__ keyword, const uint2 *__restrict__ kv,
                   const uint32_t *__restrict__ idt, SlabC sl, int nyz, uint4 *__restrict__ records,
                   uint32_t *__restrict__ mig_count)
{
    __shared__ uint32_t s_off[MG_SUB + 1];
    __shared__ uint32_t s_warp[GATHER_THREADS / 32];
    __shared__ uint32_t s_cnt[2 * SPH_MAX_SLABS];
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t t0 = blockIdx.x * MG_SUB;
    const uint32_t g0 = mig_off[blockIdx.x];
    if (g0 == mig_off[blockIdx.x + 1]) return;             // no migrant in these tiles (CTA-uniform)
    if (tid == 0) {
        uint32_t acc = g0;
        for (int q = 0; q < MG_SUB; ++q) {
            s_off[q] = acc;
            acc += (t0 + q < tiles) ? mig_tile[t0 + q] : 0u;
        }
        s_off[MG_SUB] = acc;
    }
    if (tid < 2 * SPH_MAX_SLABS) s_cnt[tid] = 0;
    __syncthreads();
    for (int q = 0; q < MG_SUB; ++q) {
        const uint32_t o0 = s_off[q];
        if (o0 == s_off[q + 1]) continue;                  // CTA-uniform
        const uint32_t j = (t0 + q) * GATHER_THREADS + tid;
        const uint32_t w = j < n ? __ldg(keyword + j) : 0u;
        const bool flag = (w >> 30) != 0;
        const uint32_t bal = __ballot_sync(0xffffffffu, flag);
        __syncthreads();                                   // s_warp of the previous round consumed
        if (lane == 0) s_warp[warp] = __popc(bal);
        __syncthreads();
        if (flag) {
            uint32_t out = o0 + __popc(bal & ((1u << lane) - 1u));
            for (uint32_t k = 0; k < warp; ++k) out += s_warp[k];
            const int cx = (int)((w & CELL_MASK) / (uint32_t)nyz);
            int slab = 0;
            for (int k = 1; k < sl.n_slabs; ++k) slab += (cx >= sl.planes[k]) ? 1 : 0;
            const uint32_t prev = kv[j].y >> 28;
            records[out] = make_uint4(__ldg(idt + j) & ID_MASK, j, prev, (uint32_t)slab);
            atomicAdd(&s_cnt[2 * prev + ((w >> 30) == 2 ? 1 : 0)], 1u);
        }
    }
    __syncthreads();
    if (tid < 2 * SPH_MAX_SLABS && s_cnt[tid]) atomicAdd(&mig_count[tid], s_cnt[tid]);
}

cudaError_t launch_migrants(sph_ctx *c)
{
    uint32_t n = (uint32_t)c->n;
    if (n == 0) return cudaSuccess;
    const uint32_t tiles = gather_tiles(n), groups = mig_groups(n);
    // counts restart at every compaction (halos may be rebuilt without a new sort)
    cudaError_t e = cudaMemsetAsync(c->mig_count, 0, sizeof(uint32_t) * 2 * SPH_MAX_SLABS, c->stream);
    if (e != cudaSuccess) return e;
    // a fresh copy of the group counts each time: the scan runs in place
    e = cudaMemcpyAsync(c->mig_off, c->mig_grp, sizeof(uint32_t) * groups, cudaMemcpyDeviceToDevice,
                                    c->stream);
    if (e != cudaSuccess) return e;
    mig_scan_kernel<<<1, MG_SCAN_THREADS, 0, c->stream>>>(groups, c->mig_off, c->mig_total);
    c->n_launches++;
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    mig_compact_kernel<<<groups, GATHER_THREADS, 0, c->stream>>>(
        n, tiles, c->mig_off, c->mig_tile, c->keyword, c->kv[c->kv_sorted], c->idt[c->cur], c->tagged_slabs, c->grid.nyz,
        c->migrants, c->mig_count);
    c->n_launches++;
    return cudaGetLastError();
}

// ---- movable slab planes ("domain decomposition with load
// balancing", L389) --------------------------------------------------------------------------------
// C[p] = number of particles in cell planes < p = cell_begin[p * nyz] (the cell table already holds
// it).  Plane s (s = 1..S-1, left to right) = the p in [planes[s-1] + 2, ncx - 2 (S - s)] that minimises
// |C[p] S - s N|, the lowest such p on ties (every slab keeps at least two cell planes, reading A14).
// C is non-decreasing, so the minimum sits at the crossing point: a few binary searches by one thread.
__global__ void balance_kernel(const uint32_t *__restrict__ cell_begin, int ncx, int nyz, uint32_t n, int S,
                               int32_t *__restrict__ planes_out)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    auto C = [&](int p) -> unsigned long long { return (unsigned long long)cell_begin[(size_t)p * (size_t)nyz]; };
    auto first_ge = [&](int lo, int hi, unsigned long long v_times_S) -> int {   // first p in [lo, hi] with C[p] S >= v, else hi + 1
        int a = lo, b = hi + 1;
        while (a < b) {
            const int m = (a + b) >> 1;
            if (C(m) * (unsigned long long)S >= v_times_S) b = m; else a = m + 1;
        }
        return a;
    };
    planes_out[0] = 0;
    planes_out[S] = ncx;
    int prev = 0;
    for (int s = 1; s < S; ++s) {
        const int lo = prev + 2, hi = ncx - 2 * (S - s);
        const unsigned long long T = (unsigned long long)s * (unsigned long long)n;
        const int a = first_ge(lo, hi, T);
        int best;
        if (a == lo) {
            best = lo;
        } else {
            const unsigned long long below = C(a - 1) * (unsigned long long)S;      // < T
            const int q = first_ge(lo, a - 1, below);                                // lowest plane of that plateau
            if (a > hi) best = q;
            else best = (T - below <= C(a) * (unsigned long long)S - T) ? q : a;
        }
        planes_out[s] = best;
        prev = best;
    }
}

cudaError_t launch_balance(sph_ctx *c, int n_slabs, int32_t *d_planes)
{
    balance_kernel<<<1, 32, 0, c->stream>>>(c->cell_begin, c->grid.nc[0], c->grid.nyz, (uint32_t)c->n, n_slabs, d_planes);
    c->n_launches++;
    return cudaGetLastError();
}

}  // namespace sph
