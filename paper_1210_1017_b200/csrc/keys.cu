// a1 - cell label + edge/migration tags per particle, scattered to id order, plus the digit
// histograms of the radix sort ("a CUDA kernel is launched, with one thread per
// particle, that assigns to each particle a label corresponding to the cell to which it
// belongs"; L240 edge labels, L264 migration labels).
//
// HBM-bound: reads pos4 (16 B) + idt (4 B), writes one (keyword, value) pair (8 B) per
// particle.  The pair is written at index id, so that the stable LSD sort that follows
// starts from id order and ends in (cell, id) order whatever the previous order was.
#include "sph_internal.cuh"

namespace sph {

// ---- state initialisation (id order) ----------------------------------------------------
__global__ void init_state_kernel(uint32_t n, const float *__restrict__ pos, const float *__restrict__ vel,
                                  const float *__restrict__ rho, const uint8_t *__restrict__ type,
                                  float4 *__restrict__ pos4, float4 *__restrict__ velrho4,
                                  float4 *__restrict__ velrhoM1, uint32_t *__restrict__ idt,
                                  uint32_t *__restrict__ flags, PhysC ph)
{
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
    float vx = vel[3 * i], vy = vel[3 * i + 1], vz = vel[3 * i + 2];
    float r = rho[i];
    if (!(isfinite(x) && isfinite(y) && isfinite(z) && isfinite(vx) && isfinite(vy) && isfinite(vz) &&
          isfinite(r) && r > 0.f))
        atomicOr(flags, FLAG_NONFINITE);
    pos4[i] = make_float4(x, y, z, tait_p_over_rho2(r, ph));
    float4 vr = make_float4(vx, vy, vz, r);
    velrho4[i] = vr;
    velrhoM1[i] = vr;
    uint32_t t = type ? (type[i] ? TYPE_BIT : 0u) : 0u;
    idt[i] = i | t;
}

cudaError_t launch_init_state(sph_ctx *c, const float *pos, const float *vel, const float *rho,
                              const uint8_t *type)
{
    uint32_t n = (uint32_t)c->n;
    if (n == 0) return cudaSuccess;
    init_state_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(
        n, pos, vel, rho, type, c->pos4[c->cur], c->velrho4[c->cur], c->velrhoM1[c->cur],
        c->idt[c->cur], c->flags, c->phys);
    c->n_launches++;
    return cudaGetLastError();
}

// ---- keys -----------------------------------------------------------------------------------
// Largest s with table[s] <= x, for a shared-memory table of 17 ascending entries padded with
// "infinity" beyond the used ones (4 probes instead of a 15-way compare chain).
template <typename T>
__device__ __forceinline__ int upper_slot(const T *table, T x)
{
    int s = 0;
#pragma unroll
    for (int step = 8; step >= 1; step >>= 1)
        s += (x >= table[s + step]) ? step : 0;
    return s;
}

// prev_mode: 0 = none (no migrants), 1 = previous slab ranges over the current order,
//            2 = caller-supplied prev_init[id]
constexpr int KEYS_CX_TAB = 4096;    // cell planes along x covered by the shared-memory slab table
constexpr int KEYS_IPT = 4;          // particles per thread per iteration (independent loads in flight)

template <int PASSES>
__global__ void __launch_bounds__(256)
keys_kernel(uint32_t n, const float4 *__restrict__ pos4, const uint32_t *__restrict__ idt,
            uint2 *__restrict__ kv_by_id, uint32_t *__restrict__ hist, uint32_t *__restrict__ flags,
            GridC g, SlabC sl, int prev_mode, int prev_n, const uint32_t *__restrict__ prev_slab_begin,
            const uint8_t *__restrict__ prev_init)
{
    __shared__ uint32_t s_hist[PASSES * 256];
    __shared__ uint32_t s_prev_begin[SPH_MAX_SLABS + 2];
    __shared__ int s_planes[SPH_MAX_SLABS + 2];
    __shared__ uint8_t s_cx_tab[KEYS_CX_TAB];     // slab | edge label << 4 of every cell plane (if nc[0] fits)
    for (int k = threadIdx.x; k < PASSES * 256; k += blockDim.x) s_hist[k] = 0;
    if (threadIdx.x <= SPH_MAX_SLABS) {
        const int t = threadIdx.x;
        s_planes[t] = t < sl.n_slabs ? sl.planes[t] : 0x7fffffff;          // planes[S] = ncx is never reached
        s_prev_begin[t] = (prev_mode == 1 && t < prev_n) ? prev_slab_begin[t] : 0xffffffffu;
        if (t == 0) { s_planes[SPH_MAX_SLABS + 1] = 0x7fffffff; s_prev_begin[0] = 0; }
    }
    __syncthreads();
    const int S = sl.n_slabs;
    const bool use_tab = g.nc[0] <= KEYS_CX_TAB;
    if (use_tab) {
        for (int cx = threadIdx.x; cx < g.nc[0]; cx += blockDim.x) {
            const int slab = upper_slot(s_planes, cx);
            uint32_t lab = 0;                                          // edge label (L240)
            if (slab > 0 && cx == s_planes[slab]) lab = 1;
            if (slab < S - 1 && cx == s_planes[slab + 1] - 1) lab = 2;
            s_cx_tab[cx] = (uint8_t)(slab | (lab << 4));
        }
        __syncthreads();
    }

    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    constexpr uint32_t WCHUNK = 32 * KEYS_IPT;
    const uint32_t stride = gridDim.x * (blockDim.x >> 5) * WCHUNK;
    // a warp owns WCHUNK consecutive particles per iteration; the loop bound is warp-uniform, so
    // the warp stays converged for match_any
    int prev_s = 0;
    uint32_t prev_lo = 1, prev_hi = 0;            // empty range: the first particle searches
    for (uint32_t base = (blockIdx.x * (blockDim.x >> 5) + warp) * WCHUNK; base < n; base += stride) {
        float4 p[KEYS_IPT];
        uint32_t w[KEYS_IPT];
#pragma unroll
        for (int k = 0; k < KEYS_IPT; ++k) {
            const uint32_t i = base + k * 32 + lane;
            if (i < n) { p[k] = __ldg(pos4 + i); w[k] = __ldg(idt + i); }
            else { p[k] = make_float4(0.f, 0.f, 0.f, 0.f); w[k] = 0; }
        }
#pragma unroll
        for (int k = 0; k < KEYS_IPT; ++k) {
            const uint32_t i = base + k * 32 + lane;
            const bool valid = i < n;
            uint32_t cell = 0;
            if (valid) {
                const uint32_t id = w[k] & ID_MASK;
                // one test for the three coordinates: NaN and Inf survive the sum (so does an overflow of finite
                // values beyond 1e38 m, which is no position either)
                if (!(fabsf(p[k].x) + fabsf(p[k].y) + fabsf(p[k].z) < __int_as_float(0x7f800000))) atomicOr(flags, FLAG_NONFINITE);
                const int cx = cell_coord(p[k].x, g.min[0], g.inv_cell, g.nc[0]);
                const int cy = cell_coord(p[k].y, g.min[1], g.inv_cell, g.nc[1]);
                const int cz = cell_coord(p[k].z, g.min[2], g.inv_cell, g.nc[2]);
                cell = (uint32_t)((cx * g.nc[1] + cy) * g.nc[2] + cz);
                int slab;
                uint32_t lab = 0;                                          // edge label (L240)
                if (use_tab) {
                    const uint32_t t = s_cx_tab[cx];
                    slab = (int)(t & 15u);
                    lab = t >> 4;
                } else {
                    slab = upper_slot(s_planes, cx);
                    if (slab > 0 && cx == s_planes[slab]) lab = 1;
                    if (slab < S - 1 && cx == s_planes[slab + 1] - 1) lab = 2;
                }
                int prev = slab;
                if (prev_mode == 1) {
                    // previous owner = slab range of the current index; consecutive indices almost
                    // always stay in the range found last
                    if (i < prev_lo || i >= prev_hi) {
                        prev_s = upper_slot(s_prev_begin, i);
                        prev_lo = s_prev_begin[prev_s];
                        prev_hi = s_prev_begin[prev_s + 1];
                    }
                    prev = prev_s;
                } else if (prev_mode == 2) prev = min((int)prev_init[id], S - 1);
                const uint32_t mig = slab < prev ? 1u : (slab > prev ? 2u : 0u);   // migration label (L264)
                const uint32_t tag = lab | (mig << 2);
                kv_by_id[id] = make_uint2((tag << TAG_SHIFT) | cell, ((uint32_t)prev << 28) | i);
            }
            // digit histograms in shared memory, all passes at once from the runs of equal CELLS in the warp:
            // the lane that starts a run adds the run's length to the run's digit of every pass.  In a
            // running simulation the 32 particles of a row lie in one to three cells (a handful of atomics
            // per row); random keys make every lane a run of one (one atomic per key and pass, which hardly
            // collide with ~28 distinct digits among 32 lanes).
            const uint32_t key = valid ? cell : 0xFFFFFFFFu;           // invalid lanes are a suffix: one last run
            const uint32_t left = __shfl_up_sync(0xffffffffu, key, 1);
            const uint32_t heads = __ballot_sync(0xffffffffu, lane == 0 || key != left);
            if (valid && ((heads >> lane) & 1u)) {
                const uint32_t after = heads & ~((2u << lane) - 1u);   // run heads to the right of this lane
                const uint32_t len = (after ? (uint32_t)__ffs(after) - 1u : 32u) - lane;
#pragma unroll
                for (int q = 0; q < PASSES; ++q) atomicAdd(&s_hist[q * 256 + ((cell >> (8 * q)) & 255u)], len);
            }
        }
    }
    __syncthreads();
    for (int k = threadIdx.x; k < PASSES * 256; k += blockDim.x) {
        uint32_t v = s_hist[k];
        if (v) atomicAdd(&hist[k], v);
    }
}

// Resident CTAs per SM of the key kernel this context uses: constant per context, asked once (sph_init)
// instead of on every step.
cudaError_t configure_keys(sph_ctx *c)
{
    int per_sm = 0;
    cudaError_t e;
    auto occ = [&](auto kern) { return cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, 256, 0); };
    switch (c->passes) {
    case 1: e = occ(keys_kernel<1>); break;
    case 2: e = occ(keys_kernel<2>); break;
    case 3: e = occ(keys_kernel<3>); break;
    default: e = occ(keys_kernel<4>); break;
    }
    c->keys_blocks_per_sm = per_sm > 0 ? per_sm : 1;
    return e;
}

cudaError_t launch_keys(sph_ctx *c)
{
    uint32_t n = (uint32_t)c->n;
    cudaError_t e = cudaMemsetAsync(c->hist, 0, sizeof(uint32_t) * 256 * 4, c->stream);
    if (e != cudaSuccess) return e;
    if (n == 0) return cudaSuccess;
    int prev_mode = c->have_prev_init ? 2 : (c->have_prev_ranges ? 1 : 0);
    uint32_t blocks = (n + 256 * KEYS_IPT - 1) / (256 * KEYS_IPT);
    // grid-stride loop: exactly one resident wave, so that no SM waits for a second, partial one
    uint32_t cap = (uint32_t)c->num_sms * (uint32_t)c->keys_blocks_per_sm;
    if (blocks > cap) blocks = cap;
    const float4 *pos4 = c->pos4[c->cur];
    const uint32_t *idt = c->idt[c->cur];
    uint2 *kv = c->kv[0];
#define SPH_KEYS(P)                                                                              \
    keys_kernel<P><<<blocks, 256, 0, c->stream>>>(n, pos4, idt, kv, c->hist, c->flags, c->grid, \
                                                  c->slabs, prev_mode, c->tagged_slabs.n_slabs, c->slab_begin, \
                                                  c->prev_init)
    switch (c->passes) {
    case 1: SPH_KEYS(1); break;
    case 2: SPH_KEYS(2); break;
    case 3: SPH_KEYS(3); break;
    default: SPH_KEYS(4); break;
    }
#undef SPH_KEYS
    c->n_launches++;
    return cudaGetLastError();
}

}  // namespace sph
