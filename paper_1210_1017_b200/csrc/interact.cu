// a7 - particle interactions ("If particle i is in cell c, the thread will
// look for neighbours only in cell c and in cells adjacent to c ... compute the interaction
// between particle i and its neighbours, that is, the sum on the right-hand side of equations
// (7)-(9)").  Physics: Eq. (7), Eq. (9) L106 (p/rho^2 form, reading A2),
// artificial viscosity and Tait equation of state L112, dynamic boundary particles L116.
//
// The production kernel lives in interact_mma.cu.  This file holds
//  * interact_simple_kernel (cross-check, SPH_OPT_INTERACT_VARIANT = 1): one thread per particle walking
//    the cell table with global loads, as the paper describes it - the independent second opinion the
//    parity tests compare the production kernel with;
//  * pair_stats_kernel: candidate and neighbour counts for the flop figure of bench.py.
// (The round-1 staged kernel with the fp16 ALU filter, variant 2, was retired in round 3: it was a third
// code path that nothing timed; git history has it.)
//
// FP32-ALU bound (no tensor cores: this is not a dense contraction).
#include "sph_internal.cuh"
#include "interact_pair.cuh"

namespace sph {

// ---- simple cross-check kernel -----------------------------------------------------------------
template <int KERNEL, bool GAMMA7, bool MU>
__global__ void __launch_bounds__(128)
interact_simple_kernel(uint32_t n, const float4 *__restrict__ pos4, const float4 *__restrict__ velrho4,
                       const uint32_t *__restrict__ idt, const uint32_t *__restrict__ keyword,
                       const uint32_t *__restrict__ cell_begin, float4 *__restrict__ acc4, float *__restrict__ mu_out,
                       GridC g, PhysC ph)
{
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float mumax = 0.f;
    float4 pi = pos4[i];
    float4 vi = velrho4[i];
    uint32_t cell = keyword[i] & CELL_MASK;
    int cz = cell % g.nc[2];
    int cy = (cell / g.nc[2]) % g.nc[1];
    int cx = cell / g.nyz;
    bool fluid = (idt[i] & TYPE_BIT) == 0;
    float ci = sound_speed<GAMMA7>(vi.w, ph);
    float ax = 0.f, ay = 0.f, az = 0.f, dr = 0.f;
    int zlo = max(cz - 1, 0), zhi = min(cz + 2, g.nc[2]);
    for (int dx = -1; dx <= 1; ++dx) {
        int x = cx + dx;
        if (x < 0 || x >= g.nc[0]) continue;
        for (int dy = -1; dy <= 1; ++dy) {
            int y = cy + dy;
            if (y < 0 || y >= g.nc[1]) continue;
            uint32_t col = (uint32_t)(x * g.nc[1] + y) * g.nc[2];
            uint32_t jb = cell_begin[col + zlo], je = cell_begin[col + zhi];
            for (uint32_t j = jb; j < je; ++j) {
                float4 pj = pos4[j];
                float ddx = pi.x - pj.x, ddy = pi.y - pj.y, ddz = pi.z - pj.z;
                float r2 = fmaf(ddz, ddz, fmaf(ddy, ddy, ddx * ddx));
                if (r2 < ph.four_h2 && r2 > 0.0f) {
                    float4 vj = velrho4[j];
                    float mj = ph.uniform_mass ? ph.mass_fluid
                                               : ((idt[j] & TYPE_BIT) ? ph.mass_bound : ph.mass_fluid);
                    pair_term<KERNEL, GAMMA7, MU>(ddx, ddy, ddz, r2, vi.x, vi.y, vi.z, vi.w, pi.w, ci, vj, pj.w, mj, ph,
                                                  ax, ay, az, dr, mumax);
                }
            }
        }
    }
    if (fluid) { ax += ph.g[0]; ay += ph.g[1]; az += ph.g[2]; }
    else { ax = ay = az = 0.f; }
    acc4[i] = make_float4(ax, ay, az, dr);
    if (MU) mu_out[i] = mumax;
}

// ---- measurement helper: candidate and neighbour pair counts -----------------------------------
__global__ void __launch_bounds__(128)
pair_stats_kernel(uint32_t n, const float4 *__restrict__ pos4, const uint32_t *__restrict__ keyword,
                  const uint32_t *__restrict__ cell_begin, GridC g, float four_h2, unsigned long long *out)
{
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long cand = 0, acc = 0;
    if (i < n) {
        float4 pi = pos4[i];
        uint32_t cell = keyword[i] & CELL_MASK;
        int cz = cell % g.nc[2], cy = (cell / g.nc[2]) % g.nc[1], cx = cell / g.nyz;
        int zlo = max(cz - 1, 0), zhi = min(cz + 2, g.nc[2]);
        for (int dx = -1; dx <= 1; ++dx)
            for (int dy = -1; dy <= 1; ++dy) {
                int x = cx + dx, y = cy + dy;
                if (x < 0 || x >= g.nc[0] || y < 0 || y >= g.nc[1]) continue;
                uint32_t col = (uint32_t)(x * g.nc[1] + y) * g.nc[2];
                uint32_t jb = cell_begin[col + zlo], je = cell_begin[col + zhi];
                cand += je - jb;
                for (uint32_t j = jb; j < je; ++j) {
                    float4 pj = pos4[j];
                    float ddx = pi.x - pj.x, ddy = pi.y - pj.y, ddz = pi.z - pj.z;
                    float r2 = fmaf(ddz, ddz, fmaf(ddy, ddy, ddx * ddx));
                    acc += (r2 < four_h2 && r2 > 0.0f) ? 1 : 0;
                }
            }
    }
    for (int o = 16; o; o >>= 1) {
        cand += __shfl_xor_sync(0xffffffffu, cand, o);
        acc += __shfl_xor_sync(0xffffffffu, acc, o);
    }
    if ((threadIdx.x & 31) == 0) { atomicAdd(out, cand); atomicAdd(out + 1, acc); }
}

cudaError_t launch_pair_stats(sph_ctx *c, unsigned long long *d_out)
{
    uint32_t n = (uint32_t)c->n;
    cudaError_t e = cudaMemsetAsync(d_out, 0, 16, c->stream);
    if (e != cudaSuccess || n == 0) return e;
    pair_stats_kernel<<<(n + 127) / 128, 128, 0, c->stream>>>(n, c->pos4[c->cur], c->keyword, c->cell_begin,
                                                             c->grid, c->phys.four_h2, d_out);
    return cudaGetLastError();
}

template <int KERNEL, bool GAMMA7, bool MU>
static cudaError_t launch_simple(sph_ctx *c)
{
    uint32_t n = (uint32_t)c->n;
    interact_simple_kernel<KERNEL, GAMMA7, MU><<<(n + 127) / 128, 128, 0, c->stream>>>(
        n, c->pos4[c->cur], c->velrho4[c->cur], c->idt[c->cur], c->keyword, c->cell_begin, c->acc4, c->mumax,
        c->grid, c->phys);
    c->n_launches++;
    return cudaGetLastError();
}

template <bool MU>
static cudaError_t launch_interact_mu(sph_ctx *c)
{
    const bool g7 = c->phys.gamma == 7;
    const int k = c->phys.kernel;
    if (c->interact_variant == 1) {
        if (k == 0) return g7 ? launch_simple<0, true, MU>(c) : launch_simple<0, false, MU>(c);
        return g7 ? launch_simple<1, true, MU>(c) : launch_simple<1, false, MU>(c);
    }
    return launch_interact_mma(c, MU);
}

// Per-device kernel attributes (dynamic shared memory opt-in) for the CURRENT device; sph_init calls this
// for every new context.
cudaError_t configure_interact() { return configure_interact_mma(); }

// with_mu: also write max_j |mu_ij| per particle (needed by the variable time step only)
cudaError_t launch_interact(sph_ctx *c, bool with_mu)
{
    if (c->n == 0) return cudaSuccess;
    return with_mu ? launch_interact_mu<true>(c) : launch_interact_mu<false>(c);
}

}  // namespace sph
