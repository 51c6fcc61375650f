// a7 - particle interactions ("If particle i is in cell c, the thread will
// look for neighbours only in cell c and in cells adjacent to c ... compute the interaction
// between particle i and its neighbours, that is, the sum on the right-hand side of equations
// (7)-(9)").  Physics: Eq. (7), Eq. (9) L106 (p/rho^2 form, reading A2),
// artificial viscosity and Tait equation of state L112, dynamic boundary particles L116.
//
// Two kernels:
//  * interact_staged_kernel (production).  A CTA owns a z-run of `zb` cells of one (cx,cy)
//    column.  With z-fastest keys the candidates of all its targets are 9 contiguous sorted
//    ranges (one per neighbouring column); they are staged once in shared memory.  Each thread
//    owns one target particle and works in two phases so that warps stay converged:
//      filter - stream its 27-cell window from an fp16 copy of the staged positions (broadcast
//               reads, two candidates per half2 instruction, conservative threshold), push the hit
//               mask of every block of 16 candidates on a private shared-memory stack;
//      drain  - whenever a stack in the warp is full (and at the end) all lanes pop pending entries
//               and evaluate the full pair term in fp32 from the exact records, so the expensive
//               path runs with (almost) all lanes active instead of the ~14 % a fused
//               test+interact loop would have.
//  * interact_simple_kernel (cross-check, SPH_OPT_INTERACT_VARIANT = 1): one thread per
//    particle walking the cell table with global loads, as the paper describes it.
//
// FP32-ALU bound (no tensor cores: this is not a dense contraction).
#include <cuda_fp16.h>
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

// ---- staged production kernel --------------------------------------------------------------------
#ifndef SPH_IA_PAD
#define SPH_IA_PAD 0          // extra dynamic shared memory per CTA (occupancy experiments)
#endif
#ifndef SPH_IA_DRAIN
#define SPH_IA_DRAIN 4
#endif
#ifndef SPH_IA_QCAP
#define SPH_IA_QCAP 11
#endif
constexpr int IA_DRAIN = SPH_IA_DRAIN;   // pairs a lane evaluates per drain round
#ifndef SPH_IA_THREADS
#define SPH_IA_THREADS 256
#endif
#ifndef SPH_IA_CAP
#define SPH_IA_CAP 2688
#endif
constexpr int IA_THREADS = SPH_IA_THREADS;
constexpr int IA_QCAP = SPH_IA_QCAP; // stack entries per thread; one entry = hit mask of one block of IA_BLK candidates
constexpr int IA_BLK = 16;           // candidates per filter block = per stack entry
constexpr int IA_ZMAX = 32;          // max cells per z-block
constexpr int IA_CAP = SPH_IA_CAP;   // staged candidates per batch (9 columns x 11 cells x 27 + slack), multiple of 16
constexpr int IA_NBLK = IA_CAP / IA_BLK;
constexpr float IA_FAR = 1e15f;      // coordinate of the dummy partner: r2 = 3e30 is finite, F = 0
constexpr float IA_TINY = 1e-30f;    // r2 floor: a coincident pair (the particle itself) adds exactly 0
static_assert(IA_CAP % IA_BLK == 0 && IA_NBLK <= 256, "block index must fit 8 bits of a stack entry");

// Shared memory of one CTA.  The filter reads ONLY `hp`: 6 bytes per candidate instead of the 16
// of an fp32 record - the filter loop is bound by shared-memory bandwidth (ncu: 79 % of the LSU
// wavefront peak with fp32 records), not by arithmetic.
struct IaSmem {
    float4 rel[IA_CAP + 1];                   // exact position relative to the CTA origin; w = p/rho^2
    float4 vr[IA_CAP + 1];                    // vx, vy, vz, rho (sign bit = boundary type if masses differ)
                                              // slot IA_CAP of both: a particle at rest far outside every
                                              // support, the partner of drain slots that have no pair
    uint4 hp[IA_NBLK * 6];                    // fp16 filter copy: per block of 16 candidates 2 x uint4 of x, of y,
                                              // of z; half2 word k = (candidate k, candidate k + 8), in units of h
                                              // about the centre of the CTA's neighbourhood
    uint32_t stack[IA_QCAP * IA_THREADS];     // [entry][thread]: 16-bit hit mask (bit c = candidate c of the block)
                                              // | block index << 16
    uint32_t cbt[9][IA_ZMAX + 3];             // cell_begin of the 9 columns over [zlo, zhi]
    uint32_t col_vstart[10];                  // virtual start of each column in the concatenation
    uint32_t stage_lo[9], stage_hi[9];        // global index range of the column staged in this batch
    int32_t stage_off[9];                     // smem index = global index + stage_off
};

int interact_threads() { return IA_THREADS; }

__device__ __forceinline__ void sts_u32(uint32_t addr, uint32_t v)
{
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ void sts_u16(uint32_t addr, unsigned short v)
{
    asm volatile("st.shared.u16 [%0], %1;" ::"r"(addr), "h"(v) : "memory");
}
__device__ __forceinline__ uint32_t lds_u32(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ float4 lds_f4(uint32_t addr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint4 lds_u4(uint32_t addr)
{
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ __half2 as_h2(uint32_t v) { return *reinterpret_cast<__half2 *>(&v); }

// Hit bits of two candidates (the halves of x, y, z) against one target: squared distance in fp16,
// in units of h, below the padded threshold.  0xFFFF per half that passes.
__device__ __forceinline__ uint32_t filt2h(__half2 xi, __half2 yi, __half2 zi, uint32_t x, uint32_t y, uint32_t z,
                                           __half2 thr)
{
    const __half2 dx = __hsub2(xi, as_h2(x)), dy = __hsub2(yi, as_h2(y)), dz = __hsub2(zi, as_h2(z));
    const __half2 r2 = __hfma2(dz, dz, __hfma2(dy, dy, __hmul2(dx, dx)));
    return __hlt2_mask(r2, thr);
}

// Origin of the CTA-relative coordinates along one axis.  x - O is EXACT in fp32 for every staged
// particle (so relative differences equal absolute differences bit for bit): O = 0 when the CTA's
// neighbourhood (reach D around `corner`) is within 2D of the coordinate plane, else `corner` with
// its two lowest mantissa bits cleared, which makes O a multiple of ulp(x) for all |x| <= |O| + D
// while |x - O| <= D <= |x| keeps the difference inside 24 bits.
__device__ __forceinline__ float rel_origin(float corner, float reach)
{
    if (fabsf(corner) < 2.0f * reach) return 0.0f;
    return __uint_as_float(__float_as_uint(corner) & ~3u);
}

template <int KERNEL, bool UNIFORM, bool GAMMA7, bool MU>
__global__ void __launch_bounds__(IA_THREADS, 2)
interact_staged_kernel(const float4 *__restrict__ pos4, const float4 *__restrict__ velrho4,
                       const uint32_t *__restrict__ idt, const uint32_t *__restrict__ keyword,
                       const uint32_t *__restrict__ cell_begin, float4 *__restrict__ acc4, float *__restrict__ mu_out,
                       GridC g, PhysC ph, int zb, int nzb, float thr_h /* filter threshold, units of h^2 */,
                       float zlim /* |z| bound the threshold was derived for, units of h */,
                       int cx_first /* first cell plane of the targets (per-slab execution), else 0 */)
{
    extern __shared__ __align__(16) unsigned char ia_raw[];
    IaSmem &S = *reinterpret_cast<IaSmem *>(ia_raw);
    __shared__ uint32_t s_wide;       // some staged particle or target lies outside the fp16 error model
    const int tid = threadIdx.x;

    // ---- which z-block
    uint32_t b = blockIdx.x;
    const int bz = b % nzb;
    b /= nzb;
    const int cy = b % g.nc[1];
    const int cx = b / g.nc[1] + cx_first;
    const int cz0 = bz * zb, cz1 = min(cz0 + zb, g.nc[2]);
    const uint32_t own_col = (uint32_t)(cx * g.nc[1] + cy) * g.nc[2];
    const uint32_t t_begin = cell_begin[own_col + cz0], t_end = cell_begin[own_col + cz1];
    if (t_begin == t_end) return;

    const int zlo = max(cz0 - 1, 0), zhi = min(cz1 + 1, g.nc[2]);
    const int nz = zhi - zlo;                                    // <= zb + 2
    if (tid == 0) {
        s_wide = 0u;
        S.rel[IA_CAP] = make_float4(IA_FAR, IA_FAR, IA_FAR, 0.f);
        S.vr[IA_CAP] = make_float4(0.f, 0.f, 0.f, 1.f);
    }
    // ---- cell-begin table of the 9 columns
    for (int k = tid; k < 9 * (nz + 1); k += IA_THREADS) {
        int col = k / (nz + 1), z = k % (nz + 1);
        int x = cx + col / 3 - 1, y = cy + col % 3 - 1;
        uint32_t v = 0;
        if (x >= 0 && x < g.nc[0] && y >= 0 && y < g.nc[1])
            v = cell_begin[(uint32_t)(x * g.nc[1] + y) * g.nc[2] + zlo + z];
        S.cbt[col][z] = v;          // columns outside the grid: all 0 => empty ranges
    }
    // ---- CTA-relative coordinate origin (same value in every thread)
    const float cell = 2.0f * ph.h;
    const float ox = rel_origin(fmaf((float)cx, cell, g.min[0]), 4.0f * cell);
    const float oy = rel_origin(fmaf((float)cy, cell, g.min[1]), 4.0f * cell);
    const float oz = rel_origin(fmaf((float)cz0, cell, g.min[2]), (float)(zb + 3) * cell);
    // centre of the neighbourhood in that frame, and the scale of the fp16 filter copy (units of h):
    // |x|, |y| <= 3 and |z| <= nz for every particle that lies inside its cell
    const float inv_h = 2.0f * ph.inv_h_half;
    const float ccx = fmaf((float)cx + 0.5f, cell, g.min[0]) - ox;
    const float ccy = fmaf((float)cy + 0.5f, cell, g.min[1]) - oy;
    const float ccz = fmaf((float)zlo + 0.5f * (float)nz, cell, g.min[2]) - oz;
    __syncthreads();
    if (tid == 0) {
        uint32_t acc = 0;
        for (int col = 0; col < 9; ++col) {
            S.col_vstart[col] = acc;
            acc += S.cbt[col][nz] - S.cbt[col][0];
        }
        S.col_vstart[9] = acc;
    }
    __syncthreads();
    const uint32_t total = S.col_vstart[9];
    const uint32_t lane_full = 0xffffffffu;
    const uint32_t rel_base = (uint32_t)__cvta_generic_to_shared(S.rel);
    const uint32_t vr_delta = (uint32_t)__cvta_generic_to_shared(S.vr) - rel_base;
    const uint32_t hp_base = (uint32_t)__cvta_generic_to_shared(S.hp);
    const uint32_t stk_base = (uint32_t)__cvta_generic_to_shared(S.stack) + 4u * tid;
    constexpr uint32_t STK_STRIDE = 4u * IA_THREADS;
    const uint32_t stk_high = stk_base + STK_STRIDE * (IA_QCAP - 1);   // sp above this = stack full

    for (uint32_t chunk = t_begin; chunk < t_end; chunk += IA_THREADS) {
        const uint32_t i = chunk + tid;
        const bool active = i < t_end;
        float4 pi = make_float4(ox + ccx, oy + ccy, oz + ccz, 0.f), vi = make_float4(0.f, 0.f, 0.f, 1.f);
        int kz = 0;
        bool fluid = false;
        if (active) {
            pi = pos4[i];
            vi = velrho4[i];
            fluid = (idt[i] & TYPE_BIT) == 0;
            kz = (int)((keyword[i] & CELL_MASK) - own_col) - zlo;   // own cz - zlo
        }
        const float xi = pi.x - ox, yi = pi.y - oy, zi = pi.z - oz;  // exact
        // fp16 filter copy of the target; a target outside the error model widens the CTA's filter
        const float xs = (xi - ccx) * inv_h, ys = (yi - ccy) * inv_h, zs = (zi - ccz) * inv_h;
        if (!(fabsf(xs) < 8.0f && fabsf(ys) < 8.0f && fabsf(zs) < zlim)) s_wide = 1u;
        const __half2 hxi = __float2half2_rn(xs), hyi = __float2half2_rn(ys), hzi = __float2half2_rn(zs);
        const float ci = sound_speed<GAMMA7>(vi.w, ph);
        const int k_lo = max(kz - 1, 0), k_hi = min(kz + 2, nz);   // own 3-cell window in cbt rows
        float ax = 0.f, ay = 0.f, az = 0.f, dr = 0.f, mumax = 0.f;
        uint32_t sp = stk_base;                                     // shared address of the stack top
        uint32_t cur_mask = 0, cur_s = 0;                           // entry being drained

        // next pending candidate of this lane: smem index s, or ok = false
        auto pop = [&](uint32_t &s, bool &ok) {
            if (cur_mask == 0 && sp > stk_base) {
                sp -= STK_STRIDE;
                const uint32_t e = lds_u32(sp);
                cur_mask = e & 0xFFFFu;                              // bit c = candidate c of the block
                cur_s = (e >> 12) & 0xFF0u;                          // block index * 16
            }
            ok = cur_mask != 0;
            s = cur_s + (uint32_t)(__ffs(cur_mask) - 1);            // garbage if !ok
            cur_mask &= cur_mask - 1;
        };
        // pair term of candidate s; ok = false turns it into a no-op without a branch: the partner is
        // the far-away dummy slot, whose F is 0.  The exact fp32 distance is
        // formed here: a candidate the fp16 filter let through although it lies outside 2h adds
        // exactly 0 because F is clamped.
        auto interact = [&](uint32_t s, bool ok) {
            s = ok ? s : (uint32_t)IA_CAP;
            const float4 rj = lds_f4(rel_base + 16u * s);
            float4 vj = lds_f4(rel_base + vr_delta + 16u * s);
            const float dx = xi - rj.x, dy = yi - rj.y, dz = zi - rj.z;     // == absolute differences
            const float r2 = fmaxf(fmaf(dz, dz, fmaf(dy, dy, dx * dx)), IA_TINY);
            float mj = 1.0f;
            if (!UNIFORM) {
                mj = vj.w < 0.f ? ph.mass_bound : ph.mass_fluid;
                vj.w = fabsf(vj.w);
            }
            pair_term<KERNEL, GAMMA7, MU>(dx, dy, dz, r2, vi.x, vi.y, vi.z, vi.w, pi.w, ci, vj, rj.w, mj, ph,
                                          ax, ay, az, dr, mumax);
        };
        // one drain round: up to IA_DRAIN pending pairs per lane, as interleaved dependency chains
        auto drain_round = [&]() {
            uint32_t s[IA_DRAIN];
            bool ok[IA_DRAIN];
#pragma unroll
            for (int q = 0; q < IA_DRAIN; ++q) pop(s[q], ok[q]);
#pragma unroll
            for (int q = 0; q < IA_DRAIN; ++q) interact(s[q], ok[q]);
        };

        for (uint32_t bstart = 0; bstart < total; bstart += IA_CAP) {
            const uint32_t bend = min(total, bstart + IA_CAP);
            __syncthreads();                       // previous batch / chunk fully consumed
            if (tid < 9) {
                uint32_t vs = S.col_vstart[tid], ve = S.col_vstart[tid + 1];
                uint32_t lo = max(vs, bstart), hi = min(ve, bend);
                uint32_t gb = S.cbt[tid][0];
                if (lo < hi) {
                    S.stage_lo[tid] = gb + (lo - vs);
                    S.stage_hi[tid] = gb + (hi - vs);
                    S.stage_off[tid] = (int32_t)(lo - bstart) - (int32_t)(gb + (lo - vs));
                } else {
                    S.stage_lo[tid] = 0; S.stage_hi[tid] = 0; S.stage_off[tid] = 0;
                }
            }
            __syncthreads();
            // ---- stage: the batch is the virtual concatenation [bstart, bend) of the 9 column ranges and
            // smem index = virtual index - bstart.  Four candidates per thread per round with all their
            // global loads issued before the first use, so a round costs one memory latency, not four.
            const uint32_t nst = bend - bstart;
            for (uint32_t k0 = tid; k0 < nst; k0 += 4u * IA_THREADS) {
                float4 p[4], v[4];
                bool bnd[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const uint32_t si = k0 + (uint32_t)u * IA_THREADS;
                    bnd[u] = false;
                    if (si < nst) {
                        const uint32_t vv = bstart + si;
                        int col = 0;
#pragma unroll
                        for (int q = 1; q < 9; ++q) col += (vv >= S.col_vstart[q]) ? 1 : 0;
                        const uint32_t j = S.cbt[col][0] + (vv - S.col_vstart[col]);
                        p[u] = __ldg(pos4 + j);
                        v[u] = __ldg(velrho4 + j);
                        if (!UNIFORM) bnd[u] = (__ldg(idt + j) & TYPE_BIT) != 0;
                    }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const uint32_t si = k0 + (uint32_t)u * IA_THREADS;
                    if (si < nst) {
                        if (!UNIFORM && bnd[u]) v[u].w = -v[u].w;
                        const float xr = p[u].x - ox, yr = p[u].y - oy, zr = p[u].z - oz;
                        S.rel[si] = make_float4(xr, yr, zr, p[u].w);
                        S.vr[si] = v[u];
                        const float xq = (xr - ccx) * inv_h, yq = (yr - ccy) * inv_h, zq = (zr - ccz) * inv_h;
                        if (!(fabsf(xq) < 8.0f && fabsf(yq) < 8.0f && fabsf(zq) < zlim)) s_wide = 1u;
                        // block si / 16: x words at +0, y at +32, z at +64; candidate c = si % 16 is half c / 8 of word c % 8
                        const uint32_t a = hp_base + 96u * (si >> 4) + 4u * (si & 7u) + ((si >> 2) & 2u);
                        sts_u16(a, __half_as_ushort(__float2half_rn(xq)));
                        sts_u16(a + 32u, __half_as_ushort(__float2half_rn(yq)));
                        sts_u16(a + 64u, __half_as_ushort(__float2half_rn(zq)));
                    }
                }
            }
            __syncthreads();
            // a particle outside the fp16 error model (it left the grid and sits clamped in an edge
            // cell): let every candidate through, the drain decides exactly
            const __half2 thr = __float2half2_rn(s_wide ? 65504.0f : thr_h);

            const bool wide = s_wide != 0u;

            // ---- filter + drain.  Blocks of 16 candidates are aligned in shared memory; the first
            // and the last block of a lane's range are trimmed with masks in the entry's bit layout.
            for (int col = 0; col < 9; ++col) {
                int lo = 0, hi = 0;
                if (active) {
                    lo = (int)max(S.cbt[col][k_lo], S.stage_lo[col]);
                    hi = (int)min(S.cbt[col][k_hi], S.stage_hi[col]);
                }
                const int off = S.stage_off[col];
                const bool work = hi > lo;
                const uint32_t slo = work ? (uint32_t)(lo + off) : 0u, shi = work ? (uint32_t)(hi + off) : 0u;
                const uint32_t blk_lo = slo >> 4;
                const int nblk = work ? (int)(((shi + 15u) >> 4) - blk_lo) : 0;
                const int maxblk = __reduce_max_sync(lane_full, nblk);
                uint32_t lin = (0xFFFFu << (slo & 15u)) & 0xFFFFu;                    // candidates >= slo
                const uint32_t first_mask = (lin & 0xFFu) | ((lin & 0xFF00u) << 8);
                lin = 0xFFFFu >> ((16u - (shi & 15u)) & 15u);                          // candidates < shi
                const uint32_t last_mask = (lin & 0xFFu) | ((lin & 0xFF00u) << 8);
                for (int it = 0; it < maxblk; ++it) {
                    const uint32_t blk = min(blk_lo + (uint32_t)it, (uint32_t)(IA_NBLK - 1));
                    const uint32_t a0 = hp_base + 96u * blk;
                    const uint4 x0 = lds_u4(a0), x1 = lds_u4(a0 + 16u);
                    const uint4 y0 = lds_u4(a0 + 32u), y1 = lds_u4(a0 + 48u);
                    const uint4 z0 = lds_u4(a0 + 64u), z1 = lds_u4(a0 + 80u);
                    uint32_t m;
                    m = filt2h(hxi, hyi, hzi, x0.x, y0.x, z0.x, thr) & 0x00010001u;
                    m |= filt2h(hxi, hyi, hzi, x0.y, y0.y, z0.y, thr) & 0x00020002u;
                    m |= filt2h(hxi, hyi, hzi, x0.z, y0.z, z0.z, thr) & 0x00040004u;
                    m |= filt2h(hxi, hyi, hzi, x0.w, y0.w, z0.w, thr) & 0x00080008u;
                    m |= filt2h(hxi, hyi, hzi, x1.x, y1.x, z1.x, thr) & 0x00100010u;
                    m |= filt2h(hxi, hyi, hzi, x1.y, y1.y, z1.y, thr) & 0x00200020u;
                    m |= filt2h(hxi, hyi, hzi, x1.z, y1.z, z1.z, thr) & 0x00400040u;
                    m |= filt2h(hxi, hyi, hzi, x1.w, y1.w, z1.w, thr) & 0x00800080u;
                    if (wide) m = 0x00FF00FFu;
                    if (it == 0) m &= first_mask;
                    if (it == nblk - 1) m &= last_mask;
                    if (it < nblk && m) {                   // entry: linear 16-bit mask | block index << 16
                        sts_u32(sp, (m & 0xFFu) | ((m >> 8) & 0xFF00u) | (blk << 16));
                        sp += STK_STRIDE;
                    }
                    while (__any_sync(lane_full, sp > stk_high)) drain_round();
                }
            }
            // ---- flush the stacks before the staged data is replaced.  Until here the stacks are
            // kept as full as they can be (drains only when some lane's stack is full), so that
            // nearly every lane has a pending pair in every drain round.
            while (__any_sync(lane_full, (sp > stk_base) || cur_mask != 0)) drain_round();
        }
        if (active) {
            if (UNIFORM) { ax *= ph.mass_fluid; ay *= ph.mass_fluid; az *= ph.mass_fluid; dr *= ph.mass_fluid; }
            if (fluid) { ax += ph.g[0]; ay += ph.g[1]; az += ph.g[2]; }
            else { ax = ay = az = 0.f; }
            acc4[i] = make_float4(ax, ay, az, dr);
            if (MU) mu_out[i] = mumax;
        }
    }
}

// Filter threshold in units of h^2 for coordinates |x|, |y| < 8 and |z| < zlim (units of h) held in
// fp16: 4 (= (2h)^2) plus a bound of the error of the fp16 squared distance of any pair with true
// distance < 2h, rounded up to a multiple of 2^-7.
static void filter_threshold(int zb, float *thr_h, float *zlim)
{
    double zl = 8.0;
    while (zl < (double)(zb + 2) + 1.0) zl *= 2.0;
    const double ex = 0.0078125 + 0.001953125;            // two half-ulps below 8 + rounding of the difference
    const double ez = zl / 2048.0 + 0.001953125;          // two half-ulps below zl + rounding of the difference
    const double m = 4.1 * sqrt(2.0 * ex * ex + ez * ez) + 3.0 * (2.0 * ex * ex + ez * ez) + 0.012;
    *thr_h = (float)(ceil((4.0 + 1.25 * m) * 128.0) / 128.0);
    *zlim = (float)zl;
}

template <int KERNEL, bool UNIFORM, bool GAMMA7, bool MU>
static cudaError_t launch_staged(sph_ctx *c)
{
    auto kern = interact_staged_kernel<KERNEL, UNIFORM, GAMMA7, MU>;
    int zb = c->zblock;
    int nzb = (c->grid.nc[2] + zb - 1) / zb;
    const IaOverride &ov = c->ia_ov;               // per-slab execution works on a local particle set
    const int cx_first = ov.on ? ov.cx_first : 0, cx_count = ov.on ? ov.cx_count : c->grid.nc[0];
    uint64_t blocks = (uint64_t)cx_count * c->grid.nc[1] * nzb;
    if (blocks == 0) return cudaSuccess;
    float thr_h, zlim;
    filter_threshold(zb, &thr_h, &zlim);
    kern<<<(uint32_t)blocks, IA_THREADS, sizeof(IaSmem) + SPH_IA_PAD, c->stream>>>(
        ov.on ? ov.pos4 : c->pos4[c->cur], ov.on ? ov.velrho4 : c->velrho4[c->cur], ov.on ? ov.idt : c->idt[c->cur],
        ov.on ? ov.keyword : c->keyword, ov.on ? ov.cell_begin : c->cell_begin, ov.on ? ov.acc4 : c->acc4, c->mumax,
        c->grid, c->phys, zb, nzb, thr_h, zlim, cx_first);
    c->n_launches++;
    return cudaGetLastError();
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
    const bool uni = c->phys.uniform_mass != 0, g7 = c->phys.gamma == 7;
    const int k = c->phys.kernel;
    if (c->interact_variant == 1) {
        if (k == 0) return g7 ? launch_simple<0, true, MU>(c) : launch_simple<0, false, MU>(c);
        return g7 ? launch_simple<1, true, MU>(c) : launch_simple<1, false, MU>(c);
    }
    if (c->interact_variant == 0) return launch_interact_mma(c, MU);
    if (k == 0) {
        if (uni) return g7 ? launch_staged<0, true, true, MU>(c) : launch_staged<0, true, false, MU>(c);
        return g7 ? launch_staged<0, false, true, MU>(c) : launch_staged<0, false, false, MU>(c);
    }
    if (uni) return g7 ? launch_staged<1, true, true, MU>(c) : launch_staged<1, true, false, MU>(c);
    return g7 ? launch_staged<1, false, true, MU>(c) : launch_staged<1, false, false, MU>(c);
}

// Dynamic shared memory opt-in of every instance of the staged kernel, for the CURRENT device (the
// attribute is per device; sph_init calls this for every new context).
template <int KERNEL, bool UNIFORM, bool GAMMA7>
static cudaError_t configure_staged()
{
    cudaError_t e = cudaFuncSetAttribute(interact_staged_kernel<KERNEL, UNIFORM, GAMMA7, false>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(IaSmem) + SPH_IA_PAD);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(interact_staged_kernel<KERNEL, UNIFORM, GAMMA7, true>,
                                cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(IaSmem) + SPH_IA_PAD);
}

cudaError_t configure_interact()
{
    cudaError_t e = configure_interact_mma();
#define SPH_CFG(K, U, G) if (e == cudaSuccess) e = configure_staged<K, U, G>()
    SPH_CFG(0, true, true); SPH_CFG(0, true, false); SPH_CFG(0, false, true); SPH_CFG(0, false, false);
    SPH_CFG(1, true, true); SPH_CFG(1, true, false); SPH_CFG(1, false, true); SPH_CFG(1, false, false);
#undef SPH_CFG
    return e;
}

// with_mu: also write max_j |mu_ij| per particle (needed by the variable time step only)
cudaError_t launch_interact(sph_ctx *c, bool with_mu)
{
    if (c->n == 0) return cudaSuccess;
    return with_mu ? launch_interact_mu<true>(c) : launch_interact_mu<false>(c);
}

}  // namespace sph
