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
//      filter - stream its 27-cell window from shared memory (broadcast reads), 6 flops + a
//               compare per candidate, push the smem index of every candidate inside 2h on a
//               private shared-memory stack;
//      drain  - whenever a stack in the warp is nearly full (and at the end) all lanes pop one
//               entry and evaluate the full pair term, so the expensive path runs with (almost)
//               all lanes active instead of the ~14 % a fused test+interact loop would have.
//  * interact_simple_kernel (cross-check, SPH_OPT_INTERACT_VARIANT = 1): one thread per
//    particle walking the cell table with global loads, as the paper describes it.
//
// FP32-ALU bound (no tensor cores: this is not a dense contraction).
#include "sph_internal.cuh"

namespace sph {

// ---- pair term ---------------------------------------------------------------------------------
__device__ __forceinline__ float rsqrt_fast(float x)        // 1 MUFU, |rel err| <= 2^-22
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_fast(float x)          // 1 MUFU, |rel err| <= 2^-23
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Returns F with grad_i W_ij = F r_ij, for 0 < r2 (F -> 0 smoothly at r = 2h and is clamped to
// 0 beyond, so a filter that lets a pair marginally outside 2h through changes nothing).
template <int KERNEL>
__device__ __forceinline__ float kernel_F(float r2, const PhysC &ph)
{
    float rinv = rsqrt_fast(r2);
    float r = r2 * rinv;
    if (KERNEL == 0) {                      // Wendland C2: F = -5 aD (1 - q/2)^3 / h^2
        float t = fmaxf(fmaf(-ph.inv_h_half, r, 1.0f), 0.0f);
        return ph.kF * t * t * t;
    } else {                                // cubic spline, kF = aD / h^2
        float q = r * (2.0f * ph.inv_h_half);
        float t = fmaxf(2.0f - q, 0.0f);
        float f = q <= 1.0f ? fmaf(2.25f, q, -3.0f) : -0.75f * t * t * rinv * ph.h;
        return ph.kF * f;
    }
}

template <bool GAMMA7>
__device__ __forceinline__ float sound_speed(float rho, const PhysC &ph)
{
    float x = rho * ph.inv_rho0;
    if (GAMMA7) return ph.c0 * x * x * x;               // c0 (rho/rho0)^((gamma-1)/2), gamma = 7
    return ph.c0 * __powf(x, 0.5f * (float)(ph.gamma - 1));
}

// Adds the contribution of neighbour j to (ax, ay, az, dr); masses are applied by the caller
// (mj = 1 in the uniform-mass path).  Branch-free: the viscous term uses min(v_ij.r_ij, 0).
template <int KERNEL, bool GAMMA7>
__device__ __forceinline__ void pair_term(float dx, float dy, float dz, float r2,
                                          float vxi, float vyi, float vzi, float rhoi, float Pi_, float ci,
                                          float4 vj, float Pj, float mj, const PhysC &ph,
                                          float &ax, float &ay, float &az, float &dr)
{
    float F = kernel_F<KERNEL>(r2, ph) * mj;
    float dvx = vxi - vj.x, dvy = vyi - vj.y, dvz = vzi - vj.z;
    float dot = fmaf(dvz, dz, fmaf(dvy, dy, dvx * dx));
    dr = fmaf(F, dot, dr);                                            // Eq. (7)
    // L112: Pi = -alpha cbar mu / rhobar = -alpha h (ci+cj) dot / ((r2+eta2)(rhoi+rhoj)) if dot < 0
    float cj = sound_speed<GAMMA7>(vj.w, ph);
    float visc = -ph.alpha_h * (ci + cj) * fminf(dot, 0.0f) * rcp_fast((r2 + ph.eta2) * (rhoi + vj.w));
    float coef = -F * (Pi_ + Pj + visc);                              // Eq. (9)
    ax = fmaf(coef, dx, ax);
    ay = fmaf(coef, dy, ay);
    az = fmaf(coef, dz, az);
}

// ---- simple cross-check kernel -----------------------------------------------------------------
template <int KERNEL, bool GAMMA7>
__global__ void __launch_bounds__(128)
interact_simple_kernel(uint32_t n, const float4 *__restrict__ pos4, const float4 *__restrict__ velrho4,
                       const uint32_t *__restrict__ idt, const uint32_t *__restrict__ keyword,
                       const uint32_t *__restrict__ cell_begin, float4 *__restrict__ acc4, GridC g, PhysC ph)
{
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
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
                    pair_term<KERNEL, GAMMA7>(ddx, ddy, ddz, r2, vi.x, vi.y, vi.z, vi.w, pi.w, ci, vj, pj.w, mj, ph,
                                      ax, ay, az, dr);
                }
            }
        }
    }
    if (fluid) { ax += ph.g[0]; ay += ph.g[1]; az += ph.g[2]; }
    else { ax = ay = az = 0.f; }
    acc4[i] = make_float4(ax, ay, az, dr);
}

// ---- staged production kernel --------------------------------------------------------------------
#ifndef SPH_IA_PAD
#define SPH_IA_PAD 0          // extra dynamic shared memory per CTA (occupancy experiments)
#endif
#ifndef SPH_IA_DRAIN
#define SPH_IA_DRAIN 2
#endif
constexpr int IA_DRAIN = SPH_IA_DRAIN;   // pairs a lane evaluates per drain round
constexpr int IA_THREADS = 256;
constexpr int IA_QCAP = 17;          // stack entries per thread; one entry = hit mask of IA_SUB candidates
constexpr int IA_SUB = 20;           // candidates tested per stack entry (entry = index << 20 | 20-bit mask)
constexpr int IA_ZMAX = 32;          // max cells per z-block
constexpr int IA_CAP = 2688;         // staged candidates per batch (9 columns x 11 cells x 27 + slack), < 4096
constexpr float IA_TINY = 1e-30f;    // r2 floor: a coincident pair (the particle itself) adds exactly 0

struct IaSmem {
    float4 rel[IA_CAP];                       // position relative to the CTA origin, and its square norm
    float4 vr[IA_CAP];                        // vx, vy, vz, rho (sign bit = boundary type if masses differ)
    float pr[IA_CAP];                         // p/rho^2
    uint32_t stack[IA_QCAP * IA_THREADS];     // [entry][thread]: first candidate index << 20 | hit mask
    uint32_t cbt[9][IA_ZMAX + 3];             // cell_begin of the 9 columns over [zlo, zhi]
    uint32_t col_vstart[10];                  // virtual start of each column in the concatenation
    uint32_t stage_lo[9], stage_hi[9];        // global index range of the column staged in this batch
    int32_t stage_off[9];                     // smem index = global index + stage_off
};

size_t interact_smem_bytes(const sph_ctx *) { return sizeof(IaSmem); }

__device__ __forceinline__ void sts_u32(uint32_t addr, uint32_t v)
{
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t lds_u32(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ float lds_f32(uint32_t addr)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ float4 lds_f4(uint32_t addr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
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

template <int KERNEL, bool UNIFORM, bool GAMMA7>
__global__ void __launch_bounds__(IA_THREADS, 2)
interact_staged_kernel(const float4 *__restrict__ pos4, const float4 *__restrict__ velrho4,
                       const uint32_t *__restrict__ idt, const uint32_t *__restrict__ keyword,
                       const uint32_t *__restrict__ cell_begin, float4 *__restrict__ acc4,
                       GridC g, PhysC ph, int zb, int nzb)
{
    extern __shared__ __align__(16) unsigned char ia_raw[];
    IaSmem &S = *reinterpret_cast<IaSmem *>(ia_raw);
    const int tid = threadIdx.x;

    // ---- which z-block
    uint32_t b = blockIdx.x;
    const int bz = b % nzb;
    b /= nzb;
    const int cy = b % g.nc[1];
    const int cx = b / g.nc[1];
    const int cz0 = bz * zb, cz1 = min(cz0 + zb, g.nc[2]);
    const uint32_t own_col = (uint32_t)(cx * g.nc[1] + cy) * g.nc[2];
    const uint32_t t_begin = cell_begin[own_col + cz0], t_end = cell_begin[own_col + cz1];
    if (t_begin == t_end) return;

    const int zlo = max(cz0 - 1, 0), zhi = min(cz1 + 1, g.nc[2]);
    const int nz = zhi - zlo;                                    // <= zb + 2
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
    const uint32_t pr_base = (uint32_t)__cvta_generic_to_shared(S.pr);
    const uint32_t stk_base = (uint32_t)__cvta_generic_to_shared(S.stack) + 4u * tid;
    constexpr uint32_t STK_STRIDE = 4u * IA_THREADS;
    const uint32_t stk_high = stk_base + STK_STRIDE * (IA_QCAP - 1);   // sp above this = stack full
    // conservative filter radius: rounding of the expanded form is < 3e-3 h^2
    const float filt2 = ph.four_h2 + 0.02f * ph.h * ph.h;

    for (uint32_t chunk = t_begin; chunk < t_end; chunk += IA_THREADS) {
        const uint32_t i = chunk + tid;
        const bool active = i < t_end;
        float4 pi = make_float4(ox, oy, oz, 0.f), vi = make_float4(0.f, 0.f, 0.f, 1.f);
        int kz = 0;
        bool fluid = false;
        if (active) {
            pi = pos4[i];
            vi = velrho4[i];
            fluid = (idt[i] & TYPE_BIT) == 0;
            kz = (int)((keyword[i] & CELL_MASK) - own_col) - zlo;   // own cz - zlo
        }
        const float xi = pi.x - ox, yi = pi.y - oy, zi = pi.z - oz;  // exact
        const float fa = -2.0f * xi, fb = -2.0f * yi, fc = -2.0f * zi;
        const float fT = filt2 - fmaf(zi, zi, fmaf(yi, yi, xi * xi));
        const float ci = sound_speed<GAMMA7>(vi.w, ph);
        const int k_lo = max(kz - 1, 0), k_hi = min(kz + 2, nz);   // own 3-cell window in cbt rows
        float ax = 0.f, ay = 0.f, az = 0.f, dr = 0.f;
        uint32_t sp = stk_base;                                     // shared address of the stack top
        uint32_t cur_mask = 0, cur_s = 0;                           // entry being drained

        // next pending candidate of this lane: smem index s, or ok = false
        auto pop = [&](uint32_t &s, bool &ok) {
            if (cur_mask == 0 && sp > stk_base) {
                sp -= STK_STRIDE;
                const uint32_t e = lds_u32(sp);
                cur_mask = e & 0xFFFFFu;
                cur_s = e >> 20;
            }
            ok = cur_mask != 0;
            s = cur_s + (uint32_t)(__ffs(cur_mask) - 1);
            cur_mask &= cur_mask - 1;
        };
        // pair term of candidate s; ok = false turns it into a no-op without a branch (s = 0 is
        // always a staged, finite candidate; its mass factor is zeroed)
        auto interact = [&](uint32_t s, bool ok) {
            s = ok ? s : 0u;
            const float4 rj = lds_f4(rel_base + 16u * s);
            float4 vj = lds_f4(rel_base + vr_delta + 16u * s);
            const float Pj = lds_f32(pr_base + 4u * s);
            const float dx = xi - rj.x, dy = yi - rj.y, dz = zi - rj.z;     // == absolute differences
            const float r2 = fmaxf(fmaf(dz, dz, fmaf(dy, dy, dx * dx)), IA_TINY);
            float mj = ok ? 1.0f : 0.0f;
            if (!UNIFORM) {
                mj = ok ? (vj.w < 0.f ? ph.mass_bound : ph.mass_fluid) : 0.0f;
                vj.w = fabsf(vj.w);
            }
            pair_term<KERNEL, GAMMA7>(dx, dy, dz, r2, vi.x, vi.y, vi.z, vi.w, pi.w, ci, vj, Pj, mj, ph,
                                      ax, ay, az, dr);
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
            // ---- stage: coalesced global reads, one column after the other
            for (int col = 0; col < 9; ++col) {
                const uint32_t lo = S.stage_lo[col], hi = S.stage_hi[col];
                const int32_t off = S.stage_off[col];
                for (uint32_t j = lo + tid; j < hi; j += IA_THREADS) {
                    const float4 p = __ldg(pos4 + j);
                    float4 v = __ldg(velrho4 + j);
                    if (!UNIFORM && (__ldg(idt + j) & TYPE_BIT)) v.w = -v.w;
                    const float xr = p.x - ox, yr = p.y - oy, zr = p.z - oz;
                    S.rel[(int32_t)j + off] = make_float4(xr, yr, zr, fmaf(zr, zr, fmaf(yr, yr, xr * xr)));
                    S.vr[(int32_t)j + off] = v;
                    S.pr[(int32_t)j + off] = p.w;
                }
            }
            __syncthreads();

            // ---- filter + drain
            for (int col = 0; col < 9; ++col) {
                int lo = 0, hi = 0;
                if (active) {
                    lo = (int)max(S.cbt[col][k_lo], S.stage_lo[col]);
                    hi = (int)min(S.cbt[col][k_hi], S.stage_hi[col]);
                }
                const int off = S.stage_off[col];
                const int len = max(hi - lo, 0);
                const int maxlen = __reduce_max_sync(lane_full, len);
                // lanes without work in this column read from index 0 and record nothing
                const bool work = len > 0;
                const int minlen = __reduce_min_sync(lane_full, work ? len : 0x7fffffff);
                uint32_t s = work ? (uint32_t)(lo + off) : 0u;       // smem index of the next candidate
                const uint32_t s_hi = s + (uint32_t)len;
                int sb = 0;
                // sub-batches of IA_SUB that are complete for every working lane: no range checks.
                // |r_ij|^2 < R^2  <=>  |r_j|^2 - 2 r_i.r_j < R^2 - |r_i|^2   (3 FFMA + 1 compare)
                for (; sb + IA_SUB <= minlen && sb < maxlen; sb += IA_SUB, s += IA_SUB) {
                    uint32_t mask = 0;
                    const uint32_t a0 = rel_base + 16u * s;
#pragma unroll
                    for (int u = 0; u < IA_SUB; ++u) {
                        const float4 rj = lds_f4(a0 + 16u * u);
                        if (fmaf(fc, rj.z, fmaf(fb, rj.y, fmaf(fa, rj.x, rj.w))) < fT) mask |= 1u << u;
                    }
                    if (work && mask) { sts_u32(sp, (s << 20) | mask); sp += STK_STRIDE; }
                    while (__any_sync(lane_full, sp > stk_high)) drain_round();
                }
                // ragged remainder in groups of 4 with per-lane range checks (reads past s_hi stay
                // inside the CTA's shared memory: s < IA_CAP and advances by at most IA_CAP)
                for (; sb < maxlen; sb += 4, s += 4) {
                    uint32_t mask = 0;
                    const uint32_t a0 = rel_base + 16u * s;
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const float4 rj = lds_f4(a0 + 16u * u);
                        if (s + u < s_hi && fmaf(fc, rj.z, fmaf(fb, rj.y, fmaf(fa, rj.x, rj.w))) < fT) mask |= 1u << u;
                    }
                    if (mask) { sts_u32(sp, (s << 20) | mask); sp += STK_STRIDE; }
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
        }
    }
}

template <int KERNEL, bool UNIFORM, bool GAMMA7>
static cudaError_t launch_staged(sph_ctx *c)
{
    auto kern = interact_staged_kernel<KERNEL, UNIFORM, GAMMA7>;
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(IaSmem) + SPH_IA_PAD);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    int zb = c->zblock;
    int nzb = (c->grid.nc[2] + zb - 1) / zb;
    uint64_t blocks = (uint64_t)c->grid.nc[0] * c->grid.nc[1] * nzb;
    kern<<<(uint32_t)blocks, IA_THREADS, sizeof(IaSmem) + SPH_IA_PAD, c->stream>>>(
        c->pos4[c->cur], c->velrho4[c->cur], c->idt[c->cur], c->keyword, c->cell_begin, c->acc4, c->grid,
        c->phys, zb, nzb);
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

template <int KERNEL, bool GAMMA7>
static cudaError_t launch_simple(sph_ctx *c)
{
    uint32_t n = (uint32_t)c->n;
    interact_simple_kernel<KERNEL, GAMMA7><<<(n + 127) / 128, 128, 0, c->stream>>>(
        n, c->pos4[c->cur], c->velrho4[c->cur], c->idt[c->cur], c->keyword, c->cell_begin, c->acc4, c->grid,
        c->phys);
    c->n_launches++;
    return cudaGetLastError();
}

cudaError_t launch_interact(sph_ctx *c)
{
    if (c->n == 0) return cudaSuccess;
    const bool uni = c->phys.uniform_mass != 0, g7 = c->phys.gamma == 7;
    const int k = c->phys.kernel;
    if (c->interact_variant == 1) {
        if (k == 0) return g7 ? launch_simple<0, true>(c) : launch_simple<0, false>(c);
        return g7 ? launch_simple<1, true>(c) : launch_simple<1, false>(c);
    }
    if (k == 0) {
        if (uni) return g7 ? launch_staged<0, true, true>(c) : launch_staged<0, true, false>(c);
        return g7 ? launch_staged<0, false, true>(c) : launch_staged<0, false, false>(c);
    }
    if (uni) return g7 ? launch_staged<1, true, true>(c) : launch_staged<1, true, false>(c);
    return g7 ? launch_staged<1, false, true>(c) : launch_staged<1, false, false>(c);
}

}  // namespace sph
