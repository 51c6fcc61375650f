// a7 - particle interactions, production kernel ("If particle i is in cell c, the
// thread will look for neighbours only in cell c and in cells adjacent to c ... compute the interaction
// between particle i and its neighbours, that is, the sum on the right-hand side of equations (7)-(9)").
// Physics: Eq. (7), Eq. (9) L106 (p/rho^2 form, reading A2), artificial viscosity and
// Tait equation of state L112, dynamic boundary particles L116.
//
// Design ("a7"):
//  * A CTA owns a tile of 2 x 2 cell columns x zb cells.  The candidates of all its targets lie in the
//    4 x 4 columns x (zb + 2) cells around it: with z-fastest keys that is 16 contiguous ranges of the
//    sorted arrays, fetched into shared memory by 32 bulk asynchronous copies (cp.async.bulk, the 1-D
//    TMA path) that complete on an mbarrier; a conversion pass turns the raw records in place into
//    tile-relative coordinates (origin = tile centre) and adds  m_j = |x_j|^2 - thr.
//  * FILTER (warp-cooperative, on the tensor cores).  The distance test IS a dense contraction:
//        D_ij = |x_i|^2 + m_j - 2 x_i . x_j  =  r_ij^2 - thr        (K = 4: x, y, z, 1 | m)
//    One mma.sync m16n8k4 (tf32 inputs, fp32 accumulate; the |x_i|^2 term rides in the accumulator
//    input) tests 16 targets against 8 candidates; the B fragment is read straight from the fp32
//    records in shared memory, no separate filter copy.  A warp streams the candidates of its targets'
//    cell rows once for all its 32 targets; the sign bits of D are shifted into 16-bit pieces and
//    stored so that every target lane finds ITS hit mask of 64 candidates as one 64-bit word.
//    tf32 carries 10 mantissa bits, so thr = (2h)^2 plus a bound of the rounding errors (filter_thr):
//    the filter never loses a pair with r < 2h; what it lets through needlessly adds exactly 0 because
//    the pair term recomputes r^2 in fp32 and F is clamped beyond 2h (reading A19).
//  * DRAIN (one lane = one target).  Lanes pop their hits in ascending candidate order and evaluate the
//    pair term in fp32, two pairs per instruction with the packed FFMA2/FMUL2/FADD2 forms of sm_100a
//    (fma.rn.f32x2): the kernel is bound by instruction issue, not by the FP32 pipes.  Hits are consumed
//    in groups of four; an incomplete group is carried over to the next round of the mask ring, so the
//    summation order of a target depends only on its own hit sequence (per-sub-domain execution
//    reproduces the global pass bit for bit, slab_exec.cu).
//  * No tensor cores in the pair term: it is not a contraction.
//
// FP32-ALU bound ("bound": "alu" in bench.py).
#include "sph_internal.cuh"
#include "interact_pair.cuh"

namespace sph {

#ifndef SPH_IM_THREADS
#define SPH_IM_THREADS 352
#endif
#ifndef SPH_IM_RB
#define SPH_IM_RB 9
#endif
#ifndef SPH_IM_MINBLOCKS
#define SPH_IM_MINBLOCKS 2
#endif
constexpr int IM_THREADS = SPH_IM_THREADS;   // 11 warps: 2 x 2 x 3 cells x 27 particles = 324 targets
constexpr int IM_WARPS = IM_THREADS / 32;
constexpr int IM_COLS = 16;                  // staged columns: 4 x 4
constexpr int IM_ZMAX = 6;                   // max cells per z-block (tf32 model: |z| <= (zb + 2) h)
constexpr int IM_CAP = 2304;                 // staged record slots per batch = 36 blocks of 64
constexpr int IM_BATCH = IM_CAP - 128;       // particles per batch (16 x 5 x 27 = 2160): the 4 x-rows start at multiples
                                             // of 32 slots, which costs up to 4 x 31 padding slots
constexpr int IM_RB = SPH_IM_RB;             // mask ring: blocks of 64 candidates per warp per round
constexpr float IM_WIDE_N = -3.0e38f;        // |x|^2 stand-in of "wide" tiles: every real record is a hit
constexpr float IM_FAR = 1e15f;              // coordinate of the dummy partner: r2 = 3e30 is finite, shape = 0
constexpr float IM_TINY = 1e-30f;            // added to r2: a coincident pair (the particle itself) adds exactly 0
static_assert(IM_CAP % 64 == 0 && IM_RB >= 2, "blocks of 64; the ring doubles as scratch for the A rows");

struct __align__(1024) ImSmem {
    float4 recA[IM_CAP + 1];                 // x, y, z relative to the tile centre, p/rho^2; slot IM_CAP = dummy partner
    float4 recB[IM_CAP + 1];                 // vx, vy, vz, rho/rho0 (sign = boundary type if masses differ)
    float marr[IM_CAP + 4];                  // m_j = |x_j|^2 - thr, rounded to tf32
    uint32_t mask[IM_WARPS][IM_RB][64];      // per warp and ring slot: [half][target lane] hit masks of 32 candidates
    uint32_t cbt[IM_COLS][IM_ZMAX + 3];      // cell_begin of the 16 columns over [zlo, zhi]
    uint32_t col_vstart[IM_COLS + 1];        // virtual start of each column in the concatenation
    uint32_t stage_lo[IM_COLS], stage_hi[IM_COLS];   // global index range of the column staged in this batch
    int32_t stage_off[IM_COLS];              // arrival index = global index + stage_off
    uint32_t row_astart[5];                  // slot of the first record of each staged x-row (multiple of 32); [4] = end
    uint32_t row_len[4];                     // records of the row in this batch
    uint32_t tbase[4], tcount[4], tstart[5]; // target ranges of the 2 x 2 own columns
    uint32_t bcnt[32];                       // target sort: bucket counts, then bucket starts
    uint32_t perm[IM_THREADS];               // target sort: (global index | own column << 28) by sorted position
    unsigned long long mbar;                 // completion barrier of the bulk copies
    uint32_t wide;                           // some particle lies outside the tf32 error model
};

struct ImArgs {
    int zb, nzb;                             // cells per z-block, z-blocks per column
    int tx0, nty;                            // first x tile, tiles along y
    int cx_first, cx_end;                    // cell planes that hold the targets
    int cand_lo, cand_hi;                    // cell planes that exist in the arrays (per-slab execution), inclusive
    float thr2;                              // filter threshold, physical units
};

// ---- packed fp32 pairs (sm_100a FFMA2 / FMUL2 / FADD2) --------------------------------------------
typedef unsigned long long f2;
__device__ __forceinline__ f2 pk(float lo, float hi)
{
    f2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void upk(f2 v, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c)
{
    f2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f2 mul2(f2 a, f2 b)
{
    f2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f2 add2(f2 a, f2 b)
{
    f2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

// ---- shared memory, mbarrier and bulk-copy primitives ----------------------------------------------
__device__ __forceinline__ uint32_t im_lds_u32(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ float4 im_lds_f4(uint32_t addr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void im_sts_u16(uint32_t addr, uint32_t v)
{
    asm volatile("st.shared.u16 [%0], %1;" ::"r"(addr), "h"((unsigned short)v) : "memory");
}
__device__ __forceinline__ void mbar_init(uint32_t mbar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t mbar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t mbar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(mbar), "r"(parity) : "memory");
    } while (!done);
}
// 1-D bulk asynchronous copy global -> shared (SASS: UBLKCP); bytes % 16 == 0, both sides 16-byte aligned
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t mbar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(mbar) : "memory");
}
__device__ __forceinline__ float tf32_rna(float x)
{
    uint32_t r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
    return __uint_as_float(r);
}
// D (16 targets x 8 candidates) = A (16 x 4, row) . B (4 x 8, col) + C, tf32 in, fp32 accumulate
__device__ __forceinline__ void mma_tf32_k4(float &d0, float &d1, float &d2, float &d3, uint32_t a0, uint32_t a1,
                                            uint32_t b0, float c0, float c1, float c2, float c3)
{
    asm("mma.sync.aligned.m16n8k4.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%7,%8,%9,%10};"
        : "=f"(d0), "=f"(d1), "=f"(d2), "=f"(d3)
        : "r"(a0), "r"(a1), "r"(b0), "f"(c0), "f"(c1), "f"(c2), "f"(c3));
}
// position of the highest set bit, 0xFFFFFFFF for 0 (one FLO)
__device__ __forceinline__ uint32_t bfind(uint32_t x)
{
    uint32_t r;
    asm("bfind.u32 %0, %1;" : "=r"(r) : "r"(x));
    return r;
}
// piece = piece << 1 | sign(d): one SHF per test result
__device__ __forceinline__ uint32_t push_sign(float d, uint32_t piece)
{
    return __funnelshift_l(__float_as_uint(d), piece, 1);
}

// shape of the kernel gradient without its constant: grad_i W_ij = kF * shape * r_ij
template <int KERNEL>
__device__ __forceinline__ float kernel_shape(float r, float rinv, const PhysC &ph)
{
    if (KERNEL == 0) {                       // Wendland C2: (1 - q/2)^3
        const float t = fmaxf(fmaf(-ph.inv_h_half, r, 1.0f), 0.0f);
        return t * t * t;
    } else {                                 // cubic spline
        const float q = r * (2.0f * ph.inv_h_half);
        const float t = fmaxf(2.0f - q, 0.0f);
        return q <= 1.0f ? fmaf(2.25f, q, -3.0f) : -0.75f * t * t * rinv * ph.h;
    }
}

int interact_mma_threads() { return IM_THREADS; }
int interact_mma_zmax() { return IM_ZMAX; }

template <int KERNEL, bool UNIFORM, bool GAMMA7, bool MU>
__global__ void __launch_bounds__(IM_THREADS, SPH_IM_MINBLOCKS)
interact_mma_kernel(const float4 *__restrict__ pos4, const float4 *__restrict__ velrho4,
                    const uint32_t *__restrict__ idt, const uint32_t *__restrict__ cell_begin,
                    float4 *__restrict__ acc4, float *__restrict__ mu_out, GridC g, PhysC ph, ImArgs A)
{
    extern __shared__ __align__(1024) unsigned char im_raw[];
    ImSmem &S = *reinterpret_cast<ImSmem *>(im_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // ---- which tile
    uint32_t b = blockIdx.x;
    const int bz = b % A.nzb;
    b /= A.nzb;
    const int cy0 = (int)(b % A.nty) * 2;
    const int cx0 = ((int)(b / A.nty) + A.tx0) * 2;
    const int cz0 = bz * A.zb, cz1 = min(cz0 + A.zb, g.nc[2]);
    const int zlo = max(cz0 - 1, 0), zhi = min(cz1 + 1, g.nc[2]);
    const int nz = zhi - zlo;                                    // <= zb + 2
    // ---- empty tiles (most of a dam-break tank) leave at once
    {
        uint32_t any = 0;
#pragma unroll
        for (int t = 0; t < 4; ++t) {
            const int x = cx0 + (t >> 1), y = cy0 + (t & 1);
            if (x >= A.cx_first && x < A.cx_end && y < g.nc[1]) {
                const uint32_t colbase = (uint32_t)(x * g.nc[1] + y) * g.nc[2];
                any |= cell_begin[colbase + cz1] - cell_begin[colbase + cz0];
            }
        }
        if (any == 0) return;
    }
    const uint32_t mbar = (uint32_t)__cvta_generic_to_shared(&S.mbar);
    if (tid == 0) {
        S.wide = 0u;
        mbar_init(mbar, 1u);
        S.recA[IM_CAP] = make_float4(IM_FAR, IM_FAR, IM_FAR, 0.f);
        S.recB[IM_CAP] = make_float4(0.f, 0.f, 0.f, 1.f);
    }
    if (tid < 4) {
        const int x = cx0 + (tid >> 1), y = cy0 + (tid & 1);
        uint32_t tb = 0, te = 0;
        if (x >= A.cx_first && x < A.cx_end && y < g.nc[1]) {
            const uint32_t colbase = (uint32_t)(x * g.nc[1] + y) * g.nc[2];
            tb = cell_begin[colbase + cz0];
            te = cell_begin[colbase + cz1];
        }
        S.tbase[tid] = tb;
        S.tcount[tid] = te - tb;
    }
    for (int k = tid; k < IM_COLS * (nz + 1); k += IM_THREADS) {
        const int col = k / (nz + 1), z = k % (nz + 1);
        const int x = cx0 - 1 + (col >> 2), y = cy0 - 1 + (col & 3);
        uint32_t v = 0;
        if (x >= A.cand_lo && x <= A.cand_hi && y >= 0 && y < g.nc[1])
            v = cell_begin[(uint32_t)(x * g.nc[1] + y) * g.nc[2] + zlo + z];
        S.cbt[col][z] = v;                   // columns that do not exist: all 0 => empty ranges
    }
    __syncthreads();
    if (tid == 0) {
        uint32_t acc = 0;
        for (int col = 0; col < IM_COLS; ++col) {
            S.col_vstart[col] = acc;
            acc += S.cbt[col][nz] - S.cbt[col][0];
        }
        S.col_vstart[IM_COLS] = acc;
        acc = 0;
        for (int t = 0; t < 4; ++t) { S.tstart[t] = acc; acc += S.tcount[t]; }
        S.tstart[4] = acc;
    }
    __syncthreads();
    const uint32_t total = S.col_vstart[IM_COLS];
    const uint32_t ttotal = S.tstart[4];

    // ---- tile-relative coordinates: origin = centre of the staged region.  |x|, |y| <= 4h and
    // |z| <= nz h for every particle that lies inside its cell - the range the tf32 error model
    // (filter_thr) assumes; a particle outside it (it left the grid and sits clamped in an edge cell,
    // reading A13) switches the tile's filter off ("wide": every candidate passes, the drain decides).
    const float cell = 2.0f * ph.h;
    const float ox = fmaf((float)(cx0 + 1), cell, g.min[0]);
    const float oy = fmaf((float)(cy0 + 1), cell, g.min[1]);
    const float oz = fmaf((float)zlo + 0.5f * (float)nz, cell, g.min[2]);
    const float bxy = 2.0f * cell * 1.002f, bzz = 0.5f * (float)nz * cell * 1.002f;

    const uint32_t recA_addr = (uint32_t)__cvta_generic_to_shared(S.recA);
    const uint32_t recB_addr = (uint32_t)__cvta_generic_to_shared(S.recB);
    const uint32_t marr_addr = (uint32_t)__cvta_generic_to_shared(S.marr);
    const uint32_t mwarp = (uint32_t)__cvta_generic_to_shared(&S.mask[warp][0][0]);
    const uint32_t ab_delta = recB_addr - recA_addr;
    const uint32_t dummy_addr = recA_addr + 16u * (uint32_t)IM_CAP;
    const int g8 = lane >> 2, qd = lane & 3;
    const uint32_t full_mask = 0xffffffffu;

    // constants of the pair term (the packed instructions take a scalar operand for both lanes)
    const float kvisc = -ph.alpha_h * ph.c0 * ph.inv_rho0;       // Pi_ij = kvisc * poly * min(v.r, 0) / (r2 + eta2)
    const f2 c_tiny = pk(IM_TINY, IM_TINY), c_eta2 = pk(ph.eta2, ph.eta2);
    const f2 c_mih = pk(-ph.inv_h_half, -ph.inv_h_half), c_one = pk(1.0f, 1.0f), c_kv = pk(kvisc, kvisc);
    const float cexp = 0.5f * (float)(ph.gamma - 1);

    uint32_t phase = 0;
    for (uint32_t chunk = 0; chunk < ttotal; chunk += IM_THREADS) {
        // ---- targets of this chunk, handed to the threads SORTED by (x-row, position inside the cell
        // along x).  How many hits a target meets in each x-row of the staged region depends on where it
        // sits in its cell along x; the drain works row by row, so a warp whose lanes share that position
        // keeps all its lanes busy in every row (a lattice block at rest: 32 instead of 44 rounds of four
        // pairs per target).  The order of a target's own sum does not depend on its lane.
        const uint32_t nchunk = min((uint32_t)IM_THREADS, ttotal - chunk);
        if (tid < 32) S.bcnt[tid] = 0u;
        __syncthreads();
        uint32_t my_i = 0, my_b = 0, my_r = 0, my_tcol = 0;
        if ((uint32_t)tid < nchunk) {
            const uint32_t tq = chunk + tid;
            int tc = 0;
#pragma unroll
            for (int t = 1; t < 4; ++t) tc += (tq >= S.tstart[t]) ? 1 : 0;
            my_tcol = (uint32_t)tc;
            my_i = S.tbase[tc] + (tq - S.tstart[tc]);
            const float px = __ldg(reinterpret_cast<const float *>(pos4 + my_i)) - ox;      // column tc >> 1 spans
            const float ph16 = (px - (float)((tc >> 1) - 1) * cell) * (16.0f / cell);           // [(tx-1) cell, tx cell)
            my_b = (uint32_t)(tc >> 1) * 16u + (uint32_t)min(max(__float2int_rd(ph16), 0), 15);
            my_r = atomicAdd(&S.bcnt[my_b], 1u);
        }
        __syncthreads();
        if (tid < 32) {                               // exclusive scan of the 32 bucket counts
            const uint32_t v = S.bcnt[tid];
            uint32_t inc = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t t = __shfl_up_sync(full_mask, inc, o);
                if (lane >= o) inc += t;
            }
            S.bcnt[tid] = inc - v;
        }
        __syncthreads();
        if ((uint32_t)tid < nchunk) S.perm[S.bcnt[my_b] + my_r] = my_i | (my_tcol << 28);
        __syncthreads();
        const bool active = (uint32_t)tid < nchunk;
        const uint32_t pe = active ? S.perm[tid] : 0u;
        const uint32_t i = pe & 0x0FFFFFFFu;
        const int tcol = (int)(pe >> 28);
        const int tx = tcol >> 1;
        float4 pi = make_float4(ox, oy, oz, 0.f), vi = make_float4(0.f, 0.f, 0.f, ph.rho0);
        bool fluid = false;
        if (active) {
            pi = pos4[i];
            vi = velrho4[i];
            fluid = (idt[i] & TYPE_BIT) == 0;
        }
        const float xi = pi.x - ox, yi = pi.y - oy, zi = pi.z - oz;
        if (active && !(fabsf(xi) <= bxy && fabsf(yi) <= bxy && fabsf(zi) <= bzz)) S.wide = 1u;
        const float ui = vi.w * ph.inv_rho0;
        const float ui2 = GAMMA7 ? ui * ui : __powf(ui, cexp);   // gamma = 7: u^2; else u^((gamma-1)/2)
        // x-rows of the staged region this warp's targets need: [txmin, txmax + 2]
        const int txmin = __reduce_min_sync(full_mask, active ? tx : 2);
        const int txmax = __reduce_max_sync(full_mask, active ? tx : -1);
        const bool warp_has = txmax >= 0;
        // target side of the distance product
        const float xh = tf32_rna(xi), yh = tf32_rna(yi), zh = tf32_rna(zi);
        const float nn = fmaf(zh, zh, fmaf(yh, yh, xh * xh));

        // fragment addressing: lanes 0..2 of a quad read x, y, z of the record, lane 3 reads m.
        // mma group j of a block of 64 slots holds the slots 16 (n >> 1) + 2 j + (n & 1), n = 0..7, so that
        // the 16 sign bits a lane collects for one target are 16 CONSECUTIVE slots of the target's mask.
        const uint32_t sh = qd < 3 ? 4u : 2u;
        const uint32_t lbase = (qd < 3 ? recA_addr + 4u * qd : marr_addr) + ((uint32_t)(16 * (g8 >> 1)) << sh);
        uint32_t foff[4];                         // swizzled slot of group j (j + 4: 8 slots further)
#pragma unroll
        for (int j = 0; j < 4; ++j) foff[j] = (uint32_t)((2 * j + (g8 & 1)) ^ (2 * (g8 >> 1))) << sh;
        // masks are stored bit-reversed (slot s of the block = bit 63 - s of the target's 64-bit word), so
        // that "highest set bit first" (one FLO) walks the candidates in ascending order
        const uint32_t piece_addr = (uint32_t)((qd >> 1) * 128 + ((qd & 1) ^ 1) * 2 + 4 * g8);

        f2 ax2 = pk(0.f, 0.f), ay2 = ax2, az2 = ax2, dr2 = ax2;
        float mumax = 0.f;
        uint32_t odd = 0;                         // parity of the hits consumed so far: the next hit's sub-lane

        // two pairs at once: candidates at the shared addresses sa (low lane) and sb (high lane) of recA
        // against this lane's target
        auto pair2 = [&](uint32_t sa, uint32_t sb) {
            const float4 ra = im_lds_f4(sa), rb = im_lds_f4(sb);
            float4 va = im_lds_f4(sa + ab_delta), vb = im_lds_f4(sb + ab_delta);
            const f2 dx = pk(xi - ra.x, xi - rb.x), dy = pk(yi - ra.y, yi - rb.y), dz = pk(zi - ra.z, zi - rb.z);
            const f2 r2 = add2(fma2(dz, dz, fma2(dy, dy, mul2(dx, dx))), c_tiny);
            float r2a, r2b;
            upk(r2, r2a, r2b);
            const float ia = rsqrt_fast(r2a), ib = rsqrt_fast(r2b);
            float ma = 1.0f, mb = 1.0f;
            if (!UNIFORM) {
                ma = va.w < 0.f ? ph.mass_bound : ph.mass_fluid;
                mb = vb.w < 0.f ? ph.mass_bound : ph.mass_fluid;
                va.w = fabsf(va.w);
                vb.w = fabsf(vb.w);
            }
            f2 F;
            if (KERNEL == 0) {
                const f2 r = mul2(r2, pk(ia, ib));
                f2 t = fma2(r, c_mih, c_one);
                float ta, tb;
                upk(t, ta, tb);
                t = pk(fmaxf(ta, 0.0f), fmaxf(tb, 0.0f));
                F = mul2(mul2(t, t), t);
            } else {
                F = pk(kernel_shape<KERNEL>(r2a * ia, ia, ph), kernel_shape<KERNEL>(r2b * ib, ib, ph));
            }
            if (!UNIFORM) F = mul2(F, pk(ma, mb));
            const f2 dvx = pk(vi.x - va.x, vi.x - vb.x), dvy = pk(vi.y - va.y, vi.y - vb.y),
                     dvz = pk(vi.z - va.z, vi.z - vb.z);
            const f2 dot = fma2(dvz, dz, fma2(dvy, dy, mul2(dvx, dx)));
            dr2 = fma2(F, dot, dr2);                                     // Eq. (7)
            // L112 with c = c0 u^e, rho = rho0 u:  Pi = -alpha h c0/rho0 * (ui^e + uj^e)/(ui + uj) * min(v.r,0)/(r2+eta2);
            // for gamma = 7 (e = 3) the quotient is ui^2 - ui uj + uj^2
            f2 poly;
            if (GAMMA7) {
                poly = pk(fmaf(va.w, va.w - ui, ui2), fmaf(vb.w, vb.w - ui, ui2));
            } else {
                poly = pk(__fdividef(ui2 + __powf(va.w, cexp), ui + va.w), __fdividef(ui2 + __powf(vb.w, cexp), ui + vb.w));
            }
            float qa, qb;
            upk(add2(r2, c_eta2), qa, qb);
            const float rca = rcp_fast(qa), rcb = rcp_fast(qb);
            float da, db;
            upk(dot, da, db);
            const f2 w = mul2(pk(fminf(da, 0.0f), fminf(db, 0.0f)), pk(rca, rcb));
            if (MU) {
                const float mua = ph.h * fabsf(da) * rca, mub = ph.h * fabsf(db) * rcb;
                mumax = fmaxf(mumax, (r2a < ph.four_h2 && ma != 0.0f) ? mua : 0.0f);
                mumax = fmaxf(mumax, (r2b < ph.four_h2 && mb != 0.0f) ? mub : 0.0f);
            }
            const f2 ps = pk(pi.w + ra.w, pi.w + rb.w);
            const f2 coef = mul2(F, fma2(mul2(poly, w), c_kv, ps));      // Eq. (9) without its sign and constants
            ax2 = fma2(coef, dx, ax2);
            ay2 = fma2(coef, dy, ay2);
            az2 = fma2(coef, dz, az2);
        };

        for (uint32_t bstart = 0; bstart < total; bstart += IM_BATCH) {
            const uint32_t bend = min(total, bstart + IM_BATCH);
            __syncthreads();                       // records of the previous batch / chunk are no longer read
            // ---- slots of this batch: x-row r starts at a multiple of 32 (a target's window of three rows is
            // then a whole number of 32-candidate mask words)
            if (tid == 0) {
                uint32_t a = 0;
                for (int r = 0; r < 4; ++r) {
                    const uint32_t lo = min(max(S.col_vstart[4 * r], bstart), bend);
                    const uint32_t hi = min(max(S.col_vstart[4 * r + 4], bstart), bend);
                    S.row_astart[r] = a;
                    S.row_len[r] = hi - lo;
                    a = (a + (hi - lo) + 31u) & ~31u;
                }
                S.row_astart[4] = a;
            }
            __syncthreads();
            if (tid < IM_COLS) {
                const int r = tid >> 2;
                const uint32_t vs = S.col_vstart[tid], ve = S.col_vstart[tid + 1];
                const uint32_t lo = max(vs, bstart), hi = min(ve, bend);
                const uint32_t rlo = min(max(S.col_vstart[4 * r], bstart), bend);    // first particle of the row in the batch
                const uint32_t gb = S.cbt[tid][0];
                if (lo < hi) {
                    S.stage_lo[tid] = gb + (lo - vs);
                    S.stage_hi[tid] = gb + (hi - vs);
                    S.stage_off[tid] = (int32_t)(S.row_astart[r] + (lo - rlo)) - (int32_t)(gb + (lo - vs));
                } else {
                    S.stage_lo[tid] = 0; S.stage_hi[tid] = 0; S.stage_off[tid] = 0;
                }
            }
            __syncthreads();
            // ---- stage: one bulk copy per column and array, all completing on the mbarrier
            if (warp == 0) {
                if (lane == 0) {
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    mbar_arrive_expect_tx(mbar, (bend - bstart) * 32u);
                }
                __syncwarp();
                if (lane < IM_COLS) {
                    const uint32_t lo = S.stage_lo[lane], cnt = S.stage_hi[lane] - lo;
                    if (cnt) {
                        const uint32_t a = (uint32_t)((int32_t)lo + S.stage_off[lane]);
                        bulk_g2s(recA_addr + 16u * a, pos4 + lo, 16u * cnt, mbar);
                        bulk_g2s(recB_addr + 16u * a, velrho4 + lo, 16u * cnt, mbar);
                    }
                }
            }
            mbar_wait(mbar, phase);
            phase ^= 1u;
            // ---- convert in place: tile-relative coordinates, m = |x|^2 - thr (tf32), rho -> rho/rho0; the
            // padding slots between the rows and up to the next block of 64 become records that never hit
            const uint32_t aend = S.row_astart[4];
            const uint32_t nconv = (aend + 63u) & ~63u;
            for (uint32_t a = (uint32_t)tid; a < nconv; a += IM_THREADS) {
                int r = 0;
#pragma unroll
                for (int q = 1; q < 4; ++q) r += (a >= S.row_astart[q]) ? 1 : 0;
                const uint32_t k = a - S.row_astart[r];
                float4 ra = make_float4(0.f, 0.f, 0.f, 0.f), rb = make_float4(0.f, 0.f, 0.f, 1.f);
                float m = __int_as_float(0x7f800000);                        // +inf: D > 0 against any target
                if (a < aend && k < S.row_len[r]) {
                    ra = S.recA[a];
                    rb = S.recB[a];
                    ra.x -= ox; ra.y -= oy; ra.z -= oz;
                    if (!(fabsf(ra.x) <= bxy && fabsf(ra.y) <= bxy && fabsf(ra.z) <= bzz)) S.wide = 1u;
                    m = tf32_rna(fmaf(ra.z, ra.z, fmaf(ra.y, ra.y, ra.x * ra.x)) - A.thr2);
                    rb.w *= ph.inv_rho0;
                    if (!UNIFORM) {
                        const uint32_t vv = min(max(S.col_vstart[4 * r], bstart), bend) + k;   // index in the concatenation
                        int col = 0;
#pragma unroll
                        for (int q = 1; q < IM_COLS; ++q) col += (vv >= S.col_vstart[q]) ? 1 : 0;
                        const uint32_t j = S.cbt[col][0] + (vv - S.col_vstart[col]);
                        if (__ldg(idt + j) & TYPE_BIT) rb.w = -rb.w;
                    }
                }
                __syncwarp();                                // the 32 lanes of a warp cover an aligned run of 32 slots
                const uint32_t sw = a ^ ((a >> 3) & 6u);     // swizzle: the 8 records of an mma B fragment (slots
                S.recA[sw] = ra;                             // 2j + c + 16 q') fall on 8 different 16-byte bank groups
                S.recB[sw] = rb;
                S.marr[sw] = m;
            }
            __syncthreads();
            const bool wide = S.wide != 0u;

            if (warp_has) {
                // ---- A rows of the distance product, handed to the lanes that hold them as mma fragments.
                // "wide" tiles: D = m - 3e38 < 0 for every real record, +inf for the padding slots.
                uint32_t af[4];
                float nf[4];
                {
                    float4 *scratch = reinterpret_cast<float4 *>(&S.mask[warp][0][0]);
                    float4 row = make_float4(-2.0f * xh, -2.0f * yh, -2.0f * zh, nn);
                    if (wide) row = make_float4(0.f, 0.f, 0.f, IM_WIDE_N);
                    if (!active) row = make_float4(0.f, 0.f, 0.f, __int_as_float(0x7f800000));
                    scratch[lane] = row;
                    __syncwarp();
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        const float4 r = scratch[g8 + 8 * k];
                        const float a = qd == 0 ? r.x : (qd == 1 ? r.y : (qd == 2 ? r.z : 1.0f));
                        af[k] = __float_as_uint(a);
                        nf[k] = r.w;
                    }
                    __syncwarp();
                }
                // ---- one round of the mask ring per x-row of the staged region (sub-rounds if a row is longer
                // than the ring): all lanes of a warp meet about the same number of hits in a row, so the
                // drain that follows each filter pass keeps them busy together
                for (int r = txmin; r <= min(txmax + 2, 3); ++r) {
                const uint32_t e0 = S.row_astart[r] >> 5, e1 = S.row_astart[r + 1] >> 5;     // mask words of the row
                const uint32_t e_cnt = (active && r >= tx && r <= tx + 2) ? e1 - e0 : 0u;     // ... that are this lane's
                for (uint32_t rb0 = e0 >> 1; rb0 < ((e1 + 1u) >> 1); rb0 += IM_RB) {
                    const uint32_t nb = min((uint32_t)IM_RB, ((e1 + 1u) >> 1) - rb0);
                    // ---- FILTER: nb blocks of 64 slots against the warp's 32 targets
                    for (uint32_t bi = 0; bi < nb; ++bi) {
                        const uint32_t bb = lbase + (((rb0 + bi) * 64u) << sh);
                        uint32_t p0 = 0, p1 = 0, p2 = 0, p3 = 0;
#pragma unroll
                        for (int j = 0; j < 8; ++j) {
                            const uint32_t bf = im_lds_u32(bb + foff[j & 3] + ((uint32_t)(8 * (j >> 2)) << sh));
                            float d0, d1, d2, d3, d4, d5, d6, d7;
                            mma_tf32_k4(d0, d1, d2, d3, af[0], af[1], bf, nf[0], nf[0], nf[1], nf[1]);
                            mma_tf32_k4(d4, d5, d6, d7, af[2], af[3], bf, nf[2], nf[2], nf[3], nf[3]);
                            p0 = push_sign(d1, push_sign(d0, p0));
                            p1 = push_sign(d3, push_sign(d2, p1));
                            p2 = push_sign(d5, push_sign(d4, p2));
                            p3 = push_sign(d7, push_sign(d6, p3));
                        }
                        const uint32_t ma = mwarp + bi * 256u + piece_addr;
                        im_sts_u16(ma, p0);
                        im_sts_u16(ma + 32u, p1);
                        im_sts_u16(ma + 64u, p2);
                        im_sts_u16(ma + 96u, p3);
                    }
                    __syncwarp();
                    // ---- DRAIN.  Survey of this lane's mask words of the round: which are non-empty (nz,
                    // bit 31 - k = word k) and how many hits they hold; the number of rounds of four pairs
                    // is then known for the whole warp.
                    uint32_t nz = 0, tot = 0;
                    const uint32_t mlane = mwarp + 4u * (uint32_t)lane;          // word k of the round at mlane + 128 k
                    for (uint32_t k = 0; k < 2u * nb; ++k) {
                        uint32_t w = im_lds_u32(mlane + 128u * k);
                        if ((2u * rb0 + k) - e0 >= e_cnt) w = 0u;                  // another row, or not this lane's row
                        tot += (uint32_t)__popc(w);
                        nz |= w ? (0x80000000u >> k) : 0u;
                    }
                    // a lane whose hit count is odd so far leaves its last hit alone in the LOW sub-lane; the
                    // next hit then belongs in the HIGH one: start with the dummy partner in the low sub-lane.
                    // cur = remaining hits of the current word (bit 31 - t = slot t of the word);
                    // atop = shared address of recA[slot of bit 0 of cur] (bit hb is 16 hb bytes below it)
                    uint32_t cur = odd ? 1u : 0u;
                    uint32_t atop = dummy_addr;
                    const uint32_t steps = __reduce_max_sync(full_mask, (tot + odd + 3u) >> 2);
                    odd = (odd + tot) & 1u;
                    const uint32_t atop0 = recA_addr + 16u * (rb0 * 64u + 32u * 31u + 31u);   // word k: atop0 - 512 (31 - k)
                    const uint32_t mtop = mlane + 128u * 31u;                                   // word k at mtop - 128 (31 - k)
                    // branch-free: the next non-empty word is read in any case (word 0 when none is left)
                    auto pop = [&]() -> uint32_t {
                        const uint32_t kb = bfind(nz);                                      // highest bit = lowest word
                        const uint32_t w = im_lds_u32(mtop - 128u * (kb & 31u));
                        const bool take = cur == 0u && nz != 0u;
                        cur = take ? w : cur;
                        atop = take ? atop0 - 512u * kb : atop;
                        nz = take ? nz ^ (1u << (kb & 31u)) : nz;
                        const uint32_t hb = bfind(cur);                                     // 0xFFFFFFFF if cur == 0
                        const uint32_t lin = cur ? atop - 16u * hb : dummy_addr;
                        cur &= ~(1u << (hb & 31u));
                        return lin ^ ((lin >> 3) & 0x60u);                                  // slot swizzle, in bytes
                    };
                    for (uint32_t st = 0; st < steps; ++st) {
                        const uint32_t sa = pop(), sb = pop(), sc = pop(), sd = pop();
                        pair2(sa, sb);
                        pair2(sc, sd);
                    }
                    __syncwarp();
                }
                }
            }
        }
        if (active) {
            float a0, a1, b0, b1, c0, c1, d0, d1;
            upk(ax2, a0, a1); upk(ay2, b0, b1); upk(az2, c0, c1); upk(dr2, d0, d1);
            const float k = UNIFORM ? ph.kF * ph.mass_fluid : ph.kF;
            float ax = -k * (a0 + a1), ay = -k * (b0 + b1), az = -k * (c0 + c1);
            const float dr = k * (d0 + d1);
            if (fluid) { ax += ph.g[0]; ay += ph.g[1]; az += ph.g[2]; }
            else { ax = ay = az = 0.f; }
            acc4[i] = make_float4(ax, ay, az, dr);
            if (MU) mu_out[i] = mumax;
        }
    }
}

// Filter threshold in units of h^2 for tile-relative coordinates |x|, |y| <= 4 and |z| <= zb + 2 (units
// of h): 4 (= (2h)^2) plus a bound of the error of D = |x^_i|^2 + m^_j - 2 x^_i . x~_j against the true
// squared distance of a pair at the cut-off.  x^_i: target rounded to tf32 by this kernel (<= 2^-11
// relative); x~_j: the tensor core's own view of the fp32 candidate coordinates (truncation or rounding,
// <= 2^-10 relative either way); m^_j: rounded to tf32 by this kernel.
static float filter_thr(int zb)
{
    const double rz = (double)(zb + 2), R2 = 16.0 + 16.0 + rz * rz;
    const double e1 = 2.0 * 2.1 * sqrt(R2) / 2048.0;                 // 2 |x^_i - x_i| |x_i - x_j|
    const double e2 = 2.0 * R2 / 1024.0;                              // 2 x^_i . (x_j - x~_j)
    const double e3 = fmax(R2 - 4.0, 4.3) / 2048.0;                   // m^_j - m_j
    const double e4 = 1e-3;                                           // fp32 accumulation of five terms <= 2 R2
    return (float)(4.0 + 1.1 * (e1 + e2 + e3 + e4));
}

template <int KERNEL, bool UNIFORM, bool GAMMA7, bool MU>
static cudaError_t launch_mma(sph_ctx *c)
{
    auto kern = interact_mma_kernel<KERNEL, UNIFORM, GAMMA7, MU>;
    const IaOverride &ov = c->ia_ov;               // per-slab execution works on a local particle set
    ImArgs A;
    A.zb = c->zblock_mma;
    A.nzb = (c->grid.nc[2] + A.zb - 1) / A.zb;
    A.cx_first = ov.on ? ov.cx_first : 0;
    A.cx_end = ov.on ? ov.cx_first + ov.cx_count : c->grid.nc[0];
    A.cand_lo = ov.on ? ov.cand_lo : 0;
    A.cand_hi = ov.on ? ov.cand_hi : c->grid.nc[0] - 1;
    if (A.cx_end <= A.cx_first) return cudaSuccess;
    A.tx0 = A.cx_first >> 1;                       // tiles are anchored at even cell planes of the GLOBAL grid
    const int ntx = ((A.cx_end - 1) >> 1) - A.tx0 + 1;
    A.nty = (c->grid.nc[1] + 1) >> 1;
    A.thr2 = filter_thr(A.zb) * c->phys.h * c->phys.h;
    const uint64_t blocks = (uint64_t)ntx * A.nty * A.nzb;
    if (blocks == 0) return cudaSuccess;
    kern<<<(uint32_t)blocks, IM_THREADS, sizeof(ImSmem), c->stream>>>(
        ov.on ? ov.pos4 : c->pos4[c->cur], ov.on ? ov.velrho4 : c->velrho4[c->cur], ov.on ? ov.idt : c->idt[c->cur],
        ov.on ? ov.cell_begin : c->cell_begin, ov.on ? ov.acc4 : c->acc4, c->mumax, c->grid, c->phys, A);
    c->n_launches++;
    return cudaGetLastError();
}

template <bool MU>
static cudaError_t launch_mma_mu(sph_ctx *c)
{
    const bool uni = c->phys.uniform_mass != 0, g7 = c->phys.gamma == 7;
    if (c->phys.kernel == 0) {
        if (uni) return g7 ? launch_mma<0, true, true, MU>(c) : launch_mma<0, true, false, MU>(c);
        return g7 ? launch_mma<0, false, true, MU>(c) : launch_mma<0, false, false, MU>(c);
    }
    if (uni) return g7 ? launch_mma<1, true, true, MU>(c) : launch_mma<1, true, false, MU>(c);
    return g7 ? launch_mma<1, false, true, MU>(c) : launch_mma<1, false, false, MU>(c);
}

cudaError_t launch_interact_mma(sph_ctx *c, bool with_mu)
{
    return with_mu ? launch_mma_mu<true>(c) : launch_mma_mu<false>(c);
}

template <int KERNEL, bool UNIFORM, bool GAMMA7>
static cudaError_t configure_mma()
{
    cudaError_t e = cudaFuncSetAttribute(interact_mma_kernel<KERNEL, UNIFORM, GAMMA7, false>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(ImSmem));
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(interact_mma_kernel<KERNEL, UNIFORM, GAMMA7, true>,
                                cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(ImSmem));
}

// dynamic shared memory opt-in of every instance, for the current device (sph_init, per context)
cudaError_t configure_interact_mma()
{
    cudaError_t e = cudaSuccess;
#define SPH_CFG(K, U, G) if (e == cudaSuccess) e = configure_mma<K, U, G>()
    SPH_CFG(0, true, true); SPH_CFG(0, true, false); SPH_CFG(0, false, true); SPH_CFG(0, false, false);
    SPH_CFG(1, true, true); SPH_CFG(1, true, false); SPH_CFG(1, false, true); SPH_CFG(1, false, false);
#undef SPH_CFG
    return e;
}

}  // namespace sph
