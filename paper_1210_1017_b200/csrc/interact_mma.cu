// a7 - particle interactions, production kernel ("If particle i is in cell c, the
// thread will look for neighbours only in cell c and in cells adjacent to c ... compute the interaction
// between particle i and its neighbours, that is, the sum on the right-hand side of equations (7)-(9)").
// Physics: Eq. (7), Eq. (9) L106 (p/rho^2 form, reading A2), artificial viscosity and
// Tait equation of state L112, dynamic boundary particles L116.
//
// Design ("a7"):
//  * Work = the non-empty TILES of 2 x 2 cell columns x zb cells, listed by ia_tile_list_kernel.  The
//    candidates of all targets of a tile lie in the 4 x 4 columns x (zb + 2) cells around it: with
//    z-fastest keys that is 16 contiguous ranges of the sorted arrays.
//  * interact_mma_kernel is PERSISTENT (one CTA per SM) and warp-specialised.  The first IM_NP warps are the
//    producers (one group, named barrier): they take the next tile from the list (atomic counter), read its piece of the cell table, fetch
//    the 16 ranges into one of two shared-memory stages with 32 bulk asynchronous copies
//    (cp.async.bulk, the 1-D TMA path, completing on an mbarrier), convert the raw records in place
//    into tile-relative coordinates (origin = tile centre) + m_j = |x_j|^2 - thr, order the tile's
//    targets and publish the stage on a "full" mbarrier.  The other warps are consumers: each takes
//    chunks of 32 targets of a published stage from a shared counter, filters and drains them (below),
//    writes their rates and, when a stage has no chunk left, releases it on an "empty" mbarrier and
//    moves on to the other stage.  Staging of tile k + 1 therefore runs under the arithmetic of tile k,
//    and there is no CTA-wide barrier anywhere after the set-up.
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
//    in groups of four; the k-th hit of a target always lands in sub-lane k & 1, so the summation order
//    of a target depends only on its own hit sequence inside a candidate batch (per-sub-domain execution,
//    slab_exec.cu, reproduces the global pass bit for bit as long as the tiles at a slab plane need one
//    batch; the batch cuts of an over-full tile depend on rows the slab run does not hold, and the two
//    runs then agree to rounding only).
//  * Tiles with more candidates than a stage holds, or more targets than its target list, are split into
//    several ITEMS (target range x candidate batch); the items of a batch after the first ADD to the
//    rates already written (the producer publishes them only after the previous item has drained).
//  * No tensor cores in the pair term: it is not a contraction.
//
// FP32-ALU bound ("bound": "alu" in bench.py).
#include "sph_internal.cuh"
#include "interact_pair.cuh"

namespace sph {

#ifndef SPH_IM_CONSUMERS
#define SPH_IM_CONSUMERS 12
#endif
#ifndef SPH_IM_PRODUCERS
#define SPH_IM_PRODUCERS 4
#endif
#ifndef SPH_IM_SLEEP_NS
#define SPH_IM_SLEEP_NS 256
#endif
#ifndef SPH_IM_RB
#define SPH_IM_RB 9
#endif
constexpr int IM_NC = SPH_IM_CONSUMERS;      // consumer warps
constexpr int IM_NP = SPH_IM_PRODUCERS;       // producer warps
constexpr int IM_THREADS = 32 * (IM_NC + IM_NP);
#ifndef SPH_IM_MAXT
#define SPH_IM_MAXT 352
#endif
#ifndef SPH_IM_CAP
#define SPH_IM_CAP 2304
#endif
constexpr int IM_MAXT = SPH_IM_MAXT;                 // targets per item: 2 x 2 x 3 cells x 27 particles = 324
constexpr int IM_COLS = 16;                  // staged columns: 4 x 4
constexpr int IM_ZMAX = 6;                   // max cells per z-block (tf32 model: |z| <= (zb + 2) h)
constexpr int IM_CAP = SPH_IM_CAP;                 // staged record slots per batch = 36 blocks of 64
constexpr int IM_BATCH = IM_CAP - 128;       // particles per batch (16 x 5 x 27 = 2160): the 4 x-rows start at multiples
                                             // of 32 slots, which costs up to 4 x 31 padding slots
constexpr int IM_RB = SPH_IM_RB;             // mask ring: blocks of 64 candidates per warp per round
constexpr int IM_STAGES = 2;
#ifndef SPH_IM_PPS
#define SPH_IM_PPS 2
#endif
constexpr int IM_PPS = SPH_IM_PPS;           // pair slots per drain step (even): IM_PPS pops, IM_PPS / 2 packed pair terms
constexpr float IM_WIDE_N = -3.0e38f;        // |x|^2 stand-in of "wide" tiles: every real record is a hit
constexpr float IM_FAR = 1e15f;              // coordinate of the dummy partner: r2 = 3e30 is finite, shape = 0
constexpr float IM_TINY = 1e-30f;            // added to r2: a coincident pair (the particle itself) adds exactly 0
constexpr uint32_t IM_CTR_NTILES = 16, IM_CTR_NEXT = 17;    // words of sph_ctx::counters
static_assert(IM_CAP % 64 == 0 && IM_RB >= 2, "blocks of 64; the ring doubles as scratch for the A rows");
static_assert(IM_MAXT % 32 == 0, "chunks of 32 targets");

struct __align__(1024) ImStage {    // recA at a multiple of 1024 B: the slot swizzle is applied to shared ADDRESSES
    float4 recA[IM_CAP + 1];                 // x, y, z relative to the tile centre, p/rho^2; slot IM_CAP = dummy partner
    float4 recB[IM_CAP + 1];                 // vx, vy, vz, rho/rho0 (sign = boundary type if masses differ)
    float marr[IM_CAP + 4];                  // m_j = |x_j|^2 - thr, rounded to tf32
    uint32_t tglob[IM_MAXT];                 // targets of the item, ordered by (x-row, position inside the cell along x):
                                             // global index | own column << 28
    uint32_t row_astart[5];                  // slot of the first record of each staged x-row (multiple of 32); [4] = end
    uint32_t ntargets;
    uint32_t chunk_ctr;                      // next chunk of 32 targets
    uint32_t wide;                           // some record lies outside the tf32 error model
    uint32_t accumulate;                     // add to the rates already in memory (second and later batches)
    uint32_t exit;                           // no more work
    uint32_t first_chunk;                    // the chunk handed out first: the one whose targets lie in both x-rows of
                                             // the tile needs four candidate rows instead of three and takes longest
    float ox, oy, oz, bxy, bzz;              // tile origin and the bounds of the tf32 error model
};

struct __align__(1024) ImSmem {
    ImStage st[IM_STAGES];
    uint32_t mask[IM_NC][IM_RB * 64 + 32];   // per consumer warp and ring slot: [half][target lane] hit masks of 32 candidates;
                                             // + one row of empty words (the sentinel that ends every lane's word list)
    // producer-private
    uint32_t cbt[IM_COLS][IM_ZMAX + 3];      // cell_begin of the 16 columns over [zlo, zhi]
    uint32_t col_vstart[IM_COLS + 1];        // virtual start of each column in the concatenation
    uint32_t tstart[5], tbase[4], tcnt[4];   // target ranges of the 2 x 2 own columns
    uint32_t wcnt[IM_NP][32];                // target ordering: per producer warp and bucket, counts, then next slots
    uint32_t tkey[IM_MAXT];                  // target ordering: bucket | own column << 28
    uint32_t tidx[IM_MAXT];                  // target ordering: global index
    uint32_t tnext[IM_MAXT];                 // target list of the item being prepared
    uint32_t row_len[4];
    uint32_t tile;                           // the tile the producers work on
    unsigned long long full[IM_STAGES], empty[IM_STAGES], tma;
};

struct ImArgs {
    int zb, nzb;                             // cells per z-block, z-blocks per column
    int tx0, nty, ntx;                       // first x tile, tiles along y and x
    int cx_first, cx_end;                    // cell planes that hold the targets
    int cand_lo, cand_hi;                    // cell planes that exist in the arrays (per-slab execution), inclusive
    float thr2;                              // filter threshold, physical units
    const uint32_t *tile_list;               // non-empty tiles (ia_tile_list_kernel)
    uint32_t *ctr;                           // [IM_CTR_NTILES] = tiles listed, [IM_CTR_NEXT] = next tile to hand out
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
}
__device__ __forceinline__ void mbar_arrive(uint32_t mbar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mbar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t mbar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try(uint32_t mbar, uint32_t parity)
{
    uint32_t done;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(done) : "r"(mbar), "r"(parity) : "memory");
    return done != 0u;
}
// waiting warps must not take issue slots from the working ones.  SPH_IM_SUSPEND_NS > 0: the wait is left to
// the hardware - try_wait with a suspend-time hint parks the warp until the phase completes or the hint
// runs out, so a long wait costs a handful of instructions; 0: poll and sleep SPH_IM_SLEEP_NS in between.
#ifndef SPH_IM_SUSPEND_NS
#define SPH_IM_SUSPEND_NS 0
#endif
__device__ __forceinline__ void mbar_wait(uint32_t mbar, uint32_t parity)
{
#if SPH_IM_SUSPEND_NS > 0
    asm volatile("{\n\t.reg .pred p;\n\t"
                 "IM_WAIT_%=:\n\t"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n\t"
                 "@p bra IM_DONE_%=;\n\t"
                 "bra IM_WAIT_%=;\n\t"
                 "IM_DONE_%=:\n\t}"
                 ::"r"(mbar), "r"(parity), "r"((uint32_t)SPH_IM_SUSPEND_NS) : "memory");
#else
    while (!mbar_try(mbar, parity)) __nanosleep(SPH_IM_SLEEP_NS);
#endif
}
// 1-D bulk asynchronous copy global -> shared (SASS: UBLKCP); bytes % 16 == 0, both sides 16-byte aligned
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t mbar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(mbar) : "memory");
}
// the same range into L2 only
__device__ __forceinline__ void bulk_prefetch_l2(const void *src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
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

int interact_mma_targets() { return IM_MAXT; }
int interact_mma_zmax() { return IM_ZMAX; }

__device__ __forceinline__ void im_tile_coords(uint32_t b, const ImArgs &A, int &cx0, int &cy0, int &cz0)
{
    cz0 = (int)(b % (uint32_t)A.nzb) * A.zb;
    b /= (uint32_t)A.nzb;
    cy0 = (int)(b % (uint32_t)A.nty) * 2;
    cx0 = ((int)(b / (uint32_t)A.nty) + A.tx0) * 2;
}

// ---- list of the non-empty tiles (most of a dam-break tank holds no particle) ------------------------
// Listed z-block fastest, then y inside strips of IM_STRIP tiles, then x, then strip: tiles that share
// staged columns are handed out close in time, so the second reader of a column finds it in L2.
constexpr int IM_STRIP = 8;
__global__ void __launch_bounds__(256)
ia_tile_list_kernel(const uint32_t *__restrict__ cell_begin, GridC g, ImArgs A, uint32_t nthreads, uint32_t *list)
{
    uint32_t q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= nthreads) return;
    const uint32_t bz = q % (uint32_t)A.nzb;
    q /= (uint32_t)A.nzb;
    const uint32_t tyl = q % IM_STRIP;
    q /= IM_STRIP;
    const uint32_t tx = q % (uint32_t)A.ntx, strip = q / (uint32_t)A.ntx;
    const uint32_t ty = strip * IM_STRIP + tyl;
    if (ty >= (uint32_t)A.nty) return;
    const uint32_t b = (tx * (uint32_t)A.nty + ty) * (uint32_t)A.nzb + bz;
    int cx0, cy0, cz0;
    im_tile_coords(b, A, cx0, cy0, cz0);
    const int cz1 = min(cz0 + A.zb, g.nc[2]);
    uint32_t any = 0;
#pragma unroll
    for (int t = 0; t < 4; ++t) {
        const int x = cx0 + (t >> 1), y = cy0 + (t & 1);
        if (x >= A.cx_first && x < A.cx_end && y < g.nc[1]) {
            const uint32_t colbase = (uint32_t)(x * g.nc[1] + y) * g.nc[2];
            any |= cell_begin[colbase + cz1] - cell_begin[colbase + cz0];
        }
    }
    if (any) list[atomicAdd(A.ctr + IM_CTR_NTILES, 1u)] = b;     // approximate order: a tile's result does not depend on it
}

// ---- producers: IM_NP warps working as one group (named barrier 1) -----------------------------------
__device__ __forceinline__ void im_pbar()
{
    asm volatile("bar.sync 1, %0;" ::"n"(32 * IM_NP) : "memory");
}

template <bool UNIFORM>
__device__ __forceinline__ void im_produce(ImSmem &S, const float4 *__restrict__ pos4, const float4 *__restrict__ velrho4,
                                           const uint32_t *__restrict__ idt, const uint32_t *__restrict__ cell_begin,
                                           const GridC &g, const PhysC &ph, const ImArgs &A)
{
    const int ptid = threadIdx.x, lane = ptid & 31, pwarp = ptid >> 5;
    constexpr int PT = 32 * IM_NP;
    const uint32_t full_mask = 0xffffffffu;
    const uint32_t tma = (uint32_t)__cvta_generic_to_shared(&S.tma);
    const uint32_t ntiles = A.ctr[IM_CTR_NTILES];
    const float cell = 2.0f * ph.h;
    uint32_t it = 0, tma_phase = 0;

    while (true) {
        im_pbar();                                                   // the previous tile's tables are no longer read
        if (ptid == 0) S.tile = atomicAdd(A.ctr + IM_CTR_NEXT, 1u);
        im_pbar();
        uint32_t b = S.tile;
        if (b >= ntiles) break;
        b = A.tile_list[b];
        int cx0, cy0, cz0;
        im_tile_coords(b, A, cx0, cy0, cz0);
        const int cz1 = min(cz0 + A.zb, g.nc[2]);
        const int zlo = max(cz0 - 1, 0), zhi = min(cz1 + 1, g.nc[2]);
        const int nz = zhi - zlo;                                    // <= zb + 2

        // ---- the tile's piece of the cell table
        if (ptid < 4) {
            const int x = cx0 + (ptid >> 1), y = cy0 + (ptid & 1);
            uint32_t tb = 0, te = 0;
            if (x >= A.cx_first && x < A.cx_end && y < g.nc[1]) {
                const uint32_t colbase = (uint32_t)(x * g.nc[1] + y) * g.nc[2];
                tb = cell_begin[colbase + cz0];
                te = cell_begin[colbase + cz1];
            }
            S.tbase[ptid] = tb;
            S.tcnt[ptid] = te - tb;
        }
        for (int k = ptid; k < IM_COLS * (nz + 1); k += PT) {
            const int col = k / (nz + 1), z = k % (nz + 1);
            const int x = cx0 - 1 + (col >> 2), y = cy0 - 1 + (col & 3);
            uint32_t v = 0;
            if (x >= A.cand_lo && x <= A.cand_hi && y >= 0 && y < g.nc[1])
                v = cell_begin[(uint32_t)(x * g.nc[1] + y) * g.nc[2] + zlo + z];
            S.cbt[col][z] = v;                   // columns that do not exist: all 0 => empty ranges
        }
        im_pbar();
        if (pwarp == 0) {
            const uint32_t len = lane < IM_COLS ? S.cbt[lane][nz] - S.cbt[lane][0] : 0u;
            const uint32_t tcount = lane < 4 ? S.tcnt[lane] : 0u;
            uint32_t inc = len, tinc = tcount;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t t = __shfl_up_sync(full_mask, inc, o), u = __shfl_up_sync(full_mask, tinc, o);
                if (lane >= o) { inc += t; tinc += u; }
            }
            if (lane <= IM_COLS) S.col_vstart[lane] = inc - len;     // lane 16: the total
            if (lane <= 4) S.tstart[lane] = tinc - tcount;           // lane 4: the total
        }
        im_pbar();
        const uint32_t total = S.col_vstart[IM_COLS];
        const uint32_t ttotal = S.tstart[4];

        // tile-relative coordinates: origin = centre of the staged region.  |x|, |y| <= 4h and |z| <= nz h for
        // every particle that lies inside its cell - the range the tf32 error model (filter_thr) assumes; a
        // particle outside it (it left the grid and sits clamped in an edge cell, reading A13) switches the
        // filter off ("wide": every candidate passes, the drain decides).
        const float ox = fmaf((float)(cx0 + 1), cell, g.min[0]);
        const float oy = fmaf((float)(cy0 + 1), cell, g.min[1]);
        const float oz = fmaf((float)zlo + 0.5f * (float)nz, cell, g.min[2]);
        const float bxy = 2.0f * cell * 1.002f, bzz = 0.5f * (float)nz * cell * 1.002f;

        for (uint32_t t0 = 0; t0 < ttotal; t0 += IM_MAXT) {
            const uint32_t nT = min((uint32_t)IM_MAXT, ttotal - t0);
            for (uint32_t bstart = 0; bstart < total; bstart += IM_BATCH) {
                const uint32_t bend = min(total, bstart + IM_BATCH);
                const uint32_t s = it & 1u, use = it >> 1;
                ImStage &T = S.st[s];
                // ---- before the stage is free: order the targets by (x-row, position inside the cell along x), and
                // inside such a bucket by their sorted index (a STABLE counting sort: every producer warp ranks a
                // contiguous piece of the targets, so that bucket order = index order and the list is the same in
                // every run).  How many hits a target meets in each x-row of the staged region depends on where
                // it sits in its cell along x; the drain works row by row, so a warp whose lanes share that
                // position keeps all its lanes busy in every row.  The order of a target's own sum does not
                // depend on its lane.
                const uint32_t per = ((nT + IM_NP - 1) / IM_NP + 31u) & ~31u;          // targets per producer warp
                const uint32_t q_lo = (uint32_t)pwarp * per, q_hi = min(nT, q_lo + per);
                S.wcnt[pwarp][lane] = 0u;
                __syncwarp();
                for (uint32_t q = q_lo + lane; q < q_lo + per; q += 32) {
                    uint32_t bk = 64u + lane;                                           // no target: a key of its own
                    if (q < q_hi) {
                        const uint32_t tq = t0 + q;
                        int tc = 0;
#pragma unroll
                        for (int t = 1; t < 4; ++t) tc += (tq >= S.tstart[t]) ? 1 : 0;
                        const uint32_t i = S.tbase[tc] + (tq - S.tstart[tc]);
                        const float px = __ldg(reinterpret_cast<const float *>(pos4 + i)) - ox;    // column tc >> 1 spans
                        const float ph16 = (px - (float)((tc >> 1) - 1) * cell) * (16.0f / cell);     // [(tx-1) cell, tx cell)
                        bk = (uint32_t)(tc >> 1) * 16u + (uint32_t)min(max(__float2int_rd(ph16), 0), 15);
                        S.tkey[q] = bk | ((uint32_t)tc << 28);
                        S.tidx[q] = i;
                    }
                    const uint32_t m = __match_any_sync(full_mask, bk);
                    if (q < q_hi && (m & ((1u << lane) - 1u)) == 0u) S.wcnt[pwarp][bk] += (uint32_t)__popc(m);
                    __syncwarp();
                }
                im_pbar();
                if (pwarp == 0) {                     // lane = bucket: first slot of every (bucket, producer warp)
                    uint32_t run = 0;
                    uint32_t part[IM_NP];
#pragma unroll
                    for (int w = 0; w < IM_NP; ++w) { part[w] = run; run += S.wcnt[w][lane]; }
                    uint32_t inc = run;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const uint32_t t = __shfl_up_sync(full_mask, inc, o);
                        if (lane >= o) inc += t;
                    }
#pragma unroll
                    for (int w = 0; w < IM_NP; ++w) S.wcnt[w][lane] = inc - run + part[w];
                }
                im_pbar();
                for (uint32_t q = q_lo + lane; q < q_lo + per; q += 32) {
                    const uint32_t k = q < q_hi ? S.tkey[q] : 0u;
                    const uint32_t bk = q < q_hi ? (k & 31u) : 64u + lane;
                    const uint32_t m = __match_any_sync(full_mask, bk);
                    const uint32_t below = (uint32_t)__popc(m & ((1u << lane) - 1u));
                    if (q < q_hi) S.tnext[S.wcnt[pwarp][bk] + below] = S.tidx[q] | (k & 0x30000000u);
                    __syncwarp();
                    if (q < q_hi && below == 0u) S.wcnt[pwarp][bk] += (uint32_t)__popc(m);
                    __syncwarp();
                }
                // ... and pull the item's records into L2, so that the bulk copies issued once the stage is free
                // do not wait for HBM
                if (ptid < IM_COLS) {
                    const uint32_t vs = S.col_vstart[ptid], ve = S.col_vstart[ptid + 1];
                    const uint32_t lo = max(vs, bstart), hi = min(ve, bend);
                    if (lo < hi) {
                        const uint32_t gl = S.cbt[ptid][0] + (lo - vs);
                        bulk_prefetch_l2(pos4 + gl, 16u * (hi - lo));
                        bulk_prefetch_l2(velrho4 + gl, 16u * (hi - lo));
                    }
                }
                mbar_wait((uint32_t)__cvta_generic_to_shared(&S.empty[s]), (use & 1u) ^ 1u);
                // a later batch adds to what the previous item wrote: wait until that item has drained
                if (bstart > 0) mbar_wait((uint32_t)__cvta_generic_to_shared(&S.empty[s ^ 1u]), ((it - 1u) >> 1) & 1u);
                const uint32_t recA_addr = (uint32_t)__cvta_generic_to_shared(T.recA);
                const uint32_t recB_addr = (uint32_t)__cvta_generic_to_shared(T.recB);

                // ---- slots of this batch: x-row r starts at a multiple of 32 (a target's window of three rows
                // is then a whole number of 32-candidate mask words)
                if (ptid == 0) {
                    uint32_t a = 0;
                    for (int r = 0; r < 4; ++r) {
                        const uint32_t lo = min(max(S.col_vstart[4 * r], bstart), bend);
                        const uint32_t hi = min(max(S.col_vstart[4 * r + 4], bstart), bend);
                        T.row_astart[r] = a;
                        S.row_len[r] = hi - lo;
                        a = (a + (hi - lo) + 31u) & ~31u;
                    }
                    T.row_astart[4] = a;
                    T.ntargets = nT;
                    T.chunk_ctr = 0u;
                    T.wide = 0u;
                    T.accumulate = bstart > 0 ? 1u : 0u;
                    T.exit = 0u;
                    {
                        const uint32_t n0 = min(max(S.tstart[2], t0), t0 + nT) - t0;      // targets of the first x-row
                        T.first_chunk = (n0 & 31u) && n0 < nT ? n0 >> 5 : 0u;
                    }
                    T.ox = ox; T.oy = oy; T.oz = oz; T.bxy = bxy; T.bzz = bzz;
                    mbar_arrive_expect_tx(tma, (bend - bstart) * 32u);
                }
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");    // generic writes of the last use < bulk copies
                im_pbar();
                // ---- stage: one bulk copy per column and array, all completing on the mbarrier
                if (ptid < IM_COLS) {
                    const int r = ptid >> 2;
                    const uint32_t vs = S.col_vstart[ptid], ve = S.col_vstart[ptid + 1];
                    const uint32_t lo = max(vs, bstart), hi = min(ve, bend);
                    const uint32_t rlo = min(max(S.col_vstart[4 * r], bstart), bend);    // first particle of the row in the batch
                    if (lo < hi) {
                        const uint32_t gl = S.cbt[ptid][0] + (lo - vs);
                        const uint32_t a = T.row_astart[r] + (lo - rlo);
                        bulk_g2s(recA_addr + 16u * a, pos4 + gl, 16u * (hi - lo), tma);
                        bulk_g2s(recB_addr + 16u * a, velrho4 + gl, 16u * (hi - lo), tma);
                    }
                }
                // ---- the target list, prepared before the stage was acquired
                for (uint32_t q = ptid; q < nT; q += PT) T.tglob[q] = S.tnext[q];
                mbar_wait(tma, tma_phase);
                tma_phase ^= 1u;
                // ---- convert in place: tile-relative coordinates, m = |x|^2 - thr (tf32), rho -> rho/rho0; the
                // padding slots between the rows and up to the next block of 64 become records that never hit
                const uint32_t aend = T.row_astart[4];
                const uint32_t nconv = (aend + 63u) & ~63u;
                uint32_t wide = 0u;
                for (uint32_t a0 = 64u * (uint32_t)pwarp; a0 < nconv; a0 += 64u * IM_NP) {
                    float4 ra[2], rb[2];
                    float m[2];
#pragma unroll
                    for (int u = 0; u < 2; ++u) {
                        const uint32_t a = a0 + 32u * u + lane;
                        int r = 0;
#pragma unroll
                        for (int q = 1; q < 4; ++q) r += (a >= T.row_astart[q]) ? 1 : 0;
                        const uint32_t k = a - T.row_astart[r];
                        ra[u] = make_float4(0.f, 0.f, 0.f, 0.f);
                        rb[u] = make_float4(0.f, 0.f, 0.f, 1.f);
                        m[u] = __int_as_float(0x7f800000);                        // +inf: D > 0 against any target
                        if (a < aend && k < S.row_len[r]) {
                            ra[u] = T.recA[a];
                            rb[u] = T.recB[a];
                            ra[u].x -= ox; ra[u].y -= oy; ra[u].z -= oz;
                            if (!(fabsf(ra[u].x) <= bxy && fabsf(ra[u].y) <= bxy && fabsf(ra[u].z) <= bzz)) wide = 1u;
                            m[u] = tf32_rna(fmaf(ra[u].z, ra[u].z, fmaf(ra[u].y, ra[u].y, ra[u].x * ra[u].x)) - A.thr2);
                            rb[u].w *= ph.inv_rho0;
                            if (!UNIFORM) {
                                const uint32_t vv = min(max(S.col_vstart[4 * r], bstart), bend) + k;   // index in the concatenation
                                int col = 0;
#pragma unroll
                                for (int q = 1; q < IM_COLS; ++q) col += (vv >= S.col_vstart[q]) ? 1 : 0;
                                const uint32_t j = S.cbt[col][0] + (vv - S.col_vstart[col]);
                                if (__ldg(idt + j) & TYPE_BIT) rb[u].w = -rb[u].w;
                            }
                        }
                    }
                    __syncwarp();                                // the 32 lanes cover aligned runs of 32 slots
#pragma unroll
                    for (int u = 0; u < 2; ++u) {
                        const uint32_t a = a0 + 32u * u + lane;
                        const uint32_t sw = a ^ ((a >> 3) & 6u);     // swizzle: the 8 records of an mma B fragment (slots
                        T.recA[sw] = ra[u];                          // 2j + c + 16 q') fall on 8 different 16-byte bank groups
                        T.recB[sw] = rb[u];
                        T.marr[sw] = m[u];
                    }
                }
                if (__any_sync(full_mask, wide != 0u) && lane == 0) T.wide = 1u;
                im_pbar();
                if (ptid == 0) mbar_arrive((uint32_t)__cvta_generic_to_shared(&S.full[s]));
                ++it;
            }
        }
    }
    // ---- no more work
    {
        const uint32_t s = it & 1u, use = it >> 1;
        mbar_wait((uint32_t)__cvta_generic_to_shared(&S.empty[s]), (use & 1u) ^ 1u);
        if (ptid == 0) {
            S.st[s].exit = 1u;
            mbar_arrive((uint32_t)__cvta_generic_to_shared(&S.full[s]));
        }
    }
}

// ---- consumer: one chunk of 32 targets against the stage --------------------------------------------
template <int KERNEL, bool UNIFORM, bool GAMMA7, bool MU>
__device__ __forceinline__ void im_chunk(ImStage &T, uint32_t mwarp, uint32_t chunk,
                                         const float4 *__restrict__ pos4, const float4 *__restrict__ velrho4,
                                         const uint32_t *__restrict__ idt, float4 *__restrict__ acc4,
                                         float *__restrict__ mu_out, const PhysC &ph)
{
    const int lane = threadIdx.x & 31;
    const uint32_t full_mask = 0xffffffffu;
    const int g8 = lane >> 2, qd = lane & 3;
    const uint32_t recA_addr = (uint32_t)__cvta_generic_to_shared(T.recA);
    const uint32_t recB_addr = (uint32_t)__cvta_generic_to_shared(T.recB);
    const uint32_t marr_addr = (uint32_t)__cvta_generic_to_shared(T.marr);
    const uint32_t ab_delta = recB_addr - recA_addr;
    const uint32_t dummy_addr = recA_addr + 16u * (uint32_t)IM_CAP;

    // constants of the pair term (the packed instructions take a scalar operand for both lanes)
    const float kvisc = -ph.alpha_h * ph.c0 * ph.inv_rho0;       // Pi_ij = kvisc * poly * min(v.r, 0) / (r2 + eta2)
    const f2 c_tiny = pk(IM_TINY, IM_TINY), c_eta2 = pk(ph.eta2, ph.eta2);
    const f2 c_mih = pk(-ph.inv_h_half, -ph.inv_h_half), c_one = pk(1.0f, 1.0f), c_kv = pk(kvisc, kvisc);
    const float cexp = 0.5f * (float)(ph.gamma - 1);

    const uint32_t tq = chunk * 32u + (uint32_t)lane;
    const bool active = tq < T.ntargets;
    const uint32_t pe = active ? T.tglob[tq] : 0u;
    const uint32_t i = pe & 0x0FFFFFFFu;
    const int tx = (int)(pe >> 29);
    float4 pi = make_float4(T.ox, T.oy, T.oz, 0.f), vi = make_float4(0.f, 0.f, 0.f, ph.rho0);
    bool fluid = false;
    if (active) {
        pi = pos4[i];
        vi = velrho4[i];
        fluid = (idt[i] & TYPE_BIT) == 0;
    }
    const float xi = pi.x - T.ox, yi = pi.y - T.oy, zi = pi.z - T.oz;
    const bool out = active && !(fabsf(xi) <= T.bxy && fabsf(yi) <= T.bxy && fabsf(zi) <= T.bzz);
    const bool wide = __any_sync(full_mask, out) || T.wide != 0u;
    const float ui = vi.w * ph.inv_rho0;
    const float ui2 = GAMMA7 ? ui * ui : __powf(ui, cexp);   // gamma = 7: u^2; else u^((gamma-1)/2)
    // x-rows of the staged region this warp's targets need: [txmin, txmax + 2]
    const int txmin = __reduce_min_sync(full_mask, active ? tx : 2);
    const int txmax = __reduce_max_sync(full_mask, active ? tx : -1);
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

    if (txmax >= 0) {
        // ---- A rows of the distance product, handed to the lanes that hold them as mma fragments.
        // "wide" tiles: D = m - 3e38 < 0 for every real record, +inf for the padding slots.
        uint32_t af[4];
        float nf[4];
        {
            const uint32_t scratch = mwarp;                      // the mask ring doubles as scratch
            float4 row = make_float4(-2.0f * xh, -2.0f * yh, -2.0f * zh, nn);
            if (wide) row = make_float4(0.f, 0.f, 0.f, IM_WIDE_N);
            if (!active) row = make_float4(0.f, 0.f, 0.f, __int_as_float(0x7f800000));
            asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(scratch + 16u * (uint32_t)lane), "f"(row.x), "f"(row.y),
                         "f"(row.z), "f"(row.w) : "memory");
            __syncwarp();
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const float4 r = im_lds_f4(scratch + 16u * (uint32_t)(g8 + 8 * k));
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
            const uint32_t e0 = T.row_astart[r] >> 5, e1 = T.row_astart[r + 1] >> 5;     // mask words of the row
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
                // atop = shared address of recA[slot of bit 0 of cur] (bit hb is 16 hb bytes below it);
                // nxtw / nxta = the next non-empty word and its atop, fetched when the current word was taken,
                // so that no shared-memory load sits on the chain from one pop to the next
                uint32_t cur = odd ? 1u : 0u;
                uint32_t atop = dummy_addr;
                const uint32_t steps = __reduce_max_sync(full_mask, tot ? (tot + odd + (uint32_t)(IM_PPS - 1)) / (uint32_t)IM_PPS : 0u);
                odd = (odd + tot) & 1u;
                const uint32_t atop0 = recA_addr + 16u * (rb0 * 64u + 32u * 31u + 31u);   // word k: atop0 - 512 (31 - k)
                const uint32_t mtop = mlane + 128u * 31u;                                   // word k at mtop - 128 (31 - k)
                // the word after the ring's last one is always empty: its bit stays in nz, so that a lane that has
                // used up its words keeps fetching an empty word (no test for "none left" in the pop)
                constexpr uint32_t sent = 0x80000000u >> (2 * IM_RB);
                nz |= sent;
                uint32_t nxtw, nxta;
                {
                    const uint32_t kb = bfind(nz);                                      // highest bit = lowest word
                    nxtw = im_lds_u32(mtop - 128u * kb);
                    nxta = atop0 - 512u * kb;
                    nz = (nz & ~(1u << kb)) | sent;
                }
                // branch-free: the word after next is read in any case
                auto pop = [&]() -> uint32_t {
                    const uint32_t kb = bfind(nz);
                    const uint32_t w = im_lds_u32(mtop - 128u * kb);
                    const bool take = cur == 0u;
                    cur = take ? nxtw : cur;
                    atop = take ? nxta : atop;
                    nxtw = take ? w : nxtw;
                    nxta = take ? atop0 - 512u * kb : nxta;
                    nz = take ? (nz & ~(1u << kb)) | sent : nz;
                    const uint32_t hb = bfind(cur);                                     // 0xFFFFFFFF if cur == 0
                    const uint32_t lin = cur ? atop - 16u * hb : dummy_addr;
                    cur &= ~(1u << (hb & 31u));
                    return lin ^ ((lin >> 3) & 0x60u);                                  // slot swizzle, in bytes
                };
                // software pipeline: the addresses of step st + 1 are popped before the pairs of step st are evaluated
                uint32_t cs[IM_PPS];
#pragma unroll
                for (int q = 0; q < IM_PPS; ++q) cs[q] = pop();
                // two steps per iteration (independent chains for the scheduler), a single one if the count is odd
                uint32_t st = 0;
                for (; st + 1u < steps; st += 2u) {
                    uint32_t n1[IM_PPS], n2[IM_PPS];                                    // past the last hit: dummy partners
#pragma unroll
                    for (int q = 0; q < IM_PPS; ++q) n1[q] = pop();
#pragma unroll
                    for (int q = 0; q < IM_PPS; ++q) n2[q] = pop();
#pragma unroll
                    for (int q = 0; q < IM_PPS; q += 2) pair2(cs[q], cs[q + 1]);
#pragma unroll
                    for (int q = 0; q < IM_PPS; q += 2) pair2(n1[q], n1[q + 1]);
#pragma unroll
                    for (int q = 0; q < IM_PPS; ++q) cs[q] = n2[q];
                }
                if (st < steps) {
#pragma unroll
                    for (int q = 0; q < IM_PPS; q += 2) pair2(cs[q], cs[q + 1]);
                }
                __syncwarp();
            }
        }
    }
    if (active) {
        float a0, a1, b0, b1, c0, c1, d0, d1;
        upk(ax2, a0, a1); upk(ay2, b0, b1); upk(az2, c0, c1); upk(dr2, d0, d1);
        const float k = UNIFORM ? ph.kF * ph.mass_fluid : ph.kF;
        float ax = -k * (a0 + a1), ay = -k * (b0 + b1), az = -k * (c0 + c1);
        float dr = k * (d0 + d1);
        if (T.accumulate) {                      // a later batch of the tile's candidates
            const float4 o = acc4[i];
            ax += o.x; ay += o.y; az += o.z; dr += o.w;
            if (MU) mumax = fmaxf(mumax, mu_out[i]);
        } else if (fluid) {
            ax += ph.g[0]; ay += ph.g[1]; az += ph.g[2];
        }
        if (!fluid) ax = ay = az = 0.f;
        acc4[i] = make_float4(ax, ay, az, dr);
        if (MU) mu_out[i] = mumax;
    }
}

template <int KERNEL, bool UNIFORM, bool GAMMA7, bool MU>
__global__ void __launch_bounds__(IM_THREADS, 1)
interact_mma_kernel(const float4 *__restrict__ pos4, const float4 *__restrict__ velrho4,
                    const uint32_t *__restrict__ idt, const uint32_t *__restrict__ cell_begin,
                    float4 *__restrict__ acc4, float *__restrict__ mu_out, GridC g, PhysC ph, ImArgs A)
{
    extern __shared__ __align__(1024) unsigned char im_raw[];
    ImSmem &S = *reinterpret_cast<ImSmem *>(im_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    for (int k = tid; k < IM_NC * 32; k += IM_THREADS) S.mask[k >> 5][IM_RB * 64 + (k & 31)] = 0u;
    if (tid == 0) {
        for (int s = 0; s < IM_STAGES; ++s) {
            mbar_init((uint32_t)__cvta_generic_to_shared(&S.full[s]), 1u);
            mbar_init((uint32_t)__cvta_generic_to_shared(&S.empty[s]), (uint32_t)IM_NC);
            S.st[s].recA[IM_CAP] = make_float4(IM_FAR, IM_FAR, IM_FAR, 0.f);
            S.st[s].recB[IM_CAP] = make_float4(0.f, 0.f, 0.f, 1.f);
        }
        mbar_init((uint32_t)__cvta_generic_to_shared(&S.tma), 1u);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp < IM_NP) {
        im_produce<UNIFORM>(S, pos4, velrho4, idt, cell_begin, g, ph, A);
        return;
    }
    const uint32_t mwarp = (uint32_t)__cvta_generic_to_shared(&S.mask[warp - IM_NP][0]);
    for (uint32_t it = 0;; ++it) {
        const uint32_t s = it & 1u;
        ImStage &T = S.st[s];
        mbar_wait((uint32_t)__cvta_generic_to_shared(&S.full[s]), (it >> 1) & 1u);
        if (T.exit) break;
        const uint32_t nchunks = (T.ntargets + 31u) >> 5;
        while (true) {
            uint32_t c = 0;
            if (lane == 0) c = atomicAdd(&T.chunk_ctr, 1u);
            c = __shfl_sync(0xffffffffu, c, 0);
            if (c >= nchunks) break;
            const uint32_t fc = T.first_chunk;
            c = c == 0u ? fc : (c <= fc ? c - 1u : c);
            im_chunk<KERNEL, UNIFORM, GAMMA7, MU>(T, mwarp, c, pos4, velrho4, idt, acc4, mu_out, ph);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive((uint32_t)__cvta_generic_to_shared(&S.empty[s]));
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
    A.ntx = ((A.cx_end - 1) >> 1) - A.tx0 + 1;
    A.nty = (c->grid.nc[1] + 1) >> 1;
    A.thr2 = filter_thr(A.zb) * c->phys.h * c->phys.h;
    A.tile_list = c->ia_tiles;
    A.ctr = c->counters;
    const uint64_t tiles = (uint64_t)A.ntx * A.nty * A.nzb;
    if (tiles == 0) return cudaSuccess;
    const uint32_t *cb = ov.on ? ov.cell_begin : c->cell_begin;
    cudaError_t e = cudaMemsetAsync(c->counters + IM_CTR_NTILES, 0, 2 * sizeof(uint32_t), c->stream);
    if (e != cudaSuccess) return e;
    const uint64_t lthreads = (uint64_t)((A.nty + IM_STRIP - 1) / IM_STRIP) * A.ntx * IM_STRIP * A.nzb;
    ia_tile_list_kernel<<<(uint32_t)((lthreads + 255) / 256), 256, 0, c->stream>>>(cb, c->grid, A, (uint32_t)lthreads, c->ia_tiles);
    c->n_launches++;
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const uint32_t grid = (uint32_t)(tiles < (uint64_t)c->num_sms ? tiles : (uint64_t)c->num_sms);
    kern<<<grid, IM_THREADS, sizeof(ImSmem), c->stream>>>(
        ov.on ? ov.pos4 : c->pos4[c->cur], ov.on ? ov.velrho4 : c->velrho4[c->cur], ov.on ? ov.idt : c->idt[c->cur],
        cb, ov.on ? ov.acc4 : c->acc4, c->mumax, c->grid, c->phys, A);
    c->n_launches++;
    return cudaGetLastError();
}

// capacity of the tile list for a grid and z-block
size_t interact_mma_tile_capacity(const int nc[3], int zb)
{
    return (size_t)((nc[0] + 1) / 2 + 1) * (size_t)((nc[1] + 1) / 2) * (size_t)((nc[2] + zb - 1) / zb);
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
