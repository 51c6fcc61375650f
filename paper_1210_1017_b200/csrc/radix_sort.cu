// a2 - onesweep-style least-significant-digit radix sort of (keyword, value) pairs on the low
// cell_bits of the keyword ("using the radix sort algorithm [18] to order the
// array holding the particle identification labels, or IDs, according to the cell"; the paper's
// three sorts per step - migration label L200, edge label L214, cell L220 - are one sort here,
// the labels ride in the keyword's top bits).
//
// One kernel per 8-bit digit.  The digit histograms come from the key kernel (keys.cu); each
// pass is a single sweep: a CTA takes a tile in launch order (dynamic tile id), ranks its keys
// with a warp-level match built in shared memory (one atomic OR per key) + per-warp
// shared-memory counters (stable), publishes its 256 digit
// counts, resolves the exclusive prefix over earlier tiles by decoupled look-back, reorders the
// tile through shared memory and writes runs of equal digits to consecutive addresses.
//
// HBM-bound: 8 B read + 8 B written per pair per pass.
#include "sph_internal.cuh"

namespace sph {

#ifndef SPH_RS_THREADS                            // tuning knobs (nvcc -D...), defaults = measured best
#define SPH_RS_THREADS 256
#endif
#ifndef SPH_RS_IPT
#define SPH_RS_IPT 32
#endif
#ifndef SPH_RS_MINBLOCKS
#define SPH_RS_MINBLOCKS 2
#endif
constexpr int RS_THREADS = SPH_RS_THREADS;        // >= 256 (one thread per digit)
constexpr int RS_IPT = SPH_RS_IPT;                // pairs per thread (even)
constexpr int RS_TILE = RS_THREADS * RS_IPT;      // 8192 pairs = 64 KB staged
constexpr int RS_WARPS = RS_THREADS / 32;
constexpr int RS_UNITS = RS_THREADS / 16;         // ranking units: half-warps (16-bit masks, 32-bit table entries)
constexpr int RS_LB = 8;                          // look-back polls in flight per thread
constexpr uint32_t LB_AGG = 1u << 30;             // look-back word: flag in bits 30..31
constexpr uint32_t LB_INC = 2u << 30;
constexpr uint32_t LB_VAL = (1u << 30) - 1u;

// Phase clocks of a tile (thread 0 of every CTA), summed over tiles: only in builds with -DSPH_RS_PROFILE
// (a measurement harness that includes this file and reads rs_prof); the product library is built without
// it.  Round-3 figures at 2^26 random keys, cycles per tile as thread 0 sees them: load 1900, rank 7200,
// counts + publish + scans 2400, reorder 4000, look-back 5200 + 900, scatter 3100.
#ifdef SPH_RS_PROFILE
__device__ unsigned long long rs_prof[8];
#define RS_MARK(k)                                                                     \
    do {                                                                               \
        if (threadIdx.x == 0) {                                                        \
            const long long now__ = clock64();                                         \
            atomicAdd(&rs_prof[k], (unsigned long long)(now__ - rs_t__));              \
            rs_t__ = now__;                                                            \
        }                                                                              \
    } while (0)
#define RS_MARK_INIT long long rs_t__ = clock64()
#else
#define RS_MARK(k) do { } while (0)
#define RS_MARK_INIT do { } while (0)
#endif

uint32_t radix_tiles(uint64_t n) { return (uint32_t)((n + RS_TILE - 1) / RS_TILE); }

__device__ __forceinline__ uint32_t ld_relaxed(const uint32_t *p)
{
    uint32_t v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed(uint32_t *p, uint32_t v)
{
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

struct __align__(16) RsSmem {
    uint2 stage[RS_TILE];                 // 64 KB
    uint32_t hw[RS_UNITS][256];           // 16 KB: per half-warp and digit, low 16 bits = match mask of the row
                                          // being ranked (scratch, 0 between rows), high 16 = running count
    uint32_t gbase[256];                  // global slot of tile-local slot 0 of each digit
    uint32_t scan_tmp[16];
    uint32_t tile;
};

// Stable ranking of one row of a half-warp (16 items, one per lane) on an 8-bit digit.  The set of
// lanes holding the same digit is built in shared memory: every lane ORs its bit into the (unit, digit)
// word - OR commutes, so the result does not depend on the order in which the hardware serialises
// lanes that hit the same word - and reads the word back: low half = the set, high half = the running
// count of that digit in earlier rows of the unit.  One ATOMS + one LDS + one STS, all 32-bit (random
// digits spread over all 32 banks), replace the eight ballots (about 50 ALU-pipe instructions) of a
// register-only match.  Both half-warps of a warp work on their own tables in the same instructions.
__device__ __forceinline__ uint32_t rank_row(uint32_t table /* shared address of S.hw[unit] */, uint32_t d,
                                             uint32_t bit16, uint32_t lt16)
{
    const uint32_t e = table + 4u * d;
    uint32_t w;
    asm volatile("red.shared.or.b32 [%0], %1;" ::"r"(e), "r"(bit16) : "memory");
    __syncwarp();
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(w) : "r"(e) : "memory");
    __syncwarp();
    const uint32_t m = w & 0xFFFFu, cnt = w >> 16;
    const uint32_t below = m & lt16;
    if (below == 0)                                                    // lowest lane of the set
        asm volatile("st.shared.u32 [%0], %1;" ::"r"(e), "r"((cnt + __popc(m)) << 16) : "memory");
    __syncwarp();
    return cnt + __popc(below);
}

template <bool FULL>
__device__ __forceinline__ void onesweep_tile(RsSmem &S, uint32_t n, const uint2 *__restrict__ in,
                                              uint2 *__restrict__ out, const uint32_t *__restrict__ hist,
                                              uint32_t *tile_state, int shift, uint32_t dmask, uint32_t tile)
{
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t unit = tid >> 4, lane16 = tid & 15u;
    const uint32_t bit16 = 1u << lane16, lt16 = bit16 - 1u;
    const uint32_t base = tile * RS_TILE;
    const uint32_t tile_n = FULL ? (uint32_t)RS_TILE : n - base;
    RS_MARK_INIT;
    const uint32_t hcount_pre = hist[tid & 255u];       // whole-array count of this thread's digit: needed only
                                                        // after the ranking, fetched now so that nobody waits for it
                                                        // between two barriers (1200 cycles per tile in the
                                                        // instrumented harness; no gain in the product build)

    // ---- load, striped per half-warp: the unit owns a contiguous chunk; item k of its lane l is
    // chunk[k*16+l], so that (unit, row, lane) order is index order.
    // Slots past the end of the array hold the key 0xFFFFFFFF: its digit is dmask, the largest digit
    // of the pass, and a stable ranking puts those slots after every real pair of the tile, i.e. at
    // staged positions >= tile_n, which are never written out.
    uint2 kv[RS_IPT];
    const uint32_t ubase = unit * (16 * RS_IPT);
#pragma unroll
    for (int k = 0; k < RS_IPT; ++k) {
        const uint32_t li = ubase + k * 16 + lane16;
        kv[k] = (FULL || li < tile_n) ? __ldcs(in + base + li) : make_uint2(0xFFFFFFFFu, 0u);
    }
#ifdef SPH_RS_PROFILE
    if (kv[RS_IPT - 1].x == 0x12345678u && kv[0].y == 0x9ABCDEF0u) rs_prof[7] = 1;      // wait for the loads
#endif
    RS_MARK(0);                                                                          // load
    // ---- rank inside the warp, stable in item order; two 16-bit ranks per register
    uint32_t rank2[RS_IPT / 2];
    const uint32_t tab_addr = (uint32_t)__cvta_generic_to_shared(S.hw[unit]);
    const uint32_t *tab = S.hw[unit];
#pragma unroll
    for (int k = 0; k < RS_IPT; ++k) {
        const uint32_t d = (kv[k].x >> shift) & dmask;
        const uint32_t r = rank_row(tab_addr, d, bit16, lt16);
        if (k & 1) rank2[k >> 1] |= r << 16; else rank2[k >> 1] = r;
    }
    __syncthreads();
    RS_MARK(1);                                                                          // rank

    // ---- per digit (threads 0..255): counts over warps, publish the tile aggregate at once, and
    // put the first round of look-back polls in flight; their latency (and the predecessors'
    // progress) overlaps the local scan and the shared-memory reordering below
    uint32_t count = 0, exc_in_warp = 0, hexc_in_warp = 0;
    uint32_t poll[RS_LB];
    uint32_t *st = tile_state + (size_t)tile * 256 + (tid & 255);
    if (tid < 256) {
#pragma unroll
        for (int u = 0; u < RS_UNITS; ++u) {
            const uint32_t t = S.hw[u][tid] >> 16;
            S.hw[u][tid] = count;                                   // from here on: plain 32-bit bases
            count += t;
        }
        const uint32_t pads = FULL ? 0u : (tid == dmask ? (uint32_t)RS_TILE - tile_n : 0u);
        const uint32_t pub = count - pads;                         // real pairs of this digit in the tile
        st_relaxed(st, (tile == 0 ? LB_INC : LB_AGG) | pub);
#pragma unroll
        for (int b = 0; b < RS_LB; ++b)
            poll[b] = ((int)tile - 1 - b >= 0) ? ld_relaxed(st - (size_t)(b + 1) * 256) : LB_INC;

        uint32_t inc = count;                                       // tile counts over digits
        uint32_t hcount = hcount_pre, hinc = hcount;                // whole-array counts over digits
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            uint32_t u = __shfl_up_sync(0xffffffffu, hinc, o);
            if (lane >= (uint32_t)o) { inc += t; hinc += u; }
        }
        if (lane == 31) { S.scan_tmp[warp] = inc; S.scan_tmp[8 + warp] = hinc; }
        exc_in_warp = inc - count;
        hexc_in_warp = hinc - hcount;
        count = pub;
    }
    __syncthreads();
    if (tid < 256) {
        uint32_t dstart = 0, hadd = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) {
            dstart += (w < (int)warp) ? S.scan_tmp[w] : 0u;
            hadd += (w < (int)warp) ? S.scan_tmp[8 + w] : 0u;
        }
        dstart += exc_in_warp;
        S.gbase[tid] = hexc_in_warp + hadd - dstart;    // + look-back, added below
        // fold the digit's first slot into the per-warp bases: one look-up per pair in the reorder
#pragma unroll
        for (int u = 0; u < RS_UNITS; ++u) S.hw[u][tid] += dstart;
    }
    __syncthreads();
    RS_MARK(2);                                                                          // counts, publish, scans

    // ---- reorder the tile through shared memory (needs only tile-local offsets)
#pragma unroll
    for (int k = 0; k < RS_IPT; ++k) {
        const uint32_t d = (kv[k].x >> shift) & dmask;
        const uint32_t r = (k & 1) ? (rank2[k >> 1] >> 16) : (rank2[k >> 1] & 0xFFFFu);
        S.stage[tab[d] + r] = kv[k];
    }

    RS_MARK(3);                                                                          // reorder (thread 0's share)
    // ---- finish the look-back: same digit in earlier tiles, RS_LB polls per round.  (Rounds of 16, 32 or 64
    // polls were measured in round 3 and are slower, 2746 / 2673 / 2464 against 2810 GB/s: the wait is for
    // predecessors that have not published yet, not for the number of words to add up.)
    if (tid < 256) {
        uint32_t lookback = 0;
        if (tile > 0) {
            int t = (int)tile - 1;
            bool done = false;
            while (true) {
                bool open = true;                                   // no unpublished predecessor met yet
#pragma unroll
                for (int b = 0; b < RS_LB; ++b) {
                    const uint32_t f = poll[b] >> 30;
                    open = open && (f != 0) && !done;
                    if (open) {
                        lookback += poll[b] & LB_VAL;
                        --t;
                        done = (f == 2);
                    }
                }
                if (done) break;
#pragma unroll
                for (int b = 0; b < RS_LB; ++b)
                    poll[b] = (t - b >= 0) ? ld_relaxed(tile_state + (size_t)(t - b) * 256 + tid) : LB_INC;
            }
            st_relaxed(st, LB_INC | (lookback + count));
        }
        S.gbase[tid] += lookback;
    }
    RS_MARK(4);                                                                          // look-back of digit 0
    __syncthreads();
    RS_MARK(5);                                                                          // ... of the slowest digit, reorder of the slowest warp
    // ---- runs of equal digits go to consecutive global addresses
#pragma unroll
    for (int k = 0; k < RS_IPT; ++k) {
        const uint32_t i = tid + k * RS_THREADS;
        if (FULL || i < tile_n) {
            const uint2 e = S.stage[i];
            const uint32_t d = (e.x >> shift) & dmask;
            out[S.gbase[d] + i] = e;
        }
    }
    RS_MARK(6);                                                                          // scatter (issue)
}

__global__ void __launch_bounds__(RS_THREADS, SPH_RS_MINBLOCKS)
onesweep_kernel(uint32_t n, const uint2 *__restrict__ in, uint2 *__restrict__ out,
                const uint32_t *__restrict__ hist, uint32_t *tile_state, uint32_t *tile_counter, int shift,
                uint32_t dmask /* keeps the tag bits 28..31 out of the last digit */)
{
    extern __shared__ __align__(16) unsigned char rs_raw[];
    RsSmem &S = *reinterpret_cast<RsSmem *>(rs_raw);
    const uint32_t tid = threadIdx.x;
    if (tid == 0) S.tile = atomicAdd(tile_counter, 1u);
    {
        uint4 *z = reinterpret_cast<uint4 *>(&S.hw[0][0]);
        for (int k = tid; k < RS_UNITS * 256 / 4; k += RS_THREADS) z[k] = make_uint4(0u, 0u, 0u, 0u);
    }
    __syncthreads();
    const uint32_t tile = S.tile;
    if ((uint64_t)(tile + 1) * RS_TILE <= n) onesweep_tile<true>(S, n, in, out, hist, tile_state, shift, dmask, tile);
    else onesweep_tile<false>(S, n, in, out, hist, tile_state, shift, dmask, tile);
}

// per-device attribute, set by sph_init for every new context
cudaError_t configure_sort()
{
    return cudaFuncSetAttribute(onesweep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(RsSmem));
}

cudaError_t launch_sort(sph_ctx *c)
{
    uint32_t n = (uint32_t)c->n;
    c->kv_sorted = c->passes & 1;
    if (n == 0) return cudaSuccess;
    uint32_t tiles = c->rs_tiles;
    cudaError_t e = cudaMemsetAsync(c->tile_state, 0, sizeof(uint32_t) * 256 * (size_t)tiles * c->passes, c->stream);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(c->counters, 0, sizeof(uint32_t) * 64, c->stream);
    if (e != cudaSuccess) return e;
    for (int p = 0; p < c->passes; ++p) {
        onesweep_kernel<<<tiles, RS_THREADS, sizeof(RsSmem), c->stream>>>(
            n, c->kv[p & 1], c->kv[(p + 1) & 1], c->hist + 256 * p,
            c->tile_state + (size_t)p * tiles * 256, c->counters + p, 8 * p,
            (CELL_MASK >> (8 * p)) & 255u);
        c->n_launches++;
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace sph
