// Internal declarations shared by the translation units of libsph_b200.so.
// Nothing here is part of the ABI (include/sph_b200.h is).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "sph_b200.h"

namespace sph {

constexpr uint32_t CELL_MASK = 0x0FFFFFFFu;   // keyword bits 0..27 = cell label
constexpr int TAG_SHIFT = 28;                 // bits 28..29 edge label, 30..31 migration label
constexpr uint32_t ID_MASK = 0x0FFFFFFFu;     // idt bits 0..27 = id, bit 31 = type
constexpr uint32_t TYPE_BIT = 0x80000000u;
constexpr int NUM_SMS = 148;                  // B200 (fallback; sph_ctx::num_sms is the device's own count)
constexpr int GATHER_THREADS = 256;           // slots per tile of gather_kernel = tile of the migrant counts
constexpr int MG_SUB = 16;                    // tiles per group = per CTA of the migrant compaction

// sticky device flags
constexpr uint32_t FLAG_NONFINITE = 1u;

// ---- constants handed to kernels by value -------------------------------------------
struct GridC {
    float min[3];
    float inv_cell;          // 1.0f / (2.0f * h), one fp32 op each (key arithmetic)
    int nc[3];
    int nyz;                 // nc[1]*nc[2]
    uint32_t ncells;
};

struct SlabC {
    int n_slabs;
    int planes[SPH_MAX_SLABS + 1];
};

struct PhysC {
    float h, inv_h_half;     // 0.5/h
    float four_h2;           // (2h)^2
    float eta2;              // 0.01 h^2
    float kF;                // Wendland: -5 aD / h^2 ; cubic spline: aD / h^2 (see interact.cu)
    float alpha_h;           // alpha * h
    float rho0, inv_rho0, c0, B;
    float tait[16];          // binomial coefficients C(gamma, k), k = 1..gamma
    int gamma;
    float g[3];
    float mass_fluid, mass_bound;
    int uniform_mass;
    int kernel;
};

// ---- per-slab execution: arrays and cell planes the interaction kernel works on instead of the
// context's own (sph_interact_slab, slab_exec.cu) ----------------------------------------------
struct IaOverride {
    bool on;
    const float4 *pos4, *velrho4;
    const uint32_t *idt, *keyword, *cell_begin;
    float4 *acc4;
    int cx_first, cx_count;      // cell planes [cx_first, cx_first + cx_count) hold the targets
    int cand_lo, cand_hi;        // cell planes that exist in the local arrays (own + halo planes), inclusive
};

// ---- profiling ------------------------------------------------------------------------
struct StageTimer {
    static constexpr int MAX_PAIRS = 16384;
    cudaEvent_t ev[2 * MAX_PAIRS];
    int stage[MAX_PAIRS];
    int n_pairs = 0;
    int n_created = 0;
    bool enabled = false;
};

}  // namespace sph

struct sph_ctx {
    sph_params P;
    sph::GridC grid;
    sph::SlabC slabs;          // planes used by the next sort
    sph::SlabC tagged_slabs;   // planes the last sort (or retag) labelled with
    sph::PhysC phys;
    uint64_t n;
    int max_slabs;
    int cell_bits, passes;
    int num_sms;               // multiProcessorCount of the context's device (read once in sph_init)
    int keys_blocks_per_sm;    // resident CTAs per SM of this context's keys_kernel<passes> (one wave per launch)
    cudaStream_t stream;
    int sticky;                // SPH_OK or SPH_ERR_CUDA

    // state (double-buffered for the permutation); cur = live buffer
    float4 *pos4[2], *velrho4[2], *velrhoM1[2];
    uint32_t *idt[2];
    int cur;
    float4 *acc4;
    float *mumax;              // max_j |mu_ij| per particle (sorted order), written when adaptive_dt is set
    uint32_t *dt_red;          // 2 * SPH_MAX_SLABS float bit patterns: per slab max |a|^2 (fluid), max (c + mu)
    // sort
    uint2 *kv[2];              // (keyword, prevSlab<<28 | sourceIndex)
    int kv_sorted;             // which kv buffer holds the sorted pairs
    uint32_t *keyword;         // sorted keywords
    uint32_t *hist;            // passes*256 digit histograms
    uint32_t *tile_state;      // passes * rs_tiles * 256 look-back words
    uint32_t *counters;        // 64 words: dynamic tile counters of the sort passes [0..3], gap work-list
                               // counter [8], interaction kernel: tiles listed [16], next tile to hand out [17]
    uint32_t rs_tiles;
    // cells / slabs
    uint32_t *cell_begin;      // ncells+1
    uint4 *gap_list;           // work list of long runs of empty cells (lo, hi, value, -)
    uint32_t *mig_tile;        // migrants per 256-slot tile, written by gather_kernel
    uint32_t *mig_grp;         // migrants per group of MG_SUB tiles, accumulated by gather_kernel
    uint32_t *mig_off;         // exclusive scan of mig_grp (+ total), rebuilt by every halo build
    unsigned long long *scratch64;    // 2 words for measurement helpers
    uint32_t *slab_begin;      // max_slabs+1 (current), also "previous owner" ranges of the next sort
    uint32_t *halo_range;      // 2*max_slabs * 2 (begin, count)
    uint32_t *halo_offset;     // 2*max_slabs+1
    float4 *halo_pos4, *halo_velrho4;
    uint32_t *halo_idt;
    uint4 *migrants;
    uint32_t *mig_total, *mig_count;
    uint8_t *prev_init;        // n bytes: caller-supplied previous owner for the first sort
    uint32_t *flags;           // sticky device flags

    bool have_prev_init;       // prev_init valid for the next sort
    bool have_prev_ranges;     // slab_begin valid as previous-owner ranges
    bool sort_had_prev;        // the last sort labelled migrants (it had previous owners)
    bool sorted_valid;         // arrays sorted + cell table valid for the current positions
    bool halos_valid;
    bool rates_valid;
    bool mu_valid;             // mumax belongs to the current rates
    int adaptive_dt;           // SPH_OPT_ADAPTIVE_DT: sph_interact also produces mumax
    uint64_t step_index;
    int interact_variant;
    int zblock_mma;            // cells per z-block of a tile of the production interaction kernel

    uint64_t n_launches;       // kernels launched so far (memsets and copies not counted)
    bool id_order;             // live state arrays are still in id order (no sort since the last upload)
    char last_cuda_error[160]; // text of the last failed CUDA call (sph_last_cuda_error)

    sph::StageTimer timer;
    sph::IaOverride ia_ov;     // off except inside sph_interact_slab
    uint32_t *cell_loc;        // ncells+1: cell table a slab rebuilds from its own + halo particles
    uint32_t *ia_tiles;        // list of the non-empty tiles of the production interaction kernel
};

namespace sph {

// every launcher enqueues on ctx->stream and returns a cudaError_t
cudaError_t launch_init_state(sph_ctx *c, const float *pos, const float *vel, const float *rho,
                              const uint8_t *type);
cudaError_t launch_keys(sph_ctx *c);
cudaError_t launch_sort(sph_ctx *c);
cudaError_t launch_gather_cells(sph_ctx *c);
cudaError_t launch_cell_fill(sph_ctx *c);
cudaError_t launch_slab_meta(sph_ctx *c);
cudaError_t launch_retag(sph_ctx *c, bool have_prev);
cudaError_t launch_halo_gather(sph_ctx *c);
cudaError_t launch_migrants(sph_ctx *c);
cudaError_t launch_interact(sph_ctx *c, bool with_mu);
cudaError_t launch_dt_reduce(sph_ctx *c);
cudaError_t launch_gap_fill(sph_ctx *c, uint32_t *table);
cudaError_t launch_interact_slab(sph_ctx *c, int slab, const uint32_t *h_slab_begin, const uint32_t *h_halo_range,
                                 const uint32_t *h_halo_offset);
cudaError_t launch_verlet(sph_ctx *c, float dt, int corrective);
cudaError_t launch_pair_stats(sph_ctx *c, unsigned long long *d_out);
cudaError_t launch_download_pack(sph_ctx *c, float *pos3, float *vel3, float *rho, float *acc3,
                                 float *drho);
cudaError_t launch_m1_pack(sph_ctx *c, float *vel3, float *rho);
cudaError_t launch_m1_unpack(sph_ctx *c, const float *vel3, const float *rho);
cudaError_t launch_balance(sph_ctx *c, int n_slabs, int32_t *d_planes);
cudaError_t launch_fma_peak(sph_ctx *c, int variant, int iters, int blocks, float *sink);
// per-device kernel attributes (dynamic shared memory opt-in), set for every new context
cudaError_t configure_interact();
cudaError_t configure_interact_mma();
cudaError_t launch_interact_mma(sph_ctx *c, bool with_mu);
int interact_mma_targets();
size_t interact_mma_tile_capacity(const int nc[3], int zb);
int interact_mma_zmax();
cudaError_t configure_sort();
cudaError_t configure_keys(sph_ctx *c);        // fills keys_blocks_per_sm (needs c->passes)

uint32_t radix_tiles(uint64_t n);
uint32_t gather_tiles(uint64_t n);
uint32_t mig_groups(uint64_t n);
size_t gap_list_entries(uint64_t ncells);

// Tait pressure over rho^2 from rho, fp32, cancellation-free.
__device__ __forceinline__ float tait_p_over_rho2(float rho, const PhysC &ph)
{
    float d = (rho - ph.rho0) * ph.inv_rho0;        // delta = rho/rho0 - 1, subtraction exact near rho0
    float s = ph.tait[ph.gamma];                    // Horner over sum_k C(gamma,k) delta^k
    for (int k = ph.gamma - 1; k >= 1; --k) s = fmaf(s, d, ph.tait[k]);
    float p = ph.B * d * s;
    return __fdividef(p, rho * rho);
}

// Cell coordinate along one axis: one separately rounded fp32 subtract, one fp32 multiply, floor,
// clamp - the sequence ORACLE A pins (a1).
__device__ __forceinline__ int cell_coord(float x, float mn, float inv, int nc)
{
    float t = __fmul_rn(__fsub_rn(x, mn), inv);
    int ci = __float2int_rd(t);           // floor; saturates for huge |t|
    return min(max(ci, 0), nc - 1);
}

// cell_begin[lo..hi] = value: short gaps by the calling thread, long ones through the work list that
// gap_fill_kernel empties (gather_cells.cu).
constexpr uint32_t GAP_INLINE = 32;        // cells a thread fills itself
constexpr uint32_t GAP_CHUNK = 1u << 16;   // cells per work-list entry
__device__ __forceinline__ void fill_cells(uint32_t lo, uint32_t hi /* inclusive */, uint32_t value,
                                           uint32_t *__restrict__ cell_begin, uint4 *__restrict__ gap_list,
                                           uint32_t *__restrict__ gap_count)
{
    if (hi - lo < GAP_INLINE) {
        for (uint32_t cc = lo; cc <= hi; ++cc) cell_begin[cc] = value;
    } else {
        for (uint32_t a = lo; a <= hi; a += GAP_CHUNK) {
            const uint32_t b = min(hi, a + (GAP_CHUNK - 1u));
            gap_list[atomicAdd(gap_count, 1u)] = make_uint4(a, b, value, 0u);
            if (b == hi) break;              // a + GAP_CHUNK could wrap for hi near 2^32
        }
    }
}

// Warps with at most this many runs of equal digits use the hardware MATCH.ANY (about 8 cycles per
// distinct value) for their histogram contribution; beyond it plain shared-memory atomics win.
constexpr int MATCH_MAX_RUNS = 6;

}  // namespace sph
