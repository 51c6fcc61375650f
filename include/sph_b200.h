/* sph_b200.h - C ABI of libsph_b200.so: the data-parallel hot path of the SPH time step of
 * arXiv 1210.1017 (Valdez-Balderas, Dominguez, Rogers, Crespo), hand-written for NVIDIA
 * B200 (sm_100a).  Citations "Lnnn" are line numbers of the paper text PAPER.md.
 *
 * The path (one call each, or all of them through sph_step):
 *   sph_sort_and_cells  L138-140  cell label per particle, radix sort of the particles by
 *                                 (cell, id), re-ordering of all state arrays, index of the
 *                                 first particle of every cell; the same pass tags edge
 *                                 ("halo") and migrating particles (L240, L264)
 *   sph_build_halos     L192, L198-219, L224-228, L240-264  halo of every logical x-slab
 *                                 sub-domain (= edge of its neighbours, width 2h) gathered
 *                                 into halo buffers; migrating particles compacted
 *   sph_interact        L101-112, L116, L142-146  right-hand sides of Eqs. (7) and (9)
 *   sph_step            L126-150  all of the above, then the Verlet update (L150)
 *
 * Conventions
 *   - Every pointer argument says HOST or DEVICE.  The library never allocates device memory:
 *     the caller passes one DEVICE workspace of sph_workspace_bytes() bytes (256-byte
 *     aligned) that must outlive the context, and a CUDA stream (cudaStream_t as void*,
 *     NULL = legacy default stream).  Inputs are copied at sph_init / sph_set_state; no
 *     caller memory is referenced afterwards.
 *   - Calls only ENQUEUE work on the stream and return, except sph_download, sph_status,
 *     sph_profile_read and sph_init/sph_set_state with HOST inputs, which synchronise it.
 *   - Return value: SPH_OK (0) or a negative SPH_ERR_* code; no exceptions, no abort, no
 *     CPU fallback.  sph_strerror() names a code.
 *   - Particle k of the input has id k.  n <= 2^28; number of grid cells <= 2^28.
 *   - Precision: fp32 state and arithmetic (the paper does not state its precision, L35).
 */
#ifndef SPH_B200_H
#define SPH_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SPH_MAX_SLABS 16

enum {
    SPH_OK = 0,
    SPH_ERR_ARG = -1,             /* NULL / out-of-range argument */
    SPH_ERR_WORKSPACE = -2,       /* workspace NULL, misaligned or too small */
    SPH_ERR_GRID_TOO_LARGE = -3,  /* more than 2^28 cells, or n > 2^28 */
    SPH_ERR_SLABS = -4,           /* planes not 0 = p0 < p1 < ... < pS = ncx, a slab thinner
                                     than 2 cell planes (S > 1), or S > max_slabs */
    SPH_ERR_CUDA = -5,            /* a CUDA runtime call failed (sticky) */
    SPH_ERR_NONFINITE = -6,       /* a non-finite position/velocity/density was seen on the
                                     device (sticky flag, reported by sph_status) */
    SPH_ERR_ORDER = -7,           /* call order violated (e.g. sph_interact before a sort) */
    SPH_ERR_STATIC_LIMIT = -8     /* sph_cell_table_static: size beyond its fixed built-in scratch */
};

typedef struct sph_ctx sph_ctx;   /* opaque */

/* Physical and grid parameters (all plain values, copied at sph_init). */
typedef struct {
    float dp;                     /* initial particle spacing (used only to size work items) */
    float h;                      /* smoothing length; kernel support and cell side are 2h (L81, L140) */
    float rho0, c0, alpha;        /* Tait reference density and sound speed, viscosity alpha (L112) */
    int   gamma;                  /* Tait exponent, 1..15 (paper: 7) */
    float g[3];                   /* gravity, added to fluid particles (Eq. 9) */
    float mass_fluid, mass_bound; /* particle masses by type */
    float dom_min[3], dom_max[3]; /* cell grid: nc = ceil((max-min)/(2h)) per axis; cell indices
                                     are clamped to the grid (particles are never dropped) */
    int   verlet_ns;              /* every verlet_ns-th step (and step 0) is the one-sided
                                     corrective step; <= 0: step 0 only */
    int   kernel;                 /* 0 = Wendland C2 (hot path), 1 = cubic spline (paper L81) */
} sph_params;

/* Input particles, id order.  Arrays are HOST pointers (on_device = 0) or DEVICE pointers
 * (on_device = 1), owned by the caller, read during the call only. */
typedef struct {
    uint64_t n;
    const float *pos;             /* n*3 (x,y,z interleaved) */
    const float *vel;             /* n*3 */
    const float *rho;             /* n   */
    const uint8_t *type;          /* n, 0 = fluid, 1 = dynamic boundary particle (L116); NULL = all fluid */
    const uint8_t *prev_slab;     /* n, previous owner sub-domain used by the FIRST sort after
                                     this call to label migrants (L264); NULL = no migrants */
    int on_device;
} sph_particles;

/* Borrowed DEVICE pointers into the workspace; valid until the next sph_* call that
 * changes state on this context.  Arrays are in sorted (cell, id) order after a sort. */
typedef struct {
    uint64_t n;
    int32_t  nc[3];               /* cells per axis */
    uint32_t ncells;
    int32_t  cell_bits;           /* bits of the keyword that are sorted */
    int32_t  n_slabs;
    uint64_t step_index;          /* number of completed sph_step calls */
    const float *pos4;            /* n float4: x, y, z, p/rho^2 */
    const float *velrho4;         /* n float4: vx, vy, vz, rho */
    const float *velrhoM1_4;      /* n float4: Verlet n-1 velocity and density */
    const float *acc4;            /* n float4: ax, ay, az, d rho/dt (after sph_interact) */
    const uint32_t *idt;          /* n: id in bits 0..27, type in bit 31 */
    const uint32_t *keyword;      /* n: cell in bits 0..27, edge label bits 28..29 (L240: 1 left,
                                     2 right), migration label bits 30..31 (L264: 1 left, 2 right) */
    const uint32_t *cell_begin;   /* ncells+1: index of the first particle of each cell
                                     (lower bound; cell_end[c] == cell_begin[c+1]) */
    const uint32_t *slab_begin;   /* n_slabs+1: first particle of each slab; owned[s] = diff */
    const uint32_t *halo_offset;  /* 2*n_slabs+1: halo 2s = left halo of slab s, 2s+1 = right
                                     halo; entries [halo_offset[k], halo_offset[k+1]) of: */
    const float *halo_pos4;
    const float *halo_velrho4;
    const uint32_t *halo_idt;
    const uint32_t *mig_total;    /* 1: number of migrant records */
    const uint32_t *migrants;     /* mig_total uint4 records (id, sortedIndex, prevSlab, slab),
                                     in sorted order */
    const uint32_t *mig_count;    /* n_slabs*2: particles that left slab s to the left / right */
    const float *mumax;           /* n: max_j |mu_ij| of every particle over its neighbours (L112, L150), sorted
                                     order; valid after an sph_interact made with SPH_OPT_ADAPTIVE_DT = 1 */
} sph_view;

/* Stage timers (sph_profile_*): indices into the ms[] array. */
enum {
    SPH_T_KEYS = 0, SPH_T_SORT, SPH_T_GATHER, SPH_T_CELLS, SPH_T_HALO, SPH_T_MIGRATE,
    SPH_T_INTERACT, SPH_T_VERLET, SPH_T_DTREDUCE /* the reduction kernel of sph_time_step */, SPH_T_COUNT
};

/* Options for sph_set_option. */
enum {
    SPH_OPT_INTERACT_VARIANT = 0, /* 0 = production kernel, 1 = simple one-thread-per-particle
                                     kernel (cross-check); other values: SPH_ERR_ARG */
    SPH_OPT_ADAPTIVE_DT = 1       /* 1 = sph_interact also records max_j |mu_ij| of every particle,
                                     which sph_time_step needs (costs a few instructions per pair);
                                     0 (default) = fixed-dt path */
};

/* Bytes of DEVICE workspace needed for n_max particles and max_slabs sub-domains with the
 * grid of *p.  Returns 0 on bad arguments or a grid above 2^28 cells. */
size_t sph_workspace_bytes(const sph_params *p, uint64_t n_max, int max_slabs);

/* Create a context.  workspace: DEVICE, >= sph_workspace_bytes(p, part->n, max_slabs) bytes.
 * Copies the particles in (id order), computes p/rho^2, sets step_index = 0, one slab. */
int sph_init(sph_ctx **out, const sph_params *p, const sph_particles *part, int max_slabs,
             void *workspace, size_t workspace_bytes, void *cuda_stream);

/* Replace the whole particle state (same n) and reset step_index; HOST or DEVICE inputs. */
int sph_set_state(sph_ctx *ctx, const sph_particles *part);

/* Set the logical sub-domains: planes HOST int32[n_slabs+1], planes[0] = 0 < ... <
 * planes[n_slabs] = nc[0] (cell-plane indices along x, reading A14/A17).  Takes effect at the
 * next sort; sph_build_halos(planes) is the usual way to set them. */
int sph_set_slabs(sph_ctx *ctx, const int32_t *planes, int n_slabs);

/* Snap physical x bounds (HOST float[n_slabs+1]) to cell planes (HOST int32[n_slabs+1] out). */
int sph_slab_planes_from_x(const sph_ctx *ctx, const float *x_bounds, int n_slabs, int32_t *planes_out);

/* a1-a4: keys+tags, radix sort by (cell, id), payload permutation, cell table, slab ranges. */
int sph_sort_and_cells(sph_ctx *ctx);

/* a5-a6: halo gather and migrant compaction for the given planes (HOST; NULL = keep the
 * current ones).  Needs a sort since the last state change.  If the planes differ from the
 * ones the last sort tagged with, edge labels are recomputed. */
int sph_build_halos(sph_ctx *ctx, const int32_t *planes, int n_slabs);

/* a7: acc4 = (dv/dt, d rho/dt) of every particle.  Needs the cell table. */
int sph_interact(sph_ctx *ctx);

/* a7 for ONE logical sub-domain, the way GPU_k does it in the paper (L192, L218-220, L226-228): the
 * rates of the particles slab `slab` owns, computed from its own particles and the two HALO BUFFERS
 * that sph_build_halos filled, and from nothing else - the local set is assembled, its cell table is
 * rebuilt from the particles' positions, and the production interaction kernel runs on it.  Results go
 * to the slab's range of acc4; calling it for every slab reproduces sph_interact (the device-side proof
 * that a 2h halo suffices): value for value while every tile next to a slab plane fits one candidate batch of
 * the kernel (particles on or near their lattice), else to rounding, because an over-full tile is cut into
 * batches at different candidates in the two runs and its partial sums are added in a different order.  Needs sph_build_halos since the last sort (else
 * SPH_ERR_ORDER); uses the idle halves of the state buffers as scratch; synchronises the stream once
 * (the slab ranges cross to the host). */
int sph_interact_slab(sph_ctx *ctx, int slab);

/* a1-a8 in order; dt > 0. */
int sph_step(sph_ctx *ctx, float dt);

/* Variable time step (the step size "varies throughout each simulation according
 * to the Courant-Friedrichs-Lewy (CFL) condition and the magnitude of the interactions", found
 * with reductions over all particles; L222: every sub-domain determines its own dt_k and the
 * minimum is used).  The paper prints no formula; reading A8b:
 *     dt = cfl * min( sqrt(h / max_i |a_i|) over fluid particles,
 *                     h / max_i (c_i + max_j |mu_ij|) over all particles ),  mu_ij as in L112.
 * Needs the rates of an sph_interact made with SPH_OPT_ADAPTIVE_DT = 1 (else SPH_ERR_ORDER).
 * HOST outputs, any may be NULL: *dt; amax_slab[n_slabs] = max |a| and smax_slab[n_slabs] =
 * max (c + mu) of every current sub-domain (dt_k = cfl * min(sqrt(h/amax_k), h/smax_k)).
 * One reduction kernel over the sorted arrays; synchronises the stream.  cfl > 0. */
int sph_time_step(sph_ctx *ctx, float cfl, float *dt, float *amax_slab, float *smax_slab);

/* a1-a7, sph_time_step, a8 with that step; *dt_used (HOST, may be NULL) receives it.  Turns
 * SPH_OPT_ADAPTIVE_DT on.  Synchronises once per step (the step size crosses to the host, as
 * the paper's does for its MPI_Allreduce). */
int sph_step_adaptive(sph_ctx *ctx, float cfl, float *dt_used);

/* Movable slab planes (dynamic load balancing; "a multidimensional domain decomposition
 * with load balancing", L389).  From the per-plane particle counts that the cell table of the last
 * sort holds, choose planes_out[0..n_slabs] (HOST int32) so that the slabs own about n / n_slabs
 * particles each: plane s = the cell plane p in [planes[s-1] + 2, ncx - 2 (n_slabs - s)] that minimises
 * |#(particles left of p) * n_slabs - s * n|, the lowest such p on ties, chosen left to right (every
 * slab keeps >= 2 cell planes, reading A14).  Does not change the context: hand the planes to
 * sph_build_halos(planes) (new owners, edge labels, halos and migrants without a new sort: a particle
 * whose owner changes because a plane moved is a migrant, reading A15) or to sph_set_slabs.  Needs a sort
 * since the last state change; synchronises the stream.  SPH_ERR_SLABS if nc[0] < 2 n_slabs. */
int sph_balance_slabs(sph_ctx *ctx, int n_slabs, int32_t *planes_out);

/* The borrowed device pointers of the current state ("data is stored on the GPU
 * memory"; everything a4-a6 produce stays there for the next stage, L224-228). */
int sph_get_view(sph_ctx *ctx, sph_view *out);

/* Saving results (particle data "are copied to the host only when saving", L211-212
 * "copy all particle data to host").  HOST outputs in ID order, any of them may be NULL: pos n*3,
 * vel n*3, rho n, acc n*3, drho n.  Synchronises the stream. */
int sph_download(sph_ctx *ctx, float *pos, float *vel, float *rho, float *acc, float *drho);

/* Exact checkpoint / resume (same passages): the part of the state sph_download does not return - the
 * Verlet n-1 velocity and density (reading A7) in ID order, HOST vel_m1 n*3 and rho_m1 n (may be NULL),
 * and the number of completed steps.  To resume: sph_init / sph_set_state with the saved pos, vel, rho,
 * then sph_set_resume (HOST or DEVICE arrays, on_device says which) BEFORE the next sort (else
 * SPH_ERR_ORDER); the particle state then continues bit for bit as if the run had never stopped (the sort
 * order is history-free, reading A12).  One thing is NOT part of the checkpoint: the previous owner
 * sub-domain of every particle.  The first sort after a resume therefore labels no migrants (mig_total and
 * mig_count are 0 for that step, as after any sph_init without prev_slab) where the uninterrupted run
 * reports the particles that crossed a plane in that step; from the second step on the migrant records
 * agree again.  A caller that needs them across the restart passes the owners through
 * sph_particles.prev_slab.  Both synchronise the stream (sph_set_resume only for HOST inputs). */
int sph_download_resume(sph_ctx *ctx, float *vel_m1, float *rho_m1, uint64_t *step_index);
int sph_set_resume(sph_ctx *ctx, const float *vel_m1, const float *rho_m1, uint64_t step_index, int on_device);

/* Synchronise the stream; return the sticky error (SPH_OK, SPH_ERR_CUDA, SPH_ERR_NONFINITE: the device
 * flag raised by any kernel that met a non-finite position, velocity, density or rate). */
int sph_status(sph_ctx *ctx);

/* Text of the last failed CUDA runtime call of this context (ctx = NULL: of the calling thread, for
 * failures inside sph_init); "" if none.  The library never prints. */
const char *sph_last_cuda_error(const sph_ctx *ctx);

int sph_set_option(sph_ctx *ctx, int option, int value);

/* CUDA-event stage timers on the context's stream.  enable != 0 starts recording an event
 * pair around every stage of every call; sph_profile_read synchronises, ADDS the elapsed
 * milliseconds of all recorded pairs to ms[SPH_T_COUNT] and the number of pairs to
 * launches[SPH_T_COUNT] (HOST arrays, may be NULL), then clears the record. */
int sph_profile_enable(sph_ctx *ctx, int enable);
int sph_profile_read(sph_ctx *ctx, float *ms, int *launches);

/* Measurement helpers (not on the hot path).  sph_pair_stats: runs a counting kernel over the
 * current sorted state and returns, in HOST out[2], the number of candidate pairs the 27-cell
 * search examines and the number of pairs inside the support (0 < r < 2h); synchronises.
 * sph_launch_count: HOST *out = number of kernels this context has launched so far. */
int sph_pair_stats(sph_ctx *ctx, uint64_t *out);
int sph_launch_count(const sph_ctx *ctx, uint64_t *out);

/* Measured FP32 peak of this GPU: a register-resident chain of fused multiply-adds,
 * variant 0 = scalar FFMA, 1 = packed FFMA2 (two fp32 lanes per instruction); iters >= 1 rounds of 64
 * FMA lanes per thread on 8 CTAs of 256 threads per SM (148 x 8 on a B200); HOST *tflops = 2 flop per FMA / CUDA-event time.
 * The denominator bench.py reports beside the nominal 148 x 128 x 2 x clock.  Synchronises. */
int sph_fma_peak(sph_ctx *ctx, int variant, int iters, double *tflops);

/* The cell table without a context, a workspace or any allocation (a4: the "extra array
 * ... with the index of the first particle of each cell"; L276 "first and last particle in a given region").
 *
 * Why it exists: every other call works out of the workspace the caller allocated for sph_init.  A caller
 * that cannot allocate device memory has nothing to hand over - for instance an analysis or coupling code
 * that was only lent the pointers of an sph_view, a plug-in in a process whose framework already owns all
 * of the GPU's memory (a plain cudaMalloc fails there), or a loop that must not take the device-wide stall
 * of cudaMalloc / cudaFree.  This call needs from the caller only its input and its output; the scratch it
 * uses (a work list of long runs of empty cells, plus a counter) is an array of SPH_STATIC_SCRATCH_BYTES
 * (about 2 MiB) built into the library, present on every GPU that loads the library until the process ends.
 * It calls no cudaMalloc, cudaFree or allocating library routine.
 *
 *   keyword     DEVICE, n words, non-decreasing in bits 0..27 (the cell label; bits 28..31 are ignored) -
 *               e.g. sph_view.keyword, or the keywords of one sub-domain's particles.  Read only.
 *   n           number of particles, <= 2^28; n = 0 gives an all-zero table
 *   ncells      number of cells, 1 <= ncells <= SPH_STATIC_MAX_CELLS; labels >= ncells count as ncells - 1
 *   cell_begin  DEVICE, ncells + 1 words, written in full: cell_begin[c] = number of particles whose cell
 *               label is below c (index of the first particle of cell c; cell_begin[ncells] = n) - the
 *               same values sph_sort_and_cells leaves in sph_view.cell_begin
 *   cuda_stream cudaStream_t as void*, NULL = legacy default stream; work is enqueued, not waited for
 *
 * Limits and rules, all consequences of the scratch being one fixed array:
 *   - ncells > SPH_STATIC_MAX_CELLS (or n > 2^28) is refused with SPH_ERR_STATIC_LIMIT and nothing is
 *     launched; use sph_sort_and_cells with a workspace for larger grids.
 *   - All calls on one GPU share the array, from every thread and stream of the process.  Two calls whose
 *     GPU work may overlap (different streams without an ordering between them) race on it and give wrong
 *     tables; order them on one stream or with events.  The array keeps the previous call's contents; the
 *     call itself resets the one word that has to start at zero.
 *   - The first call on each GPU looks up where that GPU's copy of the array lives (cudaGetSymbolAddress,
 *     done with the calling thread's current device, result kept).  Make that first call during set-up,
 *     before any stream capture begins.  The device that is current at the call must be the one that owns
 *     keyword, cell_begin and the stream.
 * Returns SPH_OK or SPH_ERR_ARG / SPH_ERR_STATIC_LIMIT / SPH_ERR_CUDA; sph_cell_table_static_error() is the
 * text of the calling thread's last failure of this call ("" if it succeeded). */
#define SPH_STATIC_MAX_CELLS (1u << 22)
#define SPH_STATIC_SCRATCH_BYTES 2098560u
int sph_cell_table_static(const uint32_t *keyword, uint64_t n, uint32_t ncells, uint32_t *cell_begin,
                          void *cuda_stream);
const char *sph_cell_table_static_error(void);

void sph_destroy(sph_ctx *ctx);
const char *sph_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* SPH_B200_H */
