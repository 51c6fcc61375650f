// sph_cell_table_static - the cell table (a4: "an extra array is generated with the index
// of the first particle of each cell") for callers that have no device memory of their own to give.
//
// Who this is for.  Everything else in this library works out of one workspace that the caller
// allocates and hands to sph_init.  Some users of the sorted arrays cannot do that: an in-situ analysis
// or a coupling code that is only lent the device pointers of an sph_view and owns no context; a plug-in
// running inside a process whose framework has already claimed all of the GPU's memory for its own pool,
// where a raw cudaMalloc fails; a step loop that cannot afford the device-wide stall cudaMalloc and
// cudaFree bring.  For them the one piece of scratch this pass needs - the work list of long runs of
// empty cells and its fill counter - lives in a fixed array inside the library image, below.  The price:
// a hard size limit (SPH_STATIC_MAX_CELLS), about 2 MiB held on every GPU that loads the library until the
// process exits, and no two calls may overlap on one GPU, because they all share that one array.
//
// The pass itself is the cell-table half of gather_kernel (gather_cells.cu), reading the sorted keyword
// array instead of the (keyword, source) pairs: the thread of sorted slot j, where a run of cell c begins,
// writes cell_begin = j for every cell in (previous cell, c]; gaps shorter than ST_INLINE cells it fills
// itself, longer ones (the empty part of a tank) go on the work list, ST_CHUNK cells per entry, which a
// second kernel empties.  Every entry of the table is written exactly once; no memset, no scan.
// HBM-bound: 4 B read per particle, 4 B written per cell.
//
// The existing path (sph_sort_and_cells) does not go through this file.
#include <mutex>
#include <stdio.h>
#include "sph_internal.cuh"

namespace {

constexpr uint32_t ST_INLINE = 32;            // cells a thread fills itself
constexpr uint32_t ST_CHUNK = 1u << 16;       // cells per work-list entry
// A gap on the list is >= ST_INLINE cells long, the gaps are disjoint parts of the ncells + 1 entries, and
// a gap of L cells takes ceil(L / ST_CHUNK) entries: at most (ncells+1)/ST_INLINE + (ncells+1)/ST_CHUNK + 1.
constexpr size_t ST_ENTRIES = SPH_STATIC_MAX_CELLS / ST_INLINE + SPH_STATIC_MAX_CELLS / ST_CHUNK + 8;
constexpr size_t ST_HEAD = 16;                // 16 uint4 = 256 B in front of the list; word 0 = entry counter

// The scratch.  In HOST code this name is only a handle for cudaGetSymbolAddress - it is NOT a device
// address and must never be passed to a kernel or a memset; device_scratch() below turns it into one.
static __device__ __align__(256) uint4 st_scratch[ST_HEAD + ST_ENTRIES];
static_assert(sizeof(st_scratch) == SPH_STATIC_SCRATCH_BYTES, "header states the size of the static scratch");

constexpr int ST_MAX_DEVICES = 64;
std::mutex st_mutex;
uint4 *st_addr[ST_MAX_DEVICES];               // device address of st_scratch on device d, 0 = not asked yet

thread_local char st_error[200] = "";

int fail(int code, const char *what, cudaError_t e = cudaSuccess)
{
    if (e != cudaSuccess) snprintf(st_error, sizeof(st_error), "%s: %s", what, cudaGetErrorString(e));
    else snprintf(st_error, sizeof(st_error), "%s", what);
    return code;
}

// Address of this device's copy of st_scratch.  Asked once per device (every device that loads the module
// has its own copy at its own address), with that device current, and remembered.
int device_scratch(uint4 **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(SPH_ERR_CUDA, "cudaGetDevice", e);
    if (dev < 0 || dev >= ST_MAX_DEVICES) return fail(SPH_ERR_ARG, "device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(st_mutex);
    if (!st_addr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, st_scratch);
        if (e != cudaSuccess || !p) return fail(SPH_ERR_CUDA, "cudaGetSymbolAddress(st_scratch)", e);
        st_addr[dev] = (uint4 *)p;
    }
    *out = st_addr[dev];
    return SPH_OK;
}

__device__ __forceinline__ void st_fill(uint32_t lo, uint32_t hi /* inclusive */, uint32_t value,
                                        uint32_t *__restrict__ cell_begin, uint4 *__restrict__ list,
                                        uint32_t *__restrict__ count)
{
    if (hi - lo < ST_INLINE) {
        for (uint32_t c = lo; c <= hi; ++c) cell_begin[c] = value;
    } else {
        for (uint32_t a = lo;; a += ST_CHUNK) {
            const uint32_t b = min(hi, a + (ST_CHUNK - 1u));
            list[atomicAdd(count, 1u)] = make_uint4(a, b, value, 0u);
            if (b == hi) break;
        }
    }
}

__global__ void __launch_bounds__(256)
cell_table_static_kernel(uint32_t n, uint32_t ncells, const uint32_t *__restrict__ keyword,
                         uint32_t *__restrict__ cell_begin, uint4 *__restrict__ scratch)
{
    uint32_t *count = (uint32_t *)scratch;
    uint4 *list = scratch + ST_HEAD;
    const uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const uint32_t cell = min(keyword[j] & sph::CELL_MASK, ncells - 1u);
    if (j == 0) {
        st_fill(0u, cell, 0u, cell_begin, list, count);
    } else {
        const uint32_t prev = min(keyword[j - 1] & sph::CELL_MASK, ncells - 1u);
        if (cell > prev) st_fill(prev + 1u, cell, j, cell_begin, list, count);
    }
    if (j == n - 1) st_fill(cell + 1u, ncells, n, cell_begin, list, count);      // up to the sentinel entry
}

// One CTA per work-list entry (grid-stride): cell_begin[lo..hi] = value.
__global__ void __launch_bounds__(256)
cell_table_static_fill_kernel(const uint4 *__restrict__ scratch, uint32_t *__restrict__ cell_begin)
{
    const uint32_t count = *(const uint32_t *)scratch;
    const uint4 *list = scratch + ST_HEAD;
    for (uint32_t e = blockIdx.x; e < count; e += gridDim.x) {
        const uint4 g = list[e];
        for (uint32_t c = g.x + threadIdx.x; c <= g.y; c += blockDim.x) cell_begin[c] = g.z;
    }
}

}  // namespace

extern "C" {

int sph_cell_table_static(const uint32_t *keyword, uint64_t n, uint32_t ncells, uint32_t *cell_begin,
                          void *cuda_stream)
{
    st_error[0] = 0;
    if (!cell_begin || (n && !keyword) || ncells == 0) return fail(SPH_ERR_ARG, "NULL array or ncells = 0");
    if (ncells > SPH_STATIC_MAX_CELLS || n > (1ull << 28)) {
        snprintf(st_error, sizeof(st_error),
                 "sph_cell_table_static: ncells = %u, n = %llu is beyond the fixed scratch (at most %u cells, 2^28 "
                 "particles); use sph_sort_and_cells with a workspace instead",
                 ncells, (unsigned long long)n, (unsigned)SPH_STATIC_MAX_CELLS);
        return SPH_ERR_STATIC_LIMIT;
    }
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    if (n == 0) {   // no particles: every entry, sentinel included, is 0; the scratch is not needed
        cudaError_t e = cudaMemsetAsync(cell_begin, 0, sizeof(uint32_t) * ((size_t)ncells + 1), stream);
        return e == cudaSuccess ? SPH_OK : fail(SPH_ERR_CUDA, "cudaMemsetAsync", e);
    }
    uint4 *scratch = nullptr;
    int rc = device_scratch(&scratch);
    if (rc != SPH_OK) return rc;
    // the array keeps what the last call left in it: the entry counter must start at zero (the list
    // entries need no clearing, only the first `counter` of them are ever read)
    cudaError_t e = cudaMemsetAsync(scratch, 0, sizeof(uint4), stream);
    if (e != cudaSuccess) return fail(SPH_ERR_CUDA, "cudaMemsetAsync", e);
    cell_table_static_kernel<<<(uint32_t)((n + 255) / 256), 256, 0, stream>>>((uint32_t)n, ncells, keyword,
                                                                              cell_begin, scratch);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(SPH_ERR_CUDA, "cell_table_static_kernel", e);
    cell_table_static_fill_kernel<<<sph::NUM_SMS * 4, 256, 0, stream>>>(scratch, cell_begin);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(SPH_ERR_CUDA, "cell_table_static_fill_kernel", e);
    return SPH_OK;
}

const char *sph_cell_table_static_error(void) { return st_error; }

}  // extern "C"
