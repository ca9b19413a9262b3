// nf_noalloc.cu -- nf_cell_offsets_noalloc: step A2 (exclusive scan of the cell occupancies into the
// per-cell offsets of the grid order, "offset + count" per cell) for callers that must not
// allocate device memory.
//
// Who that is.  Every other entry point of this library works on an nf_ctx, and a context gets its scratch
// from cudaMalloc (nf_create, and again whenever a larger N arrives).  Two kinds of caller cannot live with
// that:
//   * a simulation that has handed the whole GPU to its own memory pool at start-up (the paper's code sizes
//     its state to fill the device): a later cudaMalloc by a library can simply fail, and no context exists
//     to fall back on;
//   * a time-step loop with copies and kernels in flight on several streams: cudaMalloc and cudaFree make the
//     device wait for all of them, so a call that allocates stalls the overlap the loop was built for.
// Such a caller already owns a cell histogram (its own, or nf_cell_histogram's output in a buffer it keeps)
// and a buffer for the offsets; the only other memory the scan needs is one partial sum per 2048-cell tile.
// Here those partial sums live in a fixed array inside the library's device image instead of in memory
// obtained at run time.  The price is a hard size limit (NF_NOALLOC_MAX_CELLS) and 16 KB of device memory
// on every GPU that loads the library, held until the process exits.
//
// The kernels below are this file's own two-launch form of the scan (the context path, nf_binner.cu, uses
// three launches and context-owned partials); integer work, so both give the same offsets bit for bit.
#include <mutex>
#include "nf_common.cuh"

#define NA_THREADS 256
#define NA_ITEMS 8
#define NA_TILE (NA_THREADS * NA_ITEMS)                         // cells per block
#define NA_MAX_TILES (NF_NOALLOC_MAX_CELLS / NA_TILE)           // 4096
#define NA_MAX_DEVICES 64
static_assert(NF_NOALLOC_MAX_CELLS % NA_TILE == 0, "the cell limit is a whole number of tiles");

// The scratch: one partial sum per tile.  In HOST code this name is only a handle for the runtime -- it is
// not a device address and must never be handed to a kernel as one; noalloc_scratch() below asks the
// runtime for the real address on the current device.
static __device__ __align__(256) uint32_t g_na_tile_sum[NA_MAX_TILES];

static std::mutex g_na_mutex;
static uint32_t *g_na_scratch[NA_MAX_DEVICES];                  // device address of g_na_tile_sum, per device ordinal
static char g_na_err[256] = "";

// sum of one value per thread over the block; every thread gets the result
__device__ __forceinline__ uint32_t na_block_sum(uint32_t v) {
    __shared__ uint32_t ws[NA_THREADS / 32];
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    __syncthreads();                                            // ws may still be read from an earlier call
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = v;
    __syncthreads();
    uint32_t s = 0;
#pragma unroll
    for (int w = 0; w < NA_THREADS / 32; ++w) s += ws[w];
    return s;
}

// launch 1: tile_sum[b] = number of particles in the cells of tile b
__global__ void __launch_bounds__(NA_THREADS) k_na_tile_sums(const int32_t *__restrict__ counts, uint32_t ncell,
                                                             uint32_t *__restrict__ tile_sum) {
    const uint32_t base = blockIdx.x * NA_TILE;
    uint32_t s = 0;
#pragma unroll
    for (int k = 0; k < NA_ITEMS; ++k) {
        const uint32_t c = base + k * NA_THREADS + threadIdx.x;
        if (c < ncell) s += (uint32_t)counts[c];
    }
    s = na_block_sum(s);
    if (threadIdx.x == 0) tile_sum[blockIdx.x] = s;
}

// launch 2: block b adds up the sums of the tiles before it (at most 4095 words, cache-resident), then scans
// its own tile in order -- thread t owns NA_ITEMS consecutive cells
__global__ void __launch_bounds__(NA_THREADS) k_na_offsets(const int32_t *__restrict__ counts, uint32_t ncell,
                                                           const uint32_t *__restrict__ tile_sum, uint32_t *__restrict__ offsets) {
    __shared__ uint32_t wtot[NA_THREADS / 32];
    uint32_t before = 0;
    for (uint32_t j = threadIdx.x; j < blockIdx.x; j += NA_THREADS) before += tile_sum[j];
    before = na_block_sum(before);

    const uint32_t c0 = blockIdx.x * NA_TILE + threadIdx.x * NA_ITEMS;
    uint32_t v[NA_ITEMS], mine = 0;
#pragma unroll
    for (int k = 0; k < NA_ITEMS; ++k) {
        v[k] = (c0 + k < ncell) ? (uint32_t)counts[c0 + k] : 0u;
        mine += v[k];
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t inc = mine;                                        // inclusive scan over the warp
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t o = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += o;
    }
    if (lane == 31) wtot[w] = inc;
    __syncthreads();
    uint32_t ex = before + inc - mine;
    for (int j = 0; j < w; ++j) ex += wtot[j];
#pragma unroll
    for (int k = 0; k < NA_ITEMS; ++k) {
        if (c0 + k < ncell) offsets[c0 + k] = ex;
        ex += v[k];
    }
    // the thread that owns the last cell (or thread 0 of an empty grid) also writes the grand total
    if (c0 < ncell ? (c0 + NA_ITEMS >= ncell) : (ncell == 0 && blockIdx.x == 0 && threadIdx.x == 0)) offsets[ncell] = ex;
}

// Set-up, once per device, with that device current: the runtime's answer to "where does g_na_tile_sum live
// on this GPU".  Allocates nothing (the array is part of the loaded module).
static nf_status noalloc_scratch(uint32_t **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= NA_MAX_DEVICES) {
        snprintf(g_na_err, sizeof g_na_err, "nf_cell_offsets_noalloc: no usable current device (%s, ordinal %d)",
                 cudaGetErrorString(e), dev);
        return NF_ECUDA;
    }
    if (!g_na_scratch[dev]) {
        uint32_t *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_na_tile_sum);
        if (e != cudaSuccess || !p) {
            snprintf(g_na_err, sizeof g_na_err, "nf_cell_offsets_noalloc: cudaGetSymbolAddress failed on device %d: %s", dev,
                     cudaGetErrorString(e));
            return NF_ECUDA;
        }
        g_na_scratch[dev] = p;
    }
    *out = g_na_scratch[dev];
    return NF_OK;
}

extern "C" nf_status nf_cell_offsets_noalloc(const int32_t *d_counts, int64_t ncell, uint32_t *d_offsets, void *cuda_stream) {
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (ncell < 0 || !d_offsets || (ncell > 0 && !d_counts)) {
        snprintf(g_na_err, sizeof g_na_err, "nf_cell_offsets_noalloc: bad argument (ncell=%lld, NULL buffer?)", (long long)ncell);
        return NF_EINVAL;
    }
    if (ncell > (int64_t)NF_NOALLOC_MAX_CELLS) {
        snprintf(g_na_err, sizeof g_na_err,
                 "nf_cell_offsets_noalloc: %lld cells exceed the fixed scratch of this entry point (NF_NOALLOC_MAX_CELLS = %d, "
                 "cpd <= 203); use a context (nf_bin) for larger grids", (long long)ncell, NF_NOALLOC_MAX_CELLS);
        return NF_EINVAL;
    }
    uint32_t *scratch = nullptr;
    nf_status rc = noalloc_scratch(&scratch);
    if (rc != NF_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint32_t n = (uint32_t)ncell;
    const uint32_t ntile = n ? (n + NA_TILE - 1) / NA_TILE : 1u;
    // nothing in the scratch has to start at zero: launch 1 writes words [0, ntile) and launch 2 reads only
    // those, so what an earlier call left behind (possibly more words, for a larger grid) is never looked at
    k_na_tile_sums<<<ntile, NA_THREADS, 0, st>>>(d_counts, n, scratch);
    k_na_offsets<<<ntile, NA_THREADS, 0, st>>>(d_counts, n, scratch, d_offsets);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(g_na_err, sizeof g_na_err, "nf_cell_offsets_noalloc: launch failed: %s", cudaGetErrorString(e));
        return NF_ECUDA;
    }
    return NF_OK;
}

extern "C" const char *nf_cell_offsets_noalloc_error(void) { return g_na_err; }
