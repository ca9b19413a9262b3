// nf_binner.cu -- steps A1..A3 of the path: counting-sort cell binner.
//
// PAPER.md:72  "Particles and other properties are stored in grid order, indexed by slab and by
//              cell";  PAPER.md:264 positions are float32 offsets from cell centres;
//              PAPER.md:399 per-cell offset + count.  The paper keeps grid order incrementally
//              (insert list + merge slabs); for a device-resident particle
//              set this build replaces that with a full counting sort per call.
//
//   A1  k_key_hist      cell key per particle (double arithmetic, half-open cells, periodic
//                       wrap) + histogram; the atomic's return value is kept as arrival rank
//   A2  scan            exclusive scan of the counts -> true offsets and padded offsets
//                       (each cell padded to an even slot count) in one 64-bit scan
//   A3  k_scatter       particle index -> its cell's slot range (arrival order)
//       k_rank_gather   within-cell rank by ascending input index (=> stable, deterministic),
//                       gather of the positions, cell-relative float32 offsets in CELL units,
//                       SoA planes x | y | z | key, plus both permutations
#include "nf_common.cuh"

// ------------------------------------------------------------------------------ A1
__global__ void __launch_bounds__(256) k_key_hist(const float *__restrict__ pos, uint32_t N, double scale, int cpd,
                                                  uint32_t *__restrict__ key, uint32_t *__restrict__ arr,
                                                  uint32_t *__restrict__ counts, uint32_t *__restrict__ ctrl) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const float *p = pos + 3ull * i;
    int bad = 0;
    int cx = nf_axis_cell(p[0], scale, cpd, bad);
    int cy = nf_axis_cell(p[1], scale, cpd, bad);
    int cz = nf_axis_cell(p[2], scale, cpd, bad);
    uint32_t k = bad ? 0u : (uint32_t)((cx * cpd + cy) * cpd + cz);
    if (bad) ctrl[2] = 1u;
    key[i] = k;
    arr[i] = atomicAdd(&counts[k], 1u);
}

// ------------------------------------------------------------------------------ A2: scan
// Three-phase exclusive scan of 64-bit items; SCAN_TILE items per block.
#define SCAN_THREADS 256
#define SCAN_ITEMS 8
#define SCAN_TILE (SCAN_THREADS * SCAN_ITEMS)

__device__ __forceinline__ unsigned long long block_excl_scan(unsigned long long v, unsigned long long *total) {
    // exclusive scan of one value per thread across the block (SCAN_THREADS threads)
    __shared__ unsigned long long wsum[SCAN_THREADS / 32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    unsigned long long inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        unsigned long long o = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += o;
    }
    if (lane == 31) wsum[w] = inc;
    __syncthreads();
    if (w == 0) {
        unsigned long long s = (lane < SCAN_THREADS / 32) ? wsum[lane] : 0ull;
#pragma unroll
        for (int d = 1; d < SCAN_THREADS / 32; d <<= 1) {
            unsigned long long o = __shfl_up_sync(0xffffffffu, s, d);
            if (lane >= d) s += o;
        }
        if (lane < SCAN_THREADS / 32) wsum[lane] = s;   // inclusive over warps
    }
    __syncthreads();
    unsigned long long base = (w > 0) ? wsum[w - 1] : 0ull;
    if (total) *total = wsum[SCAN_THREADS / 32 - 1];
    __syncthreads();
    return base + inc - v;
}

// item c of the cell scan = (padded count << 32) | true count
__device__ __forceinline__ unsigned long long cell_item(const uint32_t *counts, uint32_t c) {
    uint32_t n = counts[c];
    return ((unsigned long long)((n + (NF_CELL_PAD - 1u)) & ~(NF_CELL_PAD - 1u)) << 32) | n;
}

// item c of the sink-pair scan = occupancy rounded up to an even number (from the true offsets)
__device__ __forceinline__ unsigned long long pair_item(const uint32_t *offsets, uint32_t c) {
    return (unsigned long long)(((offsets[c + 1] - offsets[c]) + 1u) & ~1u);
}
template <int MODE> __device__ __forceinline__ unsigned long long scan_item(const uint32_t *in, uint32_t c) {
    return MODE == 0 ? cell_item(in, c) : (MODE == 1 ? (unsigned long long)in[c] : pair_item(in, c));
}

template <int MODE>   // 0: cells (from counts)  1: plain uint32 input widened to 64 bit  2: cells padded to 2 (from the true offsets)
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_reduce(const uint32_t *__restrict__ in, uint32_t n,
                                                              unsigned long long *__restrict__ blk) {
    unsigned long long s = 0;
    uint32_t base = blockIdx.x * SCAN_TILE;
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        uint32_t c = base + k * SCAN_THREADS + threadIdx.x;
        if (c < n) s += scan_item<MODE>(in, c);
    }
    unsigned long long tot;
    block_excl_scan(s, &tot);
    if (threadIdx.x == 0) blk[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_blocks(unsigned long long *blk, uint32_t nblk) {
    // single block: exclusive scan of the block totals in place; total appended at blk[nblk]
    unsigned long long carry = 0;
    for (uint32_t b0 = 0; b0 < nblk; b0 += SCAN_THREADS) {
        uint32_t b = b0 + threadIdx.x;
        unsigned long long v = (b < nblk) ? blk[b] : 0ull, tot;
        unsigned long long ex = block_excl_scan(v, &tot);
        if (b < nblk) blk[b] = carry + ex;
        carry += tot;
    }
    if (threadIdx.x == 0) blk[nblk] = carry;
}

template <int MODE>
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_apply(const uint32_t *__restrict__ in, uint32_t n,
                                                             const unsigned long long *__restrict__ blk,
                                                             uint32_t *__restrict__ out_lo, uint32_t *__restrict__ out_hi,
                                                             uint32_t *__restrict__ ctrl) {
    // thread t owns SCAN_ITEMS consecutive items (blocked arrangement) so the scan is in order
    uint32_t base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
    unsigned long long v[SCAN_ITEMS], s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        uint32_t c = base + k;
        v[k] = (c < n) ? scan_item<MODE>(in, c) : 0ull;
        s += v[k];
    }
    unsigned long long ex = block_excl_scan(s, nullptr) + blk[blockIdx.x];
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        uint32_t c = base + k;
        if (c < n) {
            out_lo[c] = (uint32_t)ex;
            if (MODE == 0) out_hi[c] = (uint32_t)(ex >> 32);
        }
        ex += v[k];
    }
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == SCAN_THREADS - 1) {
        // grand total at index n
        unsigned long long tot = blk[gridDim.x];
        out_lo[n] = (uint32_t)tot;
        if (MODE == 0) { out_hi[n] = (uint32_t)(tot >> 32); ctrl[3] = (uint32_t)(tot >> 32); }
        else if (MODE == 1) ctrl[1] = (uint32_t)tot;
        else ctrl[4] = (uint32_t)tot;
    }
}
// k_scan_reduce sums items in a strided arrangement, k_scan_apply in a blocked one; both cover
// exactly the items [blockIdx*SCAN_TILE, (blockIdx+1)*SCAN_TILE), so the block totals agree.

nf_status nf_scan_cells(nf_ctx *ctx, cudaStream_t st) {
    uint32_t n = (uint32_t)ctx->ncell;
    uint32_t nblk = (n + SCAN_TILE - 1) / SCAN_TILE;
    k_scan_reduce<0><<<nblk, SCAN_THREADS, 0, st>>>(ctx->d_counts, n, ctx->d_scan_blk); ctx->launches++;
    k_scan_blocks<<<1, SCAN_THREADS, 0, st>>>(ctx->d_scan_blk, nblk); ctx->launches++;
    k_scan_apply<0><<<nblk, SCAN_THREADS, 0, st>>>(ctx->d_counts, n, ctx->d_scan_blk, ctx->d_offsets, ctx->d_poff, ctx->d_ctrl); ctx->launches++;
    NF_CUDA_OK(ctx, cudaGetLastError());
    return NF_OK;
}

// exclusive scan of the cell occupancies rounded up to even -> d_poff2 (the sink order: two sinks per
// thread, never straddling a cell); the total also goes to ctrl[4]
nf_status nf_scan_pairs(nf_ctx *ctx, cudaStream_t st) {
    uint32_t n = (uint32_t)ctx->ncell;
    uint32_t nblk = (n + SCAN_TILE - 1) / SCAN_TILE;
    k_scan_reduce<2><<<nblk, SCAN_THREADS, 0, st>>>(ctx->d_offsets, n, ctx->d_scan_blk); ctx->launches++;
    k_scan_blocks<<<1, SCAN_THREADS, 0, st>>>(ctx->d_scan_blk, nblk); ctx->launches++;
    k_scan_apply<2><<<nblk, SCAN_THREADS, 0, st>>>(ctx->d_offsets, n, ctx->d_scan_blk, ctx->d_poff2, nullptr, ctx->d_ctrl); ctx->launches++;
    NF_CUDA_OK(ctx, cudaGetLastError());
    return NF_OK;
}

nf_status nf_scan_u32(nf_ctx *ctx, const uint32_t *in, uint32_t n, uint32_t *out, cudaStream_t st) {
    // exclusive scan of n uint32 values into out[0..n]; the total also goes to ctrl[1]
    uint32_t nblk = (n + SCAN_TILE - 1) / SCAN_TILE;
    k_scan_reduce<1><<<nblk, SCAN_THREADS, 0, st>>>(in, n, ctx->d_scan_blk); ctx->launches++;
    k_scan_blocks<<<1, SCAN_THREADS, 0, st>>>(ctx->d_scan_blk, nblk); ctx->launches++;
    k_scan_apply<1><<<nblk, SCAN_THREADS, 0, st>>>(in, n, ctx->d_scan_blk, out, nullptr, ctx->d_ctrl); ctx->launches++;
    NF_CUDA_OK(ctx, cudaGetLastError());
    return NF_OK;
}

// ------------------------------------------------------------------------------ A3
__global__ void __launch_bounds__(256) k_scatter(uint32_t N, const uint32_t *__restrict__ key, const uint32_t *__restrict__ arr,
                                                 const uint32_t *__restrict__ counts, const uint32_t *__restrict__ poff,
                                                 uint32_t *__restrict__ tmp_perm, uint32_t *__restrict__ skey, const uint32_t *__restrict__ ctrl) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    uint32_t k = key[i], r = arr[i];
    uint32_t slot = poff[k] + r;
    NF_CHECK(ctrl, slot < ctrl[3] && r < counts[k], 16);
    tmp_perm[slot] = i;
    skey[slot] = k;
    if (r == 0) {
        uint32_t n = counts[k];
        const uint32_t np = (n + (NF_CELL_PAD - 1u)) & ~(NF_CELL_PAD - 1u);
        for (uint32_t t = n; t < np; ++t) skey[poff[k] + t] = k | NF_PAD_FLAG;   // the padding slots of the cell
    }
}


// Rank within the cell by ascending input index (=> stable, run-to-run deterministic order).  The
// arrival list of a cell is cut into chunks of NF_RANK_CHUNK slots.  A slot counts the smaller indices
// of its own chunk (<= NF_RANK_CHUNK cache-hot loads); for a cell of one chunk (every cell at the
// paper's 30-100 per cell) that is its rank and the particle is gathered at once.  A longer cell
// (clustered states: 10^3-10^4 per cell) would make that count O(n_c^2); instead its chunks are
// written out SORTED and the cell goes onto a worklist, and k_rank_big adds, per slot, one binary
// search in each of the cell's other sorted chunks: O(n_c (chunk + (n_c/chunk) log chunk)).
#define NF_RANK_CHUNK 256
__device__ __forceinline__ void nf_place(const float *__restrict__ pos, double scale, uint32_t cap_pad, float *__restrict__ sorted,
                                         uint32_t *__restrict__ perm_true, uint32_t *__restrict__ perm_pad, uint32_t lo, uint32_t o0,
                                         uint32_t rank, uint32_t me) {
    const uint32_t dst = lo + rank;
    nf_store_offsets(sorted, cap_pad, dst, pos + 3ull * me, scale);
    perm_pad[dst] = me;
    perm_true[o0 + rank] = me;
}

__global__ void __launch_bounds__(256) k_rank_gather(const float *__restrict__ pos, double scale, uint32_t cap_pad,
                                                     uint32_t *__restrict__ ctrl, const uint32_t *__restrict__ offsets,
                                                     const uint32_t *__restrict__ poff, const uint32_t *__restrict__ tmp_perm,
                                                     float *__restrict__ sorted, uint32_t *__restrict__ perm_true,
                                                     uint32_t *__restrict__ perm_pad, uint32_t *__restrict__ chunk_sorted,
                                                     uint32_t *__restrict__ big_cells) {
    uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t npad = ctrl[3];
    uint32_t *skey = (uint32_t *)(sorted + 3ull * cap_pad);
    if (s >= npad) {
        if (s < npad + 8 && s < cap_pad) {    // tail slack read by 16-byte aligned bulk copies
            nf_store_padding(sorted, cap_pad, s); skey[s] = NF_PAD_FLAG; perm_pad[s] = 0xffffffffu;
        }
        return;
    }
    uint32_t k = skey[s];
    if (k & NF_PAD_FLAG) {
        nf_store_padding(sorted, cap_pad, s); perm_pad[s] = 0xffffffffu;
        return;
    }
    const uint32_t lo = poff[k], o0 = offsets[k], n = offsets[k + 1] - o0;
    const uint32_t me = tmp_perm[s];
    const uint32_t c0 = lo + ((s - lo) / NF_RANK_CHUNK) * NF_RANK_CHUNK;           // this slot's chunk: [c0, c1)
    const uint32_t c1 = (c0 + NF_RANK_CHUNK < lo + n) ? c0 + NF_RANK_CHUNK : lo + n;
    uint32_t rank = 0;
    for (uint32_t t = c0; t < c1; ++t) rank += (tmp_perm[t] < me) ? 1u : 0u;
    NF_CHECK(ctrl, rank < c1 - c0 && me < 0x7fffffffu, 17);
    if (n <= NF_RANK_CHUNK) { nf_place(pos, scale, cap_pad, sorted, perm_true, perm_pad, lo, o0, rank, me); return; }
    chunk_sorted[c0 + rank] = me;
    if (s == lo) big_cells[atomicAdd(&ctrl[7], 1u)] = k;
}

// the long cells up to NF_SORT_MAX particles: one CTA per worklist entry sorts the cell's arrival list
// (input indices) in shared memory with a bitonic network -- n log^2 n / 2 compare-exchanges against the
// n (n / chunk) log chunk probes of the chunk method below, which keeps only the cells beyond
// NF_SORT_MAX (more than fit in shared memory).
#define NF_SORT_MAX 32768
__global__ void __launch_bounds__(1024) k_sort_big(const float *__restrict__ pos, double scale, uint32_t cap_pad,
                                                  const uint32_t *__restrict__ ctrl, const uint32_t *__restrict__ offsets,
                                                  const uint32_t *__restrict__ poff, const uint32_t *__restrict__ tmp_perm,
                                                  const uint32_t *__restrict__ big_cells, float *__restrict__ sorted,
                                                  uint32_t *__restrict__ perm_true, uint32_t *__restrict__ perm_pad,
                                                  uint32_t nmin, uint32_t nmax /* this launch: cells of nmin < n <= nmax (its shared memory holds nmax) */) {
    extern __shared__ uint32_t sidx[];
    const uint32_t nbig = ctrl[7];
    for (uint32_t w = blockIdx.x; w < nbig; w += gridDim.x) {
        const uint32_t k = big_cells[w];
        const uint32_t lo = poff[k], o0 = offsets[k], n = offsets[k + 1] - o0;
        if (n <= nmin || n > nmax) continue;                                       // another launch, or k_rank_big
        uint32_t P = 512;
        while (P < n) P <<= 1;
        __syncthreads();
        for (uint32_t i = threadIdx.x; i < P; i += blockDim.x) sidx[i] = i < n ? tmp_perm[lo + i] : 0xffffffffu;
        __syncthreads();
        for (uint32_t kk = 2; kk <= P; kk <<= 1)
            for (uint32_t j = kk >> 1; j > 0; j >>= 1) {
                for (uint32_t t = threadIdx.x; t < (P >> 1); t += blockDim.x) {    // one compare-exchange per thread and step
                    const uint32_t i = ((t & ~(j - 1u)) << 1) | (t & (j - 1u)), ixj = i | j;
                    const uint32_t a = sidx[i], b = sidx[ixj];
                    if ((a > b) == ((i & kk) == 0u)) { sidx[i] = b; sidx[ixj] = a; }
                }
                __syncthreads();
            }
        for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) {
            NF_CHECK(ctrl, sidx[i] != 0xffffffffu && (i == 0 || sidx[i - 1] < sidx[i]), 19);
            nf_place(pos, scale, cap_pad, sorted, perm_true, perm_pad, lo, o0, i, sidx[i]);
        }
    }
}

// the cells beyond NF_SORT_MAX: one CTA per worklist entry strides over the cell's slots
__global__ void __launch_bounds__(256) k_rank_big(const float *__restrict__ pos, double scale, uint32_t cap_pad,
                                                  const uint32_t *__restrict__ ctrl, const uint32_t *__restrict__ offsets,
                                                  const uint32_t *__restrict__ poff, const uint32_t *__restrict__ chunk_sorted,
                                                  const uint32_t *__restrict__ big_cells, float *__restrict__ sorted,
                                                  uint32_t *__restrict__ perm_true, uint32_t *__restrict__ perm_pad) {
    const uint32_t nbig = ctrl[7];
    for (uint32_t w = blockIdx.x; w < nbig; w += gridDim.x) {
        const uint32_t k = big_cells[w];
        const uint32_t lo = poff[k], o0 = offsets[k], n = offsets[k + 1] - o0;
        if (n <= NF_SORT_MAX) continue;                                            // k_sort_big did it
        for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) {
            const uint32_t me = chunk_sorted[lo + i];
            uint32_t rank = i % NF_RANK_CHUNK;                                     // its place in its own sorted chunk
            for (uint32_t c0 = 0; c0 < n; c0 += NF_RANK_CHUNK) {
                if (c0 == i - i % NF_RANK_CHUNK) continue;
                uint32_t a = lo + c0, b = lo + ((c0 + NF_RANK_CHUNK < n) ? c0 + NF_RANK_CHUNK : n);
                const uint32_t first = a;
                while (a < b) {                                                    // entries of that chunk below `me`
                    const uint32_t mid = (a + b) >> 1;
                    if (chunk_sorted[mid] < me) a = mid + 1; else b = mid;
                }
                rank += a - first;
            }
            NF_CHECK(ctrl, rank < n, 20);
            nf_place(pos, scale, cap_pad, sorted, perm_true, perm_pad, lo, o0, rank, me);
        }
    }
}

// once per context (nf_create): k_sort_big's second launch needs 128 KB of dynamic shared memory
nf_status nf_binner_setup(nf_ctx *ctx) {
    NF_CUDA_OK(ctx, cudaFuncSetAttribute(k_sort_big, cudaFuncAttributeMaxDynamicSharedMemorySize, NF_SORT_MAX * 4));
    return NF_OK;
}

// A2 + A3 once the histogram of all N particles is complete on `st`
static nf_status binner_finish(nf_ctx *ctx, const float *d_pos, int64_t N, cudaStream_t st) {
    const uint32_t n = (uint32_t)N;
    if (ctx->opt_stage_timing) cudaEventRecord(ctx->ev[1], st);
    nf_status rc = nf_scan_cells(ctx, st);
    if (rc != NF_OK) return rc;
    if (ctx->opt_stage_timing) cudaEventRecord(ctx->ev[2], st);
    uint32_t *skey = (uint32_t *)(ctx->d_sorted + 3ull * ctx->capPad);
    k_scatter<<<(n + 255) / 256, 256, 0, st>>>(n, ctx->d_key, ctx->d_arr, ctx->d_counts, ctx->d_poff, ctx->d_tmp_perm, skey, ctx->d_ctrl); ctx->launches++;
    NF_CUDA_OK(ctx, cudaGetLastError());
    // upper bound of the padded slot count: N + ncell (+8 slack), known on the host
    uint64_t bound = (uint64_t)N + (uint64_t)(NF_CELL_PAD - 1) * (uint64_t)ctx->ncell + 8;
    if (bound > (uint64_t)ctx->capPad) bound = ctx->capPad;
    k_rank_gather<<<(uint32_t)((bound + 255) / 256), 256, 0, st>>>(d_pos, ctx->prm.scale, (uint32_t)ctx->capPad, ctx->d_ctrl,
                                                                   ctx->d_offsets, ctx->d_poff, ctx->d_tmp_perm, ctx->d_sorted,
                                                                   ctx->d_perm_true, ctx->d_perm_pad, ctx->d_chunk_sorted, ctx->d_key); ctx->launches++;
    // (d_key is free after the scatter: it holds the worklist of long cells, at most N / NF_RANK_CHUNK entries)
    // two launches: the many cells of up to 8192 particles at 32 KB of shared memory (6 CTAs per SM), the few up to NF_SORT_MAX at 128 KB
    k_sort_big<<<ctx->sm_count * 6, 256, 8192 * 4, st>>>(d_pos, ctx->prm.scale, (uint32_t)ctx->capPad, ctx->d_ctrl, ctx->d_offsets, ctx->d_poff,
                                                        ctx->d_tmp_perm, ctx->d_key, ctx->d_sorted, ctx->d_perm_true, ctx->d_perm_pad, NF_RANK_CHUNK, 8192u); ctx->launches++;
    k_sort_big<<<ctx->sm_count, 1024, NF_SORT_MAX * 4, st>>>(d_pos, ctx->prm.scale, (uint32_t)ctx->capPad, ctx->d_ctrl, ctx->d_offsets, ctx->d_poff,
                                                           ctx->d_tmp_perm, ctx->d_key, ctx->d_sorted, ctx->d_perm_true, ctx->d_perm_pad, 8192u, NF_SORT_MAX); ctx->launches++;
    k_rank_big<<<ctx->sm_count * 8, 256, 0, st>>>(d_pos, ctx->prm.scale, (uint32_t)ctx->capPad, ctx->d_ctrl, ctx->d_offsets, ctx->d_poff,
                                                  ctx->d_chunk_sorted, ctx->d_key, ctx->d_sorted, ctx->d_perm_true, ctx->d_perm_pad); ctx->launches++;
    NF_CUDA_OK(ctx, cudaGetLastError());
    if (ctx->opt_stage_timing) cudaEventRecord(ctx->ev[3], st);
    return NF_OK;
}

nf_status nf_run_binner(nf_ctx *ctx, const float *d_pos, int64_t N, cudaStream_t st) {
    const uint32_t n = (uint32_t)N;
    NF_CUDA_OK(ctx, cudaMemsetAsync(ctx->d_counts, 0, (size_t)(ctx->ncell + 1) * sizeof(uint32_t), st));
    NF_CUDA_OK(ctx, cudaMemsetAsync(ctx->d_ctrl, 0, 16 * sizeof(uint32_t), st));
    if (ctx->opt_stage_timing) cudaEventRecord(ctx->ev[0], st);
    k_key_hist<<<(n + 255) / 256, 256, 0, st>>>(d_pos, n, ctx->prm.scale, ctx->cpd, ctx->d_key, ctx->d_arr, ctx->d_counts, ctx->d_ctrl); ctx->launches++;
    NF_CUDA_OK(ctx, cudaGetLastError());
    return binner_finish(ctx, d_pos, N, st);
}

// The binner fed from HOST memory (nf_accel_host): the positions cross PCIe in NF_HOST_CHUNKS ranges on
// the context's copy stream and A1 runs on each range as it lands -- the histogram is additive and the
// arrival rank only has to be unique within a cell -- so key + histogram hide behind the copy.  A2/A3
// need the complete histogram and follow the last range.
nf_status nf_run_binner_host(nf_ctx *ctx, const float *h_pos, float *d_pos, int64_t N, cudaStream_t st) {
    NF_CUDA_OK(ctx, cudaMemsetAsync(ctx->d_counts, 0, (size_t)(ctx->ncell + 1) * sizeof(uint32_t), st));
    NF_CUDA_OK(ctx, cudaMemsetAsync(ctx->d_ctrl, 0, 16 * sizeof(uint32_t), st));
    if (ctx->opt_stage_timing) cudaEventRecord(ctx->ev[0], st);
    const int64_t per = (((N + NF_HOST_CHUNKS - 1) / NF_HOST_CHUNKS) + 255) / 256 * 256;
    for (int c = 0; c < NF_HOST_CHUNKS; ++c) {
        const int64_t i0 = (int64_t)c * per;
        if (i0 >= N) break;
        const int64_t nc = (N - i0 < per) ? N - i0 : per;
        NF_CUDA_OK(ctx, cudaMemcpyAsync(d_pos + 3 * i0, h_pos + 3 * i0, (size_t)nc * 12, cudaMemcpyHostToDevice, ctx->copy_stream));
        NF_CUDA_OK(ctx, cudaEventRecord(ctx->ev_chunk[c], ctx->copy_stream));
        NF_CUDA_OK(ctx, cudaStreamWaitEvent(st, ctx->ev_chunk[c], 0));
        k_key_hist<<<(uint32_t)((nc + 255) / 256), 256, 0, st>>>(d_pos + 3 * i0, (uint32_t)nc, ctx->prm.scale, ctx->cpd, ctx->d_key + i0, ctx->d_arr + i0,
                                                                  ctx->d_counts, ctx->d_ctrl); ctx->launches++;
    }
    NF_CUDA_OK(ctx, cudaGetLastError());
    return binner_finish(ctx, d_pos, N, st);
}
