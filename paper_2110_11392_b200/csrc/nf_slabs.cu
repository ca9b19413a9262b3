// nf_slabs.cu -- device-side support of the x-slab decomposition ("1-D slab
// decomposition", sec. 4.4; near-field radius of ghost slabs: Table 1):
//
//   nf_cell_histogram   occupancy histogram of a rank's particles (step A1's cell rule, the same
//                       nf_axis_cell the binner uses) into a caller-owned device array, so that the
//                       ranks can sum their histograms with one all-reduce;
//   nf_slab_pairs       per x slab: particles, and (sink, source) pairs whose sink lies in the slab,
//                       sum_c n_c (B*n)_c with B the periodic (2R+1)^3 box filter (pin P7) -- the
//                       work measure the slabs are balanced by;
//   nf_select_slabs     stable compaction of the particles whose x cell lies in a periodic slab
//                       range into a contiguous buffer (the halo a neighbour needs; or a check that
//                       a rank's particles all lie in its own slabs), input order kept so that the
//                       receiving rank's sums are run-to-run deterministic.
//
// All integer work; HBM-bound (12 B read per particle).
#include "nf_common.cuh"

__global__ void __launch_bounds__(256) k_cell_hist(const float *__restrict__ pos, uint32_t N, double scale, int cpd,
                                                   int32_t *__restrict__ counts, uint32_t *__restrict__ ctrl) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const float *p = pos + 3ull * i;
    int bad = 0;
    const int cx = nf_axis_cell(p[0], scale, cpd, bad), cy = nf_axis_cell(p[1], scale, cpd, bad), cz = nf_axis_cell(p[2], scale, cpd, bad);
    if (bad) { ctrl[2] = 1u; return; }
    atomicAdd(&counts[(cx * cpd + cy) * cpd + cz], 1);
}

// one thread per cell: n_c * (sum of the (2R+1)^3 neighbours' counts), reduced per x slab
__global__ void __launch_bounds__(256) k_slab_pairs(int cpd, int R, const int32_t *__restrict__ counts, long long *__restrict__ pairs,
                                                    long long *__restrict__ npart) {
    const int ncell = cpd * cpd * cpd;
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncell) return;
    const long long nc = counts[c];
    if (nc == 0) return;
    const int ck = c % cpd, cj = (c / cpd) % cpd, ci = c / (cpd * cpd);
    long long s = 0;
    for (int a = -R; a <= R; ++a) {
        int ia; const int sci = nf_wrap1(ci + a, cpd, ia);
        for (int b = -R; b <= R; ++b) {
            int ib; const int scj = nf_wrap1(cj + b, cpd, ib);
            const int cb = (sci * cpd + scj) * cpd;
            for (int u = ck - R; u <= ck + R; ++u) s += counts[cb + nf_mod(u, cpd)];
        }
    }
    atomicAdd((unsigned long long *)&pairs[ci], (unsigned long long)(nc * s));
    atomicAdd((unsigned long long *)&npart[ci], (unsigned long long)nc);
}

// ---- stable selection: flag -> per-block count -> scan of the block counts -> ordered write
#define SEL_THREADS 256
__device__ __forceinline__ bool in_slab_range(float x, double scale, int cpd, int x0, int nx) {
    int bad = 0;
    int d = nf_axis_cell(x, scale, cpd, bad) - x0;
    if (d < 0) d += cpd;
    return !bad && d < nx;
}
__global__ void __launch_bounds__(SEL_THREADS) k_select_count(const float *__restrict__ pos, uint32_t N, double scale, int cpd, int x0, int nx,
                                                               uint32_t *__restrict__ blk_cnt) {
    const uint32_t i = blockIdx.x * SEL_THREADS + threadIdx.x;
    const bool f = i < N && in_slab_range(pos[3ull * i], scale, cpd, x0, nx);
    const int n = __syncthreads_count(f);
    if (threadIdx.x == 0) blk_cnt[blockIdx.x] = (uint32_t)n;
}
__global__ void __launch_bounds__(SEL_THREADS) k_select_write(const float *__restrict__ pos, uint32_t N, double scale, int cpd, int x0, int nx,
                                                               const uint32_t *__restrict__ blk_base, float *__restrict__ out) {
    __shared__ uint32_t wbase[SEL_THREADS / 32];
    const uint32_t i = blockIdx.x * SEL_THREADS + threadIdx.x;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const bool f = i < N && in_slab_range(pos[3ull * i], scale, cpd, x0, nx);
    const unsigned m = __ballot_sync(0xffffffffu, f);
    if (lane == 0) wbase[w] = (uint32_t)__popc(m);
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t s = 0;
        for (int k = 0; k < SEL_THREADS / 32; ++k) { const uint32_t v = wbase[k]; wbase[k] = s; s += v; }
    }
    __syncthreads();
    if (f) {
        const uint64_t dst = (uint64_t)blk_base[blockIdx.x] + wbase[w] + (uint32_t)__popc(m & ((1u << lane) - 1u));
        const float *p = pos + 3ull * i;
        out[3 * dst] = p[0]; out[3 * dst + 1] = p[1]; out[3 * dst + 2] = p[2];
    }
}

nf_status nf_run_cell_histogram(nf_ctx *ctx, const float *d_pos, int64_t N, int32_t *d_counts, cudaStream_t st) {
    NF_CUDA_OK(ctx, cudaMemsetAsync(d_counts, 0, (size_t)ctx->ncell * sizeof(int32_t), st));
    // (the bad-position flag ctrl[2] is only ever SET here: a flag still pending from an earlier call that nf_sync has
    //  not reported yet must survive; the binner's reset at the start of each sort and nf_create's zero-fill clear it)
    if (N > 0) { k_cell_hist<<<(uint32_t)((N + 255) / 256), 256, 0, st>>>(d_pos, (uint32_t)N, ctx->prm.scale, ctx->cpd, d_counts, ctx->d_ctrl); ctx->launches++; }
    NF_CUDA_OK(ctx, cudaGetLastError());
    return NF_OK;
}

nf_status nf_run_slab_pairs(nf_ctx *ctx, const int32_t *d_counts, long long *d_pairs, long long *d_npart, cudaStream_t st) {
    NF_CUDA_OK(ctx, cudaMemsetAsync(d_pairs, 0, (size_t)ctx->cpd * sizeof(long long), st));
    NF_CUDA_OK(ctx, cudaMemsetAsync(d_npart, 0, (size_t)ctx->cpd * sizeof(long long), st));
    k_slab_pairs<<<((int)ctx->ncell + 255) / 256, 256, 0, st>>>(ctx->cpd, ctx->R, d_counts, d_pairs, d_npart); ctx->launches++;
    NF_CUDA_OK(ctx, cudaGetLastError());
    return NF_OK;
}

// d_blk: scratch of 2 * (nblk + 1) uint32 (counts, then their exclusive scan); the total lands in ctrl[1]
nf_status nf_run_select_slabs(nf_ctx *ctx, const float *d_pos, int64_t N, int x0, int nx, float *d_out, uint32_t *d_blk, cudaStream_t st) {
    const uint32_t nblk = (uint32_t)((N + SEL_THREADS - 1) / SEL_THREADS);
    k_select_count<<<nblk, SEL_THREADS, 0, st>>>(d_pos, (uint32_t)N, ctx->prm.scale, ctx->cpd, x0, nx, d_blk); ctx->launches++;
    nf_status rc = nf_scan_u32(ctx, d_blk, nblk, d_blk + nblk + 1, st);
    if (rc != NF_OK) return rc;
    if (d_out) { k_select_write<<<nblk, SEL_THREADS, 0, st>>>(d_pos, (uint32_t)N, ctx->prm.scale, ctx->cpd, x0, nx, d_blk + nblk + 1, d_out); ctx->launches++; }
    NF_CUDA_OK(ctx, cudaGetLastError());
    return NF_OK;
}
