// nf_rebin.cu -- nf_rebin: drift-aware update of the grid order (sec. 4.2).
//
// The paper never sorts: "most particles stay in their cell" between steps, so a particle that
// drifts out of its cell is pushed onto an INSERT LIST (atomic tail) and the
// Finish step MERGES each cell's remaining particles with the insert-list entries that fall in
// it.  This file is that scheme for a device-resident particle set, starting
// from the grid order the context already holds (perm_true + offsets of the previous positions):
//
//   R1 k_rebin_scan     one warp per OLD cell walks its slots in order: new cell key of each
//                       particle from the moved positions; a particle whose key is unchanged is a
//                       STAYER and gets its rank among the cell's stayers from a ballot prefix --
//                       the old order is ascending input index, so the stayers need no sorting;
//                       the others go onto the insert list (warp-aggregated atomic tail) and are
//                       counted into their new cells.
//   R2 scan             new occupancy = stayers + arrivals -> new true and padded offsets (A2's scan).
//   R3 k_rebin_bucket   insert-list entries are dropped into their new cell's bucket (the tail of
//                       that cell's slot range in a scratch array; order within a bucket is irrelevant).
//   R4 k_rebin_stayers  every stayer moves to  new offset + (rank among stayers) + (arrivals of its
//                       cell with a smaller input index);  R5 k_rebin_movers: every arrival to
//                       (stayers of its new cell with a smaller index: binary search in the old,
//                       ascending segment) + (arrivals with a smaller index).  Both write the
//                       cell-relative float32 offsets of the NEW positions, as A3 does.
//   R6 k_rebin_pads     padding slots of the new layout.
//
// The result is the grid order a full counting sort (A1-A3) of the new positions gives -- cell
// offsets, permutation (ascending input index within a cell) and planes bit for bit -- which is the
// test (tests/test_gpu_step.py).  No O(n_c^2) ranking and no histogram atomics for the stayers; the
// cost of a mover is O(log n_c + arrivals of its cell).  Integer work; HBM-bound.
#include "nf_common.cuh"

#define NF_MOVER 0x80000000u

struct RebinArgs {
    const float *pos;
    const uint32_t *off_old, *perm_old;    // grid order of the previous positions (true slots)
    uint32_t *key_new;                     // [old slot] new cell key
    uint32_t *srank;                       // [old slot] stayers before it in its old cell | NF_MOVER
    uint32_t *ins;                         // insert list: old slots of the movers
    uint32_t *counts, *nstay, *fill;       // per cell: new occupancy, stayers, bucket fill counter
    uint32_t *ctrl;                        // [2] bad position  [5] insert-list tail
    const uint32_t *off_new, *poff_new;    // after R2
    uint32_t *bucket;                      // padded-slot indexed scratch: arrivals of cell c at poff_new[c] + nstay[c] ...
    float *sorted;
    uint32_t *perm_true, *perm_pad;
    double scale;
    int cpd, ncell;
    uint32_t cap_pad;
};

__device__ __forceinline__ uint32_t rebin_key(const float *p, double scale, int cpd, int &bad) {
    const int cx = nf_axis_cell(p[0], scale, cpd, bad), cy = nf_axis_cell(p[1], scale, cpd, bad), cz = nf_axis_cell(p[2], scale, cpd, bad);
    return bad ? 0u : (uint32_t)((cx * cpd + cy) * cpd + cz);
}

__global__ void __launch_bounds__(256) k_rebin_scan(const RebinArgs A) {
    const int lane = threadIdx.x & 31;
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarp = (gridDim.x * blockDim.x) >> 5;
    for (int c = warp; c < A.ncell; c += nwarp) {
        const uint32_t s0 = A.off_old[c], s1 = A.off_old[c + 1];
        uint32_t base = 0;
        for (uint32_t sb = s0; sb < s1; sb += 32) {
            const uint32_t s = sb + lane;
            const bool live = s < s1;
            uint32_t k = (uint32_t)c;
            if (live) {
                int bad = 0;
                k = rebin_key(A.pos + 3ull * A.perm_old[s], A.scale, A.cpd, bad);
                if (bad) A.ctrl[2] = 1u;
            }
            const bool stay = live && k == (uint32_t)c;
            const unsigned ms = __ballot_sync(0xffffffffu, stay), mm = __ballot_sync(0xffffffffu, live && !stay);
            if (live) {
                A.key_new[s] = k;
                A.srank[s] = (base + (uint32_t)__popc(ms & ((1u << lane) - 1u))) | (stay ? 0u : NF_MOVER);
            }
            if (mm) {                                           // push the movers: one atomic on the tail per warp
                uint32_t t = 0;
                if (lane == __ffs(mm) - 1) t = atomicAdd(&A.ctrl[5], (uint32_t)__popc(mm));
                t = __shfl_sync(0xffffffffu, t, __ffs(mm) - 1);
                if (live && !stay) {
                    A.ins[t + (uint32_t)__popc(mm & ((1u << lane) - 1u))] = s;
                    atomicAdd(&A.counts[k], 1u);
                }
            }
            base += (uint32_t)__popc(ms);
        }
        if (lane == 0) {
            A.nstay[c] = base;
            if (base) atomicAdd(&A.counts[c], base);
        }
    }
}

__global__ void __launch_bounds__(256) k_rebin_bucket(const RebinArgs A) {
    const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= A.ctrl[5]) return;
    const uint32_t s = A.ins[e], k = A.key_new[s];
    A.bucket[A.poff_new[k] + A.nstay[k] + atomicAdd(&A.fill[k], 1u)] = A.perm_old[s];
}

__device__ __forceinline__ void rebin_store(const RebinArgs &A, uint32_t k, uint32_t rank, uint32_t me) {
    const float *p = A.pos + 3ull * me;
    const uint32_t dst = A.poff_new[k] + rank;
    uint32_t *skey = (uint32_t *)(A.sorted + 3ull * A.cap_pad);
    nf_store_offsets(A.sorted, A.cap_pad, dst, p, A.scale);     // offsets from the cell centre, cell units (A3's rule)
    skey[dst] = k;
    A.perm_pad[dst] = me;
    A.perm_true[A.off_new[k] + rank] = me;
}

// arrivals of cell k with a smaller input index than `me`
__device__ __forceinline__ uint32_t rebin_arrivals_before(const RebinArgs &A, uint32_t k, uint32_t me) {
    const uint32_t ns = A.nstay[k], n = A.off_new[k + 1] - A.off_new[k];
    const uint32_t *b = A.bucket + A.poff_new[k] + ns;
    uint32_t r = 0;
    for (uint32_t t = 0; t < n - ns; ++t) r += b[t] < me ? 1u : 0u;
    return r;
}

__global__ void __launch_bounds__(256) k_rebin_stayers(const RebinArgs A, uint32_t N) {
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    const uint32_t r = A.srank[s];
    if (r & NF_MOVER) return;
    const uint32_t k = A.key_new[s], me = A.perm_old[s];
    rebin_store(A, k, r + rebin_arrivals_before(A, k, me), me);
}

__global__ void __launch_bounds__(256) k_rebin_movers(const RebinArgs A) {
    const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= A.ctrl[5]) return;
    const uint32_t s = A.ins[e], k = A.key_new[s], me = A.perm_old[s];
    // stayers of the new cell with a smaller index: the old segment of k is ascending in input index
    uint32_t lo = A.off_old[k], hi = A.off_old[k + 1];
    const uint32_t end = hi;
    while (lo < hi) {
        const uint32_t mid = (lo + hi) >> 1;
        if (A.perm_old[mid] < me) lo = mid + 1; else hi = mid;
    }
    const uint32_t before = lo < end ? (A.srank[lo] & ~NF_MOVER) : A.nstay[k];
    rebin_store(A, k, before + rebin_arrivals_before(A, k, me), me);
}

__global__ void __launch_bounds__(256) k_rebin_pads(const RebinArgs A) {
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t *skey = (uint32_t *)(A.sorted + 3ull * A.cap_pad);
    if (c < (uint32_t)A.ncell) {
        const uint32_t n = A.off_new[c + 1] - A.off_new[c], p0 = A.poff_new[c], p1 = A.poff_new[c + 1];
        for (uint32_t t = p0 + n; t < p1; ++t) { nf_store_padding(A.sorted, A.cap_pad, t); skey[t] = c | NF_PAD_FLAG; A.perm_pad[t] = 0xffffffffu; }
    } else if (c < (uint32_t)A.ncell + 8u) {                    // tail slack read by 16-byte aligned bulk copies
        const uint32_t t = A.poff_new[A.ncell] + (c - (uint32_t)A.ncell);
        if (t < A.cap_pad) { nf_store_padding(A.sorted, A.cap_pad, t); skey[t] = NF_PAD_FLAG; A.perm_pad[t] = 0xffffffffu; }
    }
}

nf_status nf_scan_cells(nf_ctx *ctx, cudaStream_t st);   // nf_binner.cu: d_counts -> d_offsets, d_poff, ctrl[3]

nf_status nf_run_rebin(nf_ctx *ctx, const float *d_pos, int64_t N, cudaStream_t st) {
    // the previous grid order becomes "old"; the new one is written into the alternate buffers
    uint32_t *off_old = ctx->d_offsets, *perm_old = ctx->d_perm_true;
    ctx->d_offsets = ctx->d_offsets_alt; ctx->d_offsets_alt = off_old;
    ctx->d_perm_true = ctx->d_perm_alt; ctx->d_perm_alt = perm_old;
    RebinArgs A;
    A.pos = d_pos; A.off_old = off_old; A.perm_old = perm_old;
    A.key_new = ctx->d_key; A.srank = ctx->d_arr; A.ins = ctx->d_ins;
    A.counts = ctx->d_counts; A.nstay = ctx->d_nstay; A.fill = ctx->d_nstay + (ctx->ncell + 1);
    A.ctrl = ctx->d_ctrl; A.off_new = ctx->d_offsets; A.poff_new = ctx->d_poff; A.bucket = ctx->d_tmp_perm;
    A.sorted = ctx->d_sorted; A.perm_true = ctx->d_perm_true; A.perm_pad = ctx->d_perm_pad;
    A.scale = ctx->prm.scale; A.cpd = ctx->cpd; A.ncell = (int)ctx->ncell; A.cap_pad = (uint32_t)ctx->capPad;
    NF_CUDA_OK(ctx, cudaMemsetAsync(ctx->d_counts, 0, (size_t)(ctx->ncell + 1) * sizeof(uint32_t), st));
    NF_CUDA_OK(ctx, cudaMemsetAsync(ctx->d_nstay, 0, (size_t)(ctx->ncell + 1) * 2 * sizeof(uint32_t), st));
    NF_CUDA_OK(ctx, cudaMemsetAsync(ctx->d_ctrl, 0, 16 * sizeof(uint32_t), st));
    if (ctx->opt_stage_timing) cudaEventRecord(ctx->ev[0], st);
    const int ncell = (int)ctx->ncell;
    const int grid_cells = (int)(((int64_t)ncell * 32 + 255) / 256 < (int64_t)ctx->sm_count * 64 ? ((int64_t)ncell * 32 + 255) / 256 : (int64_t)ctx->sm_count * 64);
    k_rebin_scan<<<grid_cells, 256, 0, st>>>(A); ctx->launches++;
    NF_CUDA_OK(ctx, cudaGetLastError());
    if (ctx->opt_stage_timing) cudaEventRecord(ctx->ev[1], st);
    nf_status rc = nf_scan_cells(ctx, st);
    if (rc != NF_OK) return rc;
    if (ctx->opt_stage_timing) cudaEventRecord(ctx->ev[2], st);
    // the insert list is at most N long; its length is on the device, so the per-entry kernels are sized for N
    // and return early (a few empty waves when few particles moved)
    const uint32_t nb = (uint32_t)((N + 255) / 256);
    k_rebin_bucket<<<nb, 256, 0, st>>>(A); ctx->launches++;
    k_rebin_stayers<<<nb, 256, 0, st>>>(A, (uint32_t)N); ctx->launches++;
    k_rebin_movers<<<nb, 256, 0, st>>>(A); ctx->launches++;
    k_rebin_pads<<<(uint32_t)((ncell + 8 + 255) / 256), 256, 0, st>>>(A); ctx->launches++;
    NF_CUDA_OK(ctx, cudaGetLastError());
    if (ctx->opt_stage_timing) cudaEventRecord(ctx->ev[3], st);
    return NF_OK;
}
