// nf_interact.cu -- steps A4..A6: pencil scheduler, pencil-on-pencil interaction kernel with
// fused un-permute, plus the neighbour-list and pair-count exports.
//
// Paper basis: PAPER.md:226-236 (sec. 3.4.2 pencil-on-pencil; sink blocks; sinks in registers,
// sources staged in shared memory), PAPER.md:132 (Eq. 3), PAPER.md:254 (hand-off to 1/r^2 "with
// a min instead of a conditional").  What differs from the paper's V100 design, and why, is in
// DESIGN.md sections 6-8:
//   * sinks AND sources are z-pencils (z is the fastest cell index, so the source cells
//     (i+a, j+b, k-R..k+R) of one (a,b) column are ONE contiguous range of the sorted planes
//     -> one cp.async.bulk per coordinate plane per column window, completed on an mbarrier);
//   * 64 consecutive grid-order sinks per warp (two per thread, same cell) regardless of cell
//     boundaries; source cells c and c+2R+1, each needed by only part of the warp, are read in
//     the same pass by disjoint lane groups; a lane that needs neither is masked by moving its
//     sink to -NF_BIG, which makes its contribution exactly 0 (no per-interaction predicate);
//   * four sources per LDS.128 and plane, shared by the thread's two sinks; two sources per
//     packed fma.rn.f32x2 / add.f32x2 / mul.f32x2, so the FMA pipe is the bound, not the issue
//     slots or the LSU;
//   * source cells that cannot hold r < eps_s skip the spline (11 instead of 14 FMA-pipe ops);
//     with a close-pair radius the near cells clamp r^-3 and close_scan repairs close pairs in double;
//   * no producer warp: the consumer warps refill the NF_NSTAGE-deep full/empty mbarrier ring of
//     (column, z-run, chunk) stages themselves, from a cursor in shared memory and under a lock
//     (whichever warp runs ahead does it); persistent CTAs pull sink blocks from an atomic
//     counter in grid order;
//   * A6 is fused: each thread writes gm/cell^2 * a straight to d_acc[perm[slot]].
#include "nf_common.cuh"

// ------------------------------------------------------------------------------ PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try(uint64_t *bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0u;
}
__device__ __forceinline__ bool mbar_test(uint64_t *bar, uint32_t parity) {     // non-blocking
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0u;
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {     // try_wait suspends in hardware between polls
    while (!mbar_try(bar, parity)) {}
}
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ float mufu_rsq(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ------------------------------------------------------------------------------ A4: scheduler
// Sink work items: every z-column (cx,cy) is cut into blocks of consecutive grid-order sinks,
// balanced within the column ("sink particles are arranged into blocks").  Sinks are
// counted in the SINK ORDER: cells padded to 2 slots, not to the 4 of the source planes -- a thread
// holds the two sinks of one pair, which must share a cell, but a sink lane spent on padding is
// wasted, and at 40 per cell padding to 4 wastes 9 % of them against 1 % for 2.  k_pair_slots maps
// sink pair i to the padded slot of its first sink.
// sink slabs: only columns whose x cell index lies in the periodic range [x0, x0 + nx) hold sinks
// (slab decomposition); the other columns are sources only (ghost slabs).
__device__ __forceinline__ bool nf_sink_slab(int cx, int cpd, int x0, int nx) {
    int d = cx - x0;
    if (d < 0) d += cpd;
    return d < nx;
}
__global__ void __launch_bounds__(256) k_pair_slots(uint32_t cap_pad, const uint32_t *__restrict__ ctrl, const uint32_t *__restrict__ skey,
                                                    const uint32_t *__restrict__ offsets, const uint32_t *__restrict__ poff,
                                                    const uint32_t *__restrict__ poff2, uint32_t *__restrict__ pair_slot) {
    const uint32_t s = 2u * (blockIdx.x * blockDim.x + threadIdx.x);      // even padded slots: cells start on multiples of 4
    if (s >= ctrl[3]) return;
    const uint32_t k = skey[s] & ~NF_PAD_FLAG;
    const uint32_t t = s - poff[k];
    if (t < offsets[k + 1] - offsets[k]) {
        NF_CHECK(ctrl, ((poff2[k] + t) >> 1) < (ctrl[4] + 1u) / 2u && ((poff2[k] + t) >> 1) < cap_pad / 2u + 8u, 18);
        pair_slot[(poff2[k] + t) >> 1] = s;
    }
}

__global__ void __launch_bounds__(256) k_col_blocks(int ncol, int cpd, int x0, int nx, const uint32_t *__restrict__ poff, uint32_t *__restrict__ col_nblk) {
    int col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= ncol) return;
    uint32_t n = poff[(col + 1) * cpd] - poff[col * cpd];
    if (!nf_sink_slab(col / cpd, cpd, x0, nx)) n = 0;
    col_nblk[col] = (n + NF_BS - 1) / NF_BS;
}

__global__ void __launch_bounds__(128) k_fill_blocks(int ncol, int cpd, const uint32_t *__restrict__ poff, const uint32_t *__restrict__ col_nblk,
                                                     const uint32_t *__restrict__ col_base, NfBlockDesc *__restrict__ blk, int R) {
    int col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= ncol) return;
    const uint32_t nb = col_nblk[col];
    if (nb == 0) return;
    const uint32_t p0 = poff[col * cpd], n = poff[(col + 1) * cpd] - p0;
    const uint32_t bs = (((n + nb - 1) / nb) + (32u * NF_SINKS - 1u)) & ~(32u * NF_SINKS - 1u);
    const uint32_t base = col_base[col];
    // cost estimate: sinks x (sources of the whole home column window), cheap proxy = sinks x column density x (2R+1+span)
    for (uint32_t k = 0; k < nb; ++k) {
        NfBlockDesc d;
        d.col = (uint32_t)col;
        d.s0 = p0 + k * bs;
        uint32_t rem = (k * bs < n) ? n - k * bs : 0u;
        d.cnt = rem < bs ? rem : bs;
        unsigned long long c = (unsigned long long)d.cnt * (unsigned long long)n;
        d.cost = c > 0xffffffffull ? 0xffffffffu : (uint32_t)c;
        blk[base + k] = d;
    }
}

// Heavy-first order: counting sort of the blocks into 64 half-octave cost buckets, descending.
__device__ __forceinline__ int cost_bucket(uint32_t c) {
    if (!c) return 63;
    const int l = 31 - __clz(c);
    const int half = l > 0 ? (int)((c >> (l - 1)) & 1u) : 0;
    return 63 - (2 * l + half);
}
__global__ void __launch_bounds__(256) k_order_hist(const uint32_t *__restrict__ ctrl, const NfBlockDesc *__restrict__ blk, uint32_t *__restrict__ hist) {
    uint32_t b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= ctrl[1]) return;
    atomicAdd(&hist[cost_bucket(blk[b].cost)], 1u);
}
__global__ void k_order_scan(uint32_t *hist) {   // 64 buckets, one thread
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        uint32_t s = 0;
        for (int i = 0; i < 64; ++i) { uint32_t v = hist[i]; hist[i] = s; s += v; }
    }
}
__global__ void __launch_bounds__(256) k_order_fill(const uint32_t *__restrict__ ctrl, const NfBlockDesc *__restrict__ blk, uint32_t *__restrict__ hist,
                                                    uint32_t *__restrict__ order) {
    uint32_t b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= ctrl[1]) return;
    order[atomicAdd(&hist[cost_bucket(blk[b].cost)], 1u)] = b;
}
__global__ void __launch_bounds__(256) k_order_identity(const uint32_t *__restrict__ ctrl, uint32_t *__restrict__ order) {
    uint32_t b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < ctrl[1]) order[b] = b;
}

// Close-pair radius r_c.  Per-pair error model of the float32 fast path:
// relative error kappa(r) = 1e-6 (MUFU.RSQ cubed + roundings) + 1.2e-7/r (float32 offsets of both
// particles, up to 1.5e-8 cell each, and the shifted sink, up to 3e-8, against a separation r).
// A pair with F = 1/r^2 is sent to close_pair() when F kappa(r) > 0.4e-5 rms|a|, with the
// Holtsmark-like estimate rms|a|^2 ~ 4 pi n_pw / eps_s (cell units; n_pw = sum n_c^2 / N, the
// particle-weighted cell occupancy; measured rms is ~1.4x this, so the estimate is conservative).
// If even the softened core needs no exact path, r_c = 0 and Eq. 3 is evaluated as a min.
__global__ void __launch_bounds__(256) k_density(int ncell, const uint32_t *__restrict__ counts, unsigned long long *__restrict__ sum2) {
    int c = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long v = 0;
    if (c < ncell) { unsigned long long n = counts[c]; v = n * n; }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    if ((threadIdx.x & 31) == 0 && v) atomicAdd(sum2, v);
}
// law: NF_SOFT_SPLINE / NF_SOFT_PLUMMER / NF_SOFT_NEWTON.  For the spline the near cells of the
// close-pair regime evaluate only min(r^-3, r_c^-3) and leave Eq. 3's polynomial to close_scan,
// so a non-zero r_c must never lie below eps_s: pairs with r_c <= r < eps_s would get r^-3
// (PAPER.md:132).  Hence r_c, chosen or forced, is raised to eps_s when it falls short of it, and
// the 0.25-cell cap only applies above eps_s.  Without softening (Newton) there is no core to
// estimate rms|a| from: the estimate uses the production softening, eps_s = 2.16/40 of the
// particle-weighted mean spacing, and r_c is kept positive, so that the self pair
// and coincident pairs meet the finite clamp (f = r_c^-3, d = 0) instead of inf * 0.
__global__ void k_choose_rc(const unsigned long long *__restrict__ sum2, double N, double eps_cells, double soft2, int law, float rc_override,
                            float *__restrict__ dyn) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    double rc;
    if (rc_override >= 0.f) {
        rc = rc_override;
    } else {
        const double npw = (double)(*sum2) / N;
        const double eps_rms = law == NF_SOFT_NEWTON ? NF_SPLINE_PER_PLUMMER / 40.0 / cbrt(npw) : eps_cells;
        const double rms = sqrt(4.0 * 3.14159265358979 * npw / eps_rms);
        const double budget = 0.4e-5 * rms;
        rc = 0.05;
        for (int it = 0; it < 20; ++it) rc = sqrt((1.0e-6 + 1.2e-7 / rc) / budget);
        if (law != NF_SOFT_NEWTON && rc < eps_cells) {
            // inside the core F <= 2.01/eps^2 and |dF/dr| <= 10/eps^3
            const double core = 2.01 / (eps_cells * eps_cells) * 1.0e-6 + 10.0 / (eps_cells * eps_cells * eps_cells) * 6.0e-8;
            rc = (core <= budget) ? 0.0 : eps_cells;
        }
        if (rc > 0.25) rc = 0.25;
    }
    if (law == NF_SOFT_SPLINE && rc > 0.0 && rc < eps_cells) rc = eps_cells;
    if (law == NF_SOFT_NEWTON && rc < 1.0e-4) rc = 1.0e-4;
    dyn[0] = (float)(rc * rc);
    dyn[1] = (float)rc;
    // soft2 = eps_p^2 (cell units) for Plummer softening (the loop's r^2 carries it), 0 otherwise
    const double rs2 = rc * rc + soft2;
    dyn[2] = rc > 0.0 ? (float)(1.0 / (rs2 * sqrt(rs2))) : 0.f;   // clamp of the float32 force factor in near cells
    dyn[3] = (float)rs2;                                           // what the loop's r^2 (+ soft2) is compared with
}

nf_status nf_run_scheduler(nf_ctx *ctx, int64_t N, cudaStream_t st) {
    const int ncol = (int)ctx->ncol;
    unsigned long long *sum2 = (unsigned long long *)(ctx->d_ctrl + 100);
    NF_CUDA_OK(ctx, cudaMemsetAsync(sum2, 0, 8, st));
    k_density<<<((int)ctx->ncell + 255) / 256, 256, 0, st>>>((int)ctx->ncell, ctx->d_counts, sum2); ctx->launches++;
    {
        const double ep = ctx->eps_p * ctx->prm.scale;       // eps_p in cell units
        const bool plummer = ctx->law == NF_SOFT_PLUMMER;
        k_choose_rc<<<1, 32, 0, st>>>(sum2, (double)N, plummer ? ep : ctx->prm.eps_cells, plummer ? ep * ep : 0.0, ctx->law, ctx->opt_rc,
                                      (float *)(ctx->d_ctrl + 96)); ctx->launches++;
    }
    nf_status rc = nf_scan_pairs(ctx, st);
    if (rc != NF_OK) return rc;
    {
        uint64_t bound = (uint64_t)N + (uint64_t)(NF_CELL_PAD - 1) * (uint64_t)ctx->ncell + 8;      // of the padded slot count, as in the binner
        if (bound > (uint64_t)ctx->capPad) bound = ctx->capPad;
        k_pair_slots<<<(uint32_t)((bound / 2 + 255) / 256), 256, 0, st>>>((uint32_t)ctx->capPad, ctx->d_ctrl, (const uint32_t *)(ctx->d_sorted + 3ull * ctx->capPad),
                                                                          ctx->d_offsets, ctx->d_poff, ctx->d_poff2, ctx->d_pair_slot); ctx->launches++;
    }
    k_col_blocks<<<(ncol + 255) / 256, 256, 0, st>>>(ncol, ctx->cpd, ctx->slab_x0, ctx->slab_nx, ctx->d_poff2, ctx->d_col_nblk); ctx->launches++;
    rc = nf_scan_u32(ctx, ctx->d_col_nblk, (uint32_t)ncol, ctx->d_col_base, st);
    if (rc != NF_OK) return rc;
    k_fill_blocks<<<(ncol + 127) / 128, 128, 0, st>>>(ncol, ctx->cpd, ctx->d_poff2, ctx->d_col_nblk, ctx->d_col_base, ctx->d_blk, ctx->R); ctx->launches++;
    const uint32_t bound = (uint32_t)ctx->capBlk;
    if (ctx->opt_heavy_first) {
        uint32_t *hist = ctx->d_ctrl + 16;   // 64 words
        NF_CUDA_OK(ctx, cudaMemsetAsync(hist, 0, 64 * sizeof(uint32_t), st));
        k_order_hist<<<(bound + 255) / 256, 256, 0, st>>>(ctx->d_ctrl, ctx->d_blk, hist); ctx->launches++;
        k_order_scan<<<1, 32, 0, st>>>(hist); ctx->launches++;
        k_order_fill<<<(bound + 255) / 256, 256, 0, st>>>(ctx->d_ctrl, ctx->d_blk, hist, ctx->d_blk_order); ctx->launches++;
    } else {
        k_order_identity<<<(bound + 255) / 256, 256, 0, st>>>(ctx->d_ctrl, ctx->d_blk_order); ctx->launches++;
    }
    NF_CUDA_OK(ctx, cudaGetLastError());
    return NF_OK;
}

// ------------------------------------------------------------------------------ A5 + A6
#define NF_F_NEWBLOCK 1
#define NF_F_LAST 2
#define NF_F_EXIT 4

struct __align__(16) StageHdr {
    int flags;
    int a, b;          // column image: source column = (cx + a, cy + b) wrapped
    int zu0, nc;       // unwrapped z index of the first table cell; number of cells in the table
    uint32_t g_lo;     // first padded slot held by this stage (multiple of 4)
    int g_cnt;         // slots held
    uint32_t col, s0, cnt;   // NEWBLOCK: the sink block
    int pad0, pad1;
};

struct __align__(128) Stage {
    float xs[NF_TILE];
    float ys[NF_TILE];
    float zs[NF_TILE];
    uint32_t tab[NF_TABMAX + 1];
    StageHdr hdr;
};

struct ProdState {       // cursor of the stage producer (block, column, z-run, chunk), kept in shared memory
    int mode;            // 0 next block, 1 next z-run, 5 z-run requested, 2 next chunk of the run, 3 end of block, 4 finished
    int flags, a, b, u, U1, Z1, ci, cj, ucur, run;
    int owner;           // warp whose register holds the requested table
    uint32_t col, s0, cnt, c0, ge;
};

struct InteractArgs {
    const float *sx, *sy, *sz, *lx, *ly, *lz;   // hi planes (staged into shared memory) and lo planes (close_scan only)
    const uint32_t *skey, *poff, *perm_pad, *order;
    const uint32_t *pair_slot;                  // sink pair -> padded slot of its first sink
    uint32_t n_part;                            // particles of the call (NF_DEBUG_BOUNDS: bound of the un-permute)
    const NfBlockDesc *blk;
    uint32_t *ctrl;
    const float *dyn;        // [0] rc^2 (cell units^2; 0 = no close-pair radius, use the min form)  [1] rc  [2] rc^-3
    float *acc;
    double kfac;             // gm / cell^2 (cell units -> length units); double: a float here is a relative error of up to 6e-8
                             // on EVERY acceleration, i.e. 1.2e-5 rms on a sink pulled at 200 rms by a close neighbour
    float addend;            // addend of r^2: NF_TAU (spline) or eps_p^2 in cell units (Plummer, Eq. 2)
    float b2;                // density radius^2 (cell units) + addend; DENS only
    double wfac;             // cell^2: density sum to length units
    int ostride;             // floats per output particle: 3, or 4 with the density estimate in the 4th
    int near_cheb;           // cells within this Chebyshev distance run the near-cell form
    double close_eps;        // eps_s in cell units for close_scan's Eq. 3 branch (0: no softening, NF_SOFT_NEWTON)
    unsigned long long *count_out;   // COUNT instantiation: [0] (sink, source) deliveries, [1] deliveries of a sink to itself
    NfParams prm;
};

// Close pairs (r < r_c) in double precision.  The hot loop clamps the
// float32 r^-3 of a near cell to fmax = r_c^-3 and tracks the smallest r^2 the lane saw in that
// cell; a lane whose minimum is below r_c^2 calls close_scan() for the flagged sources.  The scan
// repeats the loop's float32 arithmetic for d and r^2 (same operations, same order, so the same
// decision), and for every pair with r^2 < r_c^2 returns  exact F(d) d - fmax d_float,  i.e. it
// replaces what the hot loop added by the exact value.  The float32 cell-relative offsets of
// the staged planes are NOT enough for the exact value: for x < box/4 the input float32 position
// is finer than a float32 offset of magnitude ~0.5 cell, and 1.5e-8 cell is 3e-6 of the force
// of a pair 0.01 cell apart.  The binner therefore keeps the float32 remainder of every offset in
// the "lo" planes (hi + lo = the double-precision offset to 2^-48): one level of independent
// global loads per close source, no gather through the permutation; the INTEGER cell shift is
// added last.  Piecewise Eq. 3.  Rare (a few per cent of the sinks have such a
// neighbour), hence noinline and out of the hot loop.
struct CloseArgs {
    const float *sx, *sy, *sz;   // hi planes (global; the sink's own offsets)
    const float *lx, *ly, *lz;   // lo planes
    const uint32_t *ctrl;
    double eps;                // eps_s in cell units (0: no softening)
    double soft2;              // eps_p^2 in cell units (Plummer) or 0
    float addend;              // the loop's r^2 addend
    int law;
};
// double-precision r^-1 from the float32 seed by two Newton steps (relative error ~1e-14; no DP sqrt, no DP division)
__device__ __forceinline__ double rsqrt_f64(double x) {
    double y = (double)mufu_rsq((float)x);
    const double hx = 0.5 * x;
    y = y * fma(-hx * y, y, 1.5);
    y = y * fma(-hx * y, y, 1.5);
    return y;
}
__device__ __noinline__ void close_scan(const CloseArgs &K, const float *xs, const float *ys, const float *zs, int lo, int hi,
                                        uint32_t bits, int seg /* sources per flagged segment: a multiple of 4 */,
                                        float pxh, float pyh, float pzh /* the sink's own float32 offsets */,
                                        float xim, float yi, float zi, float rc2, float fmax, uint32_t g_lo, uint32_t sink_slot,
                                        int a, int b, int dzc, double *corr /* shared: [3][NF_BS], this thread's column */) {
    if (!(pxh < 0.5f * NF_BIG)) return;                   // a padding sink (its result is never stored)
    const double opx = (double)pxh + (double)K.lx[sink_slot], opy = (double)pyh + (double)K.ly[sink_slot], opz = (double)pzh + (double)K.lz[sink_slot];
    const double ie = K.eps > 0.0 ? 1.0 / K.eps : 0.0, ie3 = ie * ie * ie;
    const float2 nx = make_float2(-xim, -xim), ny = make_float2(-yi, -yi), nz = make_float2(-zi, -zi), tau = make_float2(K.addend, K.addend);
    double cx = 0.0, cy = 0.0, cz = 0.0;
    while (bits) {
        const int bit = __ffs(bits) - 1;
        bits &= bits - 1u;
        const int s0 = lo + bit * seg;
        const int s1 = (s0 + seg < hi) ? s0 + seg : hi;
        for (int sq = s0; sq < s1; sq += 4) {             // four sources at a time, the hot loop's packed arithmetic (same bits, same decision)
            const float4 X = *reinterpret_cast<const float4 *>(xs + sq), Y = *reinterpret_cast<const float4 *>(ys + sq),
                         Z = *reinterpret_cast<const float4 *>(zs + sq);
            const float2 dxa = __fadd2_rn(make_float2(X.x, X.y), nx), dxb = __fadd2_rn(make_float2(X.z, X.w), nx);
            const float2 dya = __fadd2_rn(make_float2(Y.x, Y.y), ny), dyb = __fadd2_rn(make_float2(Y.z, Y.w), ny);
            const float2 dza = __fadd2_rn(make_float2(Z.x, Z.y), nz), dzb = __fadd2_rn(make_float2(Z.z, Z.w), nz);
            float2 ra = __ffma2_rn(dxa, dxa, tau), rb = __ffma2_rn(dxb, dxb, tau);
            ra = __ffma2_rn(dya, dya, ra); rb = __ffma2_rn(dyb, dyb, rb);
            ra = __ffma2_rn(dza, dza, ra); rb = __ffma2_rn(dzb, dzb, rb);
            uint32_t m4 = (ra.x < rc2 ? 1u : 0u) | (ra.y < rc2 ? 2u : 0u) | (rb.x < rc2 ? 4u : 0u) | (rb.y < rc2 ? 8u : 0u);
            while (m4) {
                const int k = __ffs(m4) - 1;
                m4 &= m4 - 1u;
                const int s = sq + k;
                const float dxf = k == 0 ? dxa.x : (k == 1 ? dxa.y : (k == 2 ? dxb.x : dxb.y));
                const float dyf = k == 0 ? dya.x : (k == 1 ? dya.y : (k == 2 ? dyb.x : dyb.y));
                const float dzf = k == 0 ? dza.x : (k == 1 ? dza.y : (k == 2 ? dzb.x : dzb.y));
                // what the hot loop added for this pair (f clamped to fmax)
                cx -= (double)fmax * (double)dxf; cy -= (double)fmax * (double)dyf; cz -= (double)fmax * (double)dzf;
                const uint32_t q = g_lo + (uint32_t)s;        // padding never gets here (x = +BIG)
                NF_CHECK(K.ctrl, q < K.ctrl[3] && s >= 0 && s < NF_TILE, 8);
                if (q == sink_slot) continue;                 // the particle itself: F(0) = 0
                const double dx = (((double)xs[s] + (double)K.lx[q]) - opx) + (double)a;
                const double dy = (((double)ys[s] + (double)K.ly[q]) - opy) + (double)b;
                const double dz = (((double)zs[s] + (double)K.lz[q]) - opz) + (double)dzc;
                const double r2 = dx * dx + dy * dy + dz * dz;
                if (r2 == 0.0) continue;                      // coincident particles: F(0) = 0
                double f;
                if (K.law == NF_SOFT_PLUMMER) {
                    const double y = rsqrt_f64(r2 + K.soft2);     // Eq. 2
                    f = y * y * y;
                } else {
                    const double y = rsqrt_f64(r2);
                    const double u = r2 * y * ie;                 // r / eps_s (0 without softening)
                    f = (u < 1.0 && K.eps > 0.0) ? (10.0 + u * (-15.0 + 6.0 * u)) * ie3 : y * y * y;      // Eq. 3
                }
                cx += f * dx; cy += f * dy; cz += f * dz;
            }
        }
    }
    corr[0] += cx; corr[NF_BS] += cy; corr[2 * NF_BS] += cz;
}

__device__ __forceinline__ float fmin3(float a, float b, float c) {
    float d;
    asm("min.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
    return d;
}

// MODE 0: far cells, pure r^-3 (11 FMA-pipe ops per pair)
// MODE 1: near cells, Eq. 3 as min(r^-3, spline) (14 ops)        -- used when no close-pair radius is needed
// MODE 2: near cells, min(r^-3, r_c^-3) and the running minimum of r^2 (close pairs are fixed up by close_scan)
// MODE 3: as 2 for the sinks' own cells: the self pair (d == 0 exactly, contributes 0) does not count as close
// Sources [lo, lo + n) of the stage (lo may differ between lanes, n is warp-uniform and a
// multiple of 4; cells start on 16-byte boundaries) against the NF_SINKS sinks of this thread:
// four sources per LDS.128 and plane, shared by the thread's sinks.
constexpr int kS = NF_SINKS;
static_assert(NF_SINKS == 2, "the sink order is made of pairs: two sinks per thread");
constexpr int kQuads = NF_QUADS_PER_TRIP;
constexpr int kShortPass = 96;                       // passes up to this many sources flag close pairs per pass, longer ones per trip
template <int MODE, bool TRIPBITS, int LAW, bool DENS>
__device__ __forceinline__ void pair_loop(const float *__restrict__ xs, const float *__restrict__ ys, const float *__restrict__ zs, int lo, int n,
                                          const float (&xim)[kS], const float (&yi)[kS], const float (&zi)[kS], float2 (&ax)[kS],
                                          float2 (&ay)[kS], float2 (&az)[kS], const float2 c0, const float2 c1, const float2 c2,
                                          const float fmax, const float rc2, const int sh, uint32_t (&bits)[kS], const float addend,
                                          const float b2, float2 (&aw)[kS]) {
    const float2 tau = (LAW == 0) ? make_float2(NF_TAU, NF_TAU) : make_float2(addend, addend);   // an immediate for the spline
    const float2 b2v = make_float2(b2, b2);
    float2 nx[kS], ny[kS], nz[kS];
#pragma unroll
    for (int j = 0; j < kS; ++j) { nx[j] = make_float2(-xim[j], -xim[j]); ny[j] = make_float2(-yi[j], -yi[j]); nz[j] = make_float2(-zi[j], -zi[j]); }
    float m[kS];
#pragma unroll
    for (int j = 0; j < kS; ++j) m[j] = NF_BIG;
    auto pair2 = [&](const int j, const float2 X, const float2 Y, const float2 Z) {
        const float2 dx = __fadd2_rn(X, nx[j]), dy = __fadd2_rn(Y, ny[j]), dz = __fadd2_rn(Z, nz[j]);
        float2 r2 = __ffma2_rn(dx, dx, tau);
        r2 = __ffma2_rn(dy, dy, r2);
        r2 = __ffma2_rn(dz, dz, r2);
        const float2 ri = make_float2(mufu_rsq(r2.x), mufu_rsq(r2.y));
        const float2 ri2 = __fmul2_rn(ri, ri);
        float2 f = __fmul2_rn(ri2, ri);                    // r^-3
        if (MODE == 1 && LAW == 0) {
            const float2 r = __fmul2_rn(r2, ri);           // r
            float2 h = __ffma2_rn(r, c2, c1);
            h = __ffma2_rn(r, h, c0);                      // (10 - 15u + 6u^2)/eps^3
            f.x = fminf(f.x, h.x);                         // Eq. 3 as a min
            f.y = fminf(f.y, h.y);
        }
        if (MODE >= 2) {
            f.x = fminf(f.x, fmax);
            f.y = fminf(f.y, fmax);
            if (MODE == 2) m[j] = fmin3(m[j], r2.x, r2.y);
            else if (LAW == 0) m[j] = fmin3(m[j], r2.x > 2.f * NF_TAU ? r2.x : NF_BIG, r2.y > 2.f * NF_TAU ? r2.y : NF_BIG);
            else                                           // Plummer: r^2 carries eps_p^2, so the self pair is told by d == 0 (home cells only)
                m[j] = fmin3(m[j], (fabsf(dx.x) + fabsf(dy.x) + fabsf(dz.x) > 0.f) ? r2.x : NF_BIG,
                             (fabsf(dx.y) + fabsf(dy.y) + fabsf(dz.y) > 0.f) ? r2.y : NF_BIG);
        }
        if (DENS && MODE >= 1) {                           // b^2 - r^2 for r < b; the self pair's b^2 is taken off at the end
            const float2 t = __fadd2_rn(b2v, make_float2(-r2.x, -r2.y));
            aw[j] = __fadd2_rn(aw[j], make_float2(fmaxf(t.x, 0.f), fmaxf(t.y, 0.f)));
        }
        ax[j] = __ffma2_rn(f, dx, ax[j]);
        ay[j] = __ffma2_rn(f, dy, ay[j]);
        az[j] = __ffma2_rn(f, dz, az[j]);
    };
    const float *px = xs + lo, *py = ys + lo, *pz = zs + lo;
    auto quad = [&](const int t) {
        const float4 X = *reinterpret_cast<const float4 *>(px + t);
        const float4 Y = *reinterpret_cast<const float4 *>(py + t);
        const float4 Z = *reinterpret_cast<const float4 *>(pz + t);
#pragma unroll
        for (int j = 0; j < kS; ++j) {
            pair2(j, make_float2(X.x, X.y), make_float2(Y.x, Y.y), make_float2(Z.x, Z.y));
            pair2(j, make_float2(X.z, X.w), make_float2(Y.z, Y.w), make_float2(Z.z, Z.w));
        }
    };
    // A trip = kQuads source quads.  In modes 2/3 the loop records, per sink, where it saw a
    // close pair, so that close_scan revisits only those sources: TRIPBITS (long passes) sets
    // bit (trip >> sh) of `bits` after every trip (at most 32 segments per pass); short passes
    // keep one running minimum and flag the whole pass (bit 0).
    const int nfull = n / (4 * kQuads);
    if (MODE >= 2 && !TRIPBITS) {
#pragma unroll
        for (int j = 0; j < kS; ++j) m[j] = NF_BIG;
    }
    int trip = 0;
    for (; trip < nfull; ++trip) {
        const int t = trip * (4 * kQuads);
        if (MODE >= 2 && TRIPBITS) {
#pragma unroll
            for (int j = 0; j < kS; ++j) m[j] = NF_BIG;
        }
#pragma unroll
        for (int q = 0; q < kQuads; ++q) quad(t + 4 * q);
        if (MODE >= 2 && TRIPBITS) {
#pragma unroll
            for (int j = 0; j < kS; ++j) bits[j] |= (m[j] < rc2 ? 1u : 0u) << (trip >> sh);
        }
    }
    if (kQuads == 2 && (n & 4)) {
        if (MODE >= 2 && TRIPBITS) {
#pragma unroll
            for (int j = 0; j < kS; ++j) m[j] = NF_BIG;
        }
        quad(trip * 8);
        if (MODE >= 2 && TRIPBITS) {
#pragma unroll
            for (int j = 0; j < kS; ++j) bits[j] |= (m[j] < rc2 ? 1u : 0u) << (trip >> sh);
        }
    }
    if (MODE >= 2 && !TRIPBITS) {
#pragma unroll
        for (int j = 0; j < kS; ++j) bits[j] = m[j] < rc2 ? 1u : 0u;
    }
}

__device__ __forceinline__ void fold(float &tot, float &comp, float v, int kahan) {
    if (kahan) {
        float y = v - comp;
        float t = tot + y;
        comp = (t - tot) - y;
        tot = t;
    } else {
        tot += v;
    }
}

// FLAG = the regime k_choose_rc picked on the device: true = a close-pair radius is in use
// (near cells: clamp + close_scan), false = Eq. 3 as a min in near cells.  Both instantiations
// are launched; the one whose regime is not in force returns at once (no host round trip).
// LAW: NF_SOFT_SPLINE (Eq. 3) or NF_SOFT_PLUMMER (Eq. 2).  DENS: also accumulate the FoF-scale density
// estimate in the near cells and store it as the 4th output component.
// COUNT: a test instantiation (nf_debug_delivered_pairs) that runs the same ring, cursor and passes
// but, instead of the pair arithmetic, counts the real sources each pass delivers to each real
// sink: the pair count of what the kernel visited, measured rather than derived from the offsets.
template <bool FLAG, int LAW, bool DENS, bool COUNT>
__global__ void __launch_bounds__(NF_CTA_THREADS, NF_MIN_CTAS) k_interact(const InteractArgs A) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    Stage *stages = reinterpret_cast<Stage *>(smem_raw);
    __shared__ uint64_t full_bar[NF_NSTAGE], empty_bar[NF_NSTAGE];
    __shared__ double close_corr[3][NF_BS];
    __shared__ float tot[DENS ? 7 : 6][NF_BS];   // per sink: running sums x, y, z, their Kahan compensations, density sum
    if ((A.dyn[0] > 0.f) != FLAG) return;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int cpd = A.prm.cpd, R = A.prm.R;

    if (threadIdx.x == 0) {
        for (int s = 0; s < NF_NSTAGE; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], NF_NW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    int stage = 0;
    uint32_t phase = 0;

    // =========================== stage production by the consumer warps ========================
    // No dedicated producer warp: its registers go to the consumers (4 CTAs x 4 warps x 128
    // registers fill the register file).  A consumer warp that reaches a stage boundary with
    // fewer than NF_REFILL_BELOW produced stages ahead of it takes a lock and refills freed ring
    // slots, so the warps that would otherwise wait for data do the production work; the (block,
    // column, z-run, chunk) cursor lives in shared memory so that it costs no registers in the
    // pair loop.  produce_one() emits exactly one stage.
    __shared__ ProdState ps;
    __shared__ uint32_t ptab[32];
    __shared__ volatile uint32_t nprod_sh;     // stages produced so far
    __shared__ volatile int pdone_sh;          // the EXIT stage has been emitted
    __shared__ int plock;
    uint32_t cons = 0;                         // stages this warp has consumed
    if (threadIdx.x == 0) { nprod_sh = 0u; pdone_sh = 0; plock = 0; ps.owner = -1; ps.mode = 0; ps.flags = 0; }
    __syncthreads();
    int pstage = 0;
    uint32_t pphase = 0;
    uint32_t tvp = 0;        // table entry of the requested run (lane l: padded offset of its cell l), in flight between calls
    // advance the cursor to the next z-run of the block's source columns and request its table
    // (padded offsets of cells wz .. wz+run); mode 5 = requested, mode 3 = the block has no more runs
    auto issue_run = [&](ProdState &q) {
        if (q.u > q.U1) {
            q.u = q.Z1 - R;
            if (++q.b > R) { q.b = -R; ++q.a; }
            if (q.a > R) { q.mode = 3; return; }
        }
        int ia; const int sci = nf_wrap1(q.ci + q.a, cpd, ia);
        int ib; const int scj = nf_wrap1(q.cj + q.b, cpd, ib);
        const int cb = (sci * cpd + scj) * cpd;
        const int wz = nf_mod(q.u, cpd);
        int run = q.U1 - q.u + 1;
        if (run > cpd - wz) run = cpd - wz;
        if (run > NF_TABMAX) run = NF_TABMAX;
        tvp = A.poff[cb + wz + (lane <= run ? lane : run)];
        q.ucur = q.u; q.run = run;
        q.u += run;
        q.mode = 5;
        q.owner = warp;
    };
    auto produce_one = [&]() -> bool {
        Stage &S = stages[pstage];
        uint64_t *fb = &full_bar[pstage];
        auto emit = [&](int flags, int a, int b, int zu0, int nc, uint32_t tabval, uint32_t g_lo, int g_cnt, uint32_t col, uint32_t s0, uint32_t cnt) {
            S.tab[lane] = tabval;
            NF_CHECK(A.ctrl, g_cnt >= 0 && g_cnt <= NF_TILE && (g_lo & 3u) == 0u && g_lo + (uint32_t)g_cnt <= A.ctrl[3] + 8u, 1);
            NF_CHECK(A.ctrl, tabval <= (uint32_t)g_cnt, 2);
            if (lane == 0) {
                StageHdr h;
                h.flags = flags; h.a = a; h.b = b; h.zu0 = zu0; h.nc = nc; h.g_lo = g_lo; h.g_cnt = g_cnt;
                h.col = col; h.s0 = s0; h.cnt = cnt; h.pad0 = 0; h.pad1 = 0;
                S.hdr = h;
            }
            __syncwarp();
            if (lane == 0) {
                if (g_cnt > 0) {
                    const uint32_t bytes = (uint32_t)g_cnt * 4u;
                    mbar_arrive_expect_tx(fb, 3u * bytes);
                    bulk_g2s(S.xs, A.sx + g_lo, bytes, fb);
                    bulk_g2s(S.ys, A.sy + g_lo, bytes, fb);
                    bulk_g2s(S.zs, A.sz + g_lo, bytes, fb);
                } else {
                    mbar_arrive(fb);
                }
            }
        };
        ProdState q = ps;
        bool last = false;
        for (;;) {
            if (q.mode == 0) {                       // next sink block
                uint32_t w = 0;
                if (lane == 0) w = atomicAdd(&A.ctrl[0], 1u);
                w = __shfl_sync(0xffffffffu, w, 0);
                if (w >= A.ctrl[1]) { emit(NF_F_EXIT, 0, 0, 0, 0, 0u, 0u, 0, 0u, 0u, 0u); q.mode = 4; last = true; break; }
                const NfBlockDesc d = A.blk[A.order[w]];
                if (d.cnt == 0) continue;
                q.col = d.col; q.s0 = d.s0; q.cnt = d.cnt;
                q.ci = (int)(d.col / (uint32_t)cpd); q.cj = (int)(d.col % (uint32_t)cpd);
                const int colbase = (int)d.col * cpd;
                q.Z1 = (int)(A.skey[A.pair_slot[d.s0 >> 1]] & ~NF_PAD_FLAG) - colbase;
                q.U1 = (int)(A.skey[A.pair_slot[(d.s0 + d.cnt - 1) >> 1]] & ~NF_PAD_FLAG) - colbase + R;
                q.a = -R; q.b = -R; q.u = q.Z1 - R; q.flags = NF_F_NEWBLOCK; q.mode = 1;
            }
            if (q.mode == 1) issue_run(q);           // (only right after a block start or an empty run: not prefetched)
            if (q.mode == 5) {                       // the run's table has been requested: is the run non-empty?
                if (q.owner != warp) {               // requested by another warp: fetch it again (cache-hot by now)
                    int ia; const int sci = nf_wrap1(q.ci + q.a, cpd, ia);
                    int ib; const int scj = nf_wrap1(q.cj + q.b, cpd, ib);
                    tvp = A.poff[(sci * cpd + scj) * cpd + nf_mod(q.ucur, cpd) + (lane <= q.run ? lane : q.run)];
                }
                const uint32_t g0 = __shfl_sync(0xffffffffu, tvp, 0);
                const uint32_t g1 = __shfl_sync(0xffffffffu, tvp, q.run);
                if (g1 <= g0) { q.mode = 1; continue; }
                q.c0 = g0 & ~3u; q.ge = (g1 + 3u) & ~3u;
                ptab[lane] = tvp;
                __syncwarp();
                q.mode = 2;
            }
            if (q.mode == 2) {                       // next chunk of the run
                const uint32_t c1 = (q.c0 + NF_TILE < q.ge) ? q.c0 + NF_TILE : q.ge;
                // table entry = first slot of the cell relative to this stage, clamped to the stage
                int tl = (int)(ptab[lane] - q.c0);
                const int tc = (int)(c1 - q.c0);
                tl = tl < 0 ? 0 : (tl > tc ? tc : tl);
                emit(q.flags, q.a, q.b, q.ucur, q.run, (uint32_t)tl, q.c0, tc, q.col, q.s0, q.cnt);
                q.flags = 0;
                q.c0 += NF_TILE;
                if (q.c0 >= q.ge) { q.mode = 1; issue_run(q); }     // request the next run's table now, use it at the next call
                break;
            }
            if (q.mode == 3) {                       // end of the block
                emit(q.flags | NF_F_LAST, 0, 0, 0, 0, 0u, 0u, 0, q.col, q.s0, q.cnt);
                q.mode = 0;
                break;
            }
        }
        if (lane == 0) ps = q;
        __syncwarp();
        return last;
    };

    // =============================== consumer warps ==========================================
    // Thread t of warp w holds the kS sinks of pair (s0 + (32 w + t) kS) / 2 of the sink order: two
    // adjacent padded slots of one cell (the second may be the padding slot of an odd cell).
    const float2 c0 = make_float2(A.prm.c0, A.prm.c0), c1 = make_float2(A.prm.c1, A.prm.c1), c2 = make_float2(A.prm.c2, A.prm.c2);
    const int near_cheb = A.near_cheb, kahan = A.prm.kahan;
    const float rc2 = A.dyn[3];
    const float fmax = A.dyn[2];
    CloseArgs K;
    K.ctrl = A.ctrl; K.sx = A.sx; K.sy = A.sy; K.sz = A.sz; K.lx = A.lx; K.ly = A.ly; K.lz = A.lz; K.eps = A.close_eps;
    K.law = LAW; K.addend = A.addend; K.soft2 = (LAW == NF_SOFT_PLUMMER) ? (double)A.addend : 0.0;
    const int tid_s = (int)threadIdx.x * kS;           // this thread's first column of close_corr / tot
    float px[kS], py[kS], pz[kS];
#pragma unroll
    for (int j = 0; j < kS; ++j) { px[j] = -NF_BIG; py[j] = 0.f; pz[j] = 0.f; }
    int zl = 0, z1 = 0, z2 = -1;
    bool valid = false;
    uint32_t slot = 0;
    const int W = 2 * R + 1;
    unsigned long long n_deliv = 0ull, n_self = 0ull;   // COUNT only

    for (;;) {
        while (!pdone_sh) {
            uint32_t np = nprod_sh;
            np = __shfl_sync(0xffffffffu, np, 0);
            if (np - cons >= (uint32_t)NF_REFILL_BELOW) break;              // enough stages ahead of this warp (or the ring is full)
            int got = 0;
            if (lane == 0) got = (atomicCAS(&plock, 0, 1) == 0) ? 1 : 0;
            got = __shfl_sync(0xffffffffu, got, 0);
            if (!got) { if (np == cons) continue; else break; }              // someone else is refilling; spin only if starved
            __threadfence_block();
            np = nprod_sh;
            np = __shfl_sync(0xffffffffu, np, 0);
            bool released = false;
            if (!pdone_sh && np - cons < (uint32_t)NF_NSTAGE) {
                pstage = (int)(np % NF_NSTAGE);
                pphase = (np / NF_NSTAGE) & 1u;
                bool ok = mbar_test(&empty_bar[pstage], pphase ^ 1u);
                if (!ok && np == cons) { mbar_wait(&empty_bar[pstage], pphase ^ 1u); ok = true; }   // starved: wait for the slot
                if (ok) {
                    const bool last = produce_one();
                    if (lane == 0) { if (last) pdone_sh = 1; __threadfence_block(); nprod_sh = np + 1u; }
                    __syncwarp();
                } else {
                    released = true;          // slot still in use and there is something to consume: try again later
                }
            } else {
                released = true;
            }
            if (lane == 0) { __threadfence_block(); atomicExch(&plock, 0); }
            __syncwarp();
            if (released) break;
        }
        Stage &S = stages[stage];
        mbar_wait(&full_bar[stage], phase);
        const int flags = S.hdr.flags;
        if (flags & NF_F_EXIT) break;
        if (flags & NF_F_NEWBLOCK) {
            const uint32_t off = (uint32_t)(warp * 32 + lane) * kS;
            valid = off < S.hdr.cnt;
            NF_CHECK(A.ctrl, ((S.hdr.s0 + (valid ? off : 0u)) >> 1) < (A.ctrl[4] + 1u) / 2u, 3);
            slot = A.pair_slot[(S.hdr.s0 + (valid ? off : 0u)) >> 1];
            NF_CHECK(A.ctrl, slot + 1u < A.ctrl[3] && (slot & 1u) == 0u, 4);
            const int colbase = (int)S.hdr.col * cpd;
            zl = (int)(A.skey[slot] & ~NF_PAD_FLAG) - colbase;
            NF_CHECK(A.ctrl, zl >= 0 && zl < cpd, 5);
#pragma unroll
            for (int j = 0; j < kS; ++j) {
                px[j] = valid ? A.sx[slot + j] : -NF_BIG;   // an idle lane sits at -BIG: contributes and receives exactly 0
                py[j] = A.sy[slot + j];
                pz[j] = A.sz[slot + j];
            }
            const unsigned vm = __ballot_sync(0xffffffffu, valid);
            z1 = 0; z2 = -4 * NF_MAX_R - 4;          // no valid sink in this warp: empty z range for every stage
            if (vm != 0u) {
                z1 = __shfl_sync(0xffffffffu, zl, 0);
                z2 = __shfl_sync(0xffffffffu, zl, 31 - __clz(vm));
                if (!valid) zl = z2;
            }
#pragma unroll
            for (int j = 0; j < kS; ++j) {
#pragma unroll
                for (int q = 0; q < (DENS ? 7 : 6); ++q) tot[q][tid_s + j] = 0.f;
#pragma unroll
                for (int q = 0; q < 3; ++q) close_corr[q][tid_s + j] = 0.0;
            }
        }
        const int zu0 = S.hdr.zu0;
        int cz0 = z1 - R, cz1 = z2 + R;              // source cells this warp needs ...
        if (cz0 < zu0) cz0 = zu0;
        if (cz1 > zu0 + S.hdr.nc - 1) cz1 = zu0 + S.hdr.nc - 1;   // ... that this stage holds
        if (S.hdr.g_cnt > 0 && cz0 <= cz1) {
            const int ha = S.hdr.a, hb = S.hdr.b;
            float xi[kS], yi[kS];
#pragma unroll
            for (int j = 0; j < kS; ++j) { xi[j] = px[j] - (float)ha; yi[j] = py[j] - (float)hb; }
            // near cells: may hold r < eps_s; home cells: the sinks' own cells (self pairs)
            int nz0 = 1 << 30, nz1 = -(1 << 30), hz0 = 1 << 30, hz1 = -(1 << 30);
            if (abs(ha) <= near_cheb && abs(hb) <= near_cheb) { nz0 = z1 - near_cheb; nz1 = z2 + near_cheb; }
            if (ha == 0 && hb == 0) { hz0 = z1; hz1 = z2; }
            // far cells 0; near cells: 1 without a close-pair radius (Eq. 3 as a min; Plummer: density only), 2/3 with one
            auto mode_of = [&](int zu) { return (zu < nz0 || zu > nz1) ? 0 : (!FLAG ? ((LAW == 0 || DENS) ? 1 : 0) : ((zu >= hz0 && zu <= hz1) ? 3 : 2)); };
            const int *tab = reinterpret_cast<const int *>(S.tab) - zu0;   // tab[zu] = first stage-local slot of source cell zu
            float2 ax[kS], ay[kS], az[kS], aw[kS];
#pragma unroll
            for (int j = 0; j < kS; ++j) { ax[j] = make_float2(0.f, 0.f); ay[j] = ax[j]; az[j] = ax[j]; aw[j] = ax[j]; }

            // One pass = sources [lo, lo + n) where a lane reads cell cA's part (from loA) if its
            // sink is within R cells of cA, else cell cB's part (from loB) if within R of cB, else
            // it is masked.  cB = cA + 2R+1, so the two lane groups are disjoint: the edge cells
            // of the warp's window, each needed by only part of the warp, are processed two at a
            // time and no lane idles.
            auto pass = [&](const int ploA, const int pcA, const int ploB, const int pcB, const int n, const int mode) __attribute__((always_inline)) {
                const bool useA = abs(zl - pcA) <= R, useB = abs(zl - pcB) <= R;
                const int cell = useA ? pcA : pcB;
                const int lo = useA ? ploA : ploB;
                const int dzc = cell - zl;
                NF_CHECK(A.ctrl, !(useA || useB) || (lo >= 0 && n > 0 && (lo & 3) == 0 && (n & 3) == 0 && lo + n <= S.hdr.g_cnt), 6);
                float xim[kS], zi[kS];
                uint32_t bits[kS];
#pragma unroll
                for (int j = 0; j < kS; ++j) {
                    xim[j] = (useA || useB) ? xi[j] : -NF_BIG;    // masked sink at -BIG, padding sources at +BIG: never coincide
                    zi[j] = pz[j] - (float)dzc;
                    bits[j] = 0u;
                }
                if (COUNT) {
                    uint32_t nreal = 0;
                    for (int s = lo; s < lo + n; ++s) nreal += S.xs[s] < 0.5f * NF_BIG ? 1u : 0u;
#pragma unroll
                    for (int j = 0; j < kS; ++j)
                        if ((useA || useB) && valid && fabsf(px[j]) < 0.5f * NF_BIG) {      // a real sink that this pass serves
                            n_deliv += nreal;
                            const uint32_t rel = slot + j - S.hdr.g_lo;                    // the sink's own slot, stage-local
                            if (rel >= (uint32_t)lo && rel < (uint32_t)(lo + n) && dzc == 0 && ha == 0 && hb == 0) n_self += 1ull;
                        }
                    return;
                }
                if (mode == 0) pair_loop<0, false, LAW, DENS>(S.xs, S.ys, S.zs, lo, n, xim, yi, zi, ax, ay, az, c0, c1, c2, fmax, rc2, 0, bits, A.addend, A.b2, aw);
                else if (!FLAG) pair_loop<1, false, LAW, DENS>(S.xs, S.ys, S.zs, lo, n, xim, yi, zi, ax, ay, az, c0, c1, c2, fmax, rc2, 0, bits, A.addend, A.b2, aw);
                else {
                    int seg = n;                     // sources per flagged segment
                    if (n <= kShortPass) {
                        if (mode == 3) pair_loop<3, false, LAW, DENS>(S.xs, S.ys, S.zs, lo, n, xim, yi, zi, ax, ay, az, c0, c1, c2, fmax, rc2, 0, bits, A.addend, A.b2, aw);
                        else pair_loop<2, false, LAW, DENS>(S.xs, S.ys, S.zs, lo, n, xim, yi, zi, ax, ay, az, c0, c1, c2, fmax, rc2, 0, bits, A.addend, A.b2, aw);
                    } else {
                        const int ntr = (n + 4 * kQuads - 1) / (4 * kQuads);
                        const int sh = ntr > 32 ? 32 - __clz((ntr - 1) >> 5) : 0;     // (trips >> sh) < 32
                        seg = (4 * kQuads) << sh;
                        if (mode == 3) pair_loop<3, true, LAW, DENS>(S.xs, S.ys, S.zs, lo, n, xim, yi, zi, ax, ay, az, c0, c1, c2, fmax, rc2, sh, bits, A.addend, A.b2, aw);
                        else pair_loop<2, true, LAW, DENS>(S.xs, S.ys, S.zs, lo, n, xim, yi, zi, ax, ay, az, c0, c1, c2, fmax, rc2, sh, bits, A.addend, A.b2, aw);
                    }
#pragma unroll
                    for (int j = 0; j < kS; ++j)
                        if (bits[j])
                            close_scan(K, S.xs, S.ys, S.zs, lo, lo + n, bits[j], seg, px[j], py[j], pz[j], xim[j], yi[j], zi[j], rc2, fmax, S.hdr.g_lo, slot + j,
                                       ha, hb, dzc, &close_corr[0][tid_s + j]);
                }
            };
            // cells cz0 + i with (i div W) even are "A" cells; each takes the cell W further on as partner
            for (int base = cz0; base <= cz1; base += 2 * W) {
                const int lastA = (base + W - 1 < cz1) ? base + W - 1 : cz1;
                for (int cA = base; cA <= lastA; ++cA) {
                    const int cB = cA + W;
                    const int a0 = tab[cA], a1 = tab[cA + 1];
                    int b0 = 0, b1 = 0;
                    const int mA = mode_of(cA);
                    int mB = 0;
                    if (cB <= cz1) { b0 = tab[cB]; b1 = tab[cB + 1]; mB = mode_of(cB); }
                    const int nA = a1 - a0, nB = b1 - b0;
                    const int ncm = nA < nB ? nA : nB;
                    // the common length of the two cells, both lane groups at once; then the rest of
                    // the longer cell, its own lanes only
                    if (ncm > 0) pass(a0, cA, b0, cB, ncm, mA > mB ? mA : mB);
                    if (nA != nB) {       // one call site for either remainder keeps the kernel's code (and its i-cache footprint) smaller
                        const bool ra = nA > nB;
                        pass((ra ? a0 : b0) + ncm, ra ? cA : cB, 0, -(1 << 28), ra ? nA - ncm : nB - ncm, ra ? mA : mB);
                    }
                }
            }
#pragma unroll
            for (int j = 0; j < kS; ++j) {
                const float v[3] = {ax[j].x + ax[j].y, ay[j].x + ay[j].y, az[j].x + az[j].y};
#pragma unroll
                for (int q = 0; q < 3; ++q) {
                    float t = tot[q][tid_s + j], c = tot[q + 3][tid_s + j];
                    fold(t, c, v[q], kahan);
                    tot[q][tid_s + j] = t; tot[q + 3][tid_s + j] = c;
                }
                if (DENS) tot[DENS ? 6 : 0][tid_s + j] += aw[j].x + aw[j].y;
            }
        }
        if ((flags & NF_F_LAST) && !COUNT) {
            if (valid) {
#pragma unroll
                for (int j = 0; j < kS; ++j) {
                    const uint32_t dst = A.perm_pad[slot + j];
                    NF_CHECK(A.ctrl, dst == 0xffffffffu || dst < A.n_part, 7);
                    if (dst != 0xffffffffu) {
                        float *o = A.acc + (size_t)A.ostride * dst;
                        o[0] = (float)(A.kfac * ((double)tot[0][tid_s + j] + close_corr[0][tid_s + j]));
                        o[1] = (float)(A.kfac * ((double)tot[1][tid_s + j] + close_corr[1][tid_s + j]));
                        o[2] = (float)(A.kfac * ((double)tot[2][tid_s + j] + close_corr[2][tid_s + j]));
                        // density: the sink met itself exactly once (r = 0 -> b^2); take that off (reading D1)
                        if (DENS) o[3] = (float)(A.wfac * ((double)tot[DENS ? 6 : 0][tid_s + j] - ((double)A.b2 - (double)A.addend)));
                    }
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty_bar[stage]);
        if (++stage == NF_NSTAGE) { stage = 0; phase ^= 1u; }
        ++cons;
    }
    if (COUNT) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) { n_deliv += __shfl_xor_sync(0xffffffffu, n_deliv, d); n_self += __shfl_xor_sync(0xffffffffu, n_self, d); }
        if (lane == 0) { atomicAdd(A.count_out, n_deliv); atomicAdd(A.count_out + 1, n_self); }
    }
}

static int g_interact_blocks_per_sm = 0;

typedef void (*InteractKernel)(const InteractArgs);
// [law][dens][flag]
static InteractKernel interact_kernel(int law, int dens, int flag) {
    static const InteractKernel tab[2][2][2] = {
        {{k_interact<false, NF_SOFT_SPLINE, false, false>, k_interact<true, NF_SOFT_SPLINE, false, false>},
         {k_interact<false, NF_SOFT_SPLINE, true, false>, k_interact<true, NF_SOFT_SPLINE, true, false>}},
        {{k_interact<false, NF_SOFT_PLUMMER, false, false>, k_interact<true, NF_SOFT_PLUMMER, false, false>},
         {k_interact<false, NF_SOFT_PLUMMER, true, false>, k_interact<true, NF_SOFT_PLUMMER, true, false>}}};
    return tab[law][dens][flag];
}
static InteractKernel count_kernel(int flag) {
    return flag ? k_interact<true, NF_SOFT_SPLINE, false, true> : k_interact<false, NF_SOFT_SPLINE, false, true>;
}

nf_status nf_interact_setup(nf_ctx *ctx) {
    const size_t smem = sizeof(Stage) * NF_NSTAGE;
    int nb = 1 << 30;
    for (int law = 0; law < 2; ++law)
        for (int dens = 0; dens < 2; ++dens)
            for (int flag = 0; flag < 2; ++flag) {
                InteractKernel k = interact_kernel(law, dens, flag);
                NF_CUDA_OK(ctx, cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                int n1 = 0;
                NF_CUDA_OK(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n1, k, NF_CTA_THREADS, smem));
                if (n1 < nb) nb = n1;
            }
    for (int flag = 0; flag < 2; ++flag) NF_CUDA_OK(ctx, cudaFuncSetAttribute(count_kernel(flag), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (nb < 1) { snprintf(ctx->err, sizeof(ctx->err), "interaction kernel does not fit on an SM"); return NF_ECUDA; }
    g_interact_blocks_per_sm = nb;
    return NF_OK;
}

static void fill_interact_args(nf_ctx *ctx, const float *d_pos, float *d_out, int ostride, double kfac, InteractArgs &A, int &law, int &dens) {
    (void)d_pos;
    A.sx = ctx->d_sorted; A.sy = ctx->d_sorted + ctx->capPad; A.sz = ctx->d_sorted + 2ull * ctx->capPad;
    A.lx = ctx->d_sorted + 4ull * ctx->capPad; A.ly = ctx->d_sorted + 5ull * ctx->capPad; A.lz = ctx->d_sorted + 6ull * ctx->capPad;
    A.skey = (const uint32_t *)(ctx->d_sorted + 3ull * ctx->capPad);
    A.poff = ctx->d_poff; A.perm_pad = ctx->d_perm_pad; A.order = ctx->d_blk_order; A.blk = ctx->d_blk; A.pair_slot = ctx->d_pair_slot;
    A.n_part = (uint32_t)ctx->lastN;
    A.ctrl = ctx->d_ctrl; A.dyn = (const float *)(ctx->d_ctrl + 96); A.acc = d_out; A.kfac = kfac; A.prm = ctx->prm;
    A.prm.kahan = ctx->opt_kahan;
    A.ostride = ostride;
    A.count_out = ctx->d_pairs + 6;
    // the unsoftened law runs the spline instantiation in its close-pair regime (k_choose_rc keeps
    // r_c > 0 for it): r^-3 clamped at r_c^-3 in the near cells, exact 1/r^2 from close_scan below r_c
    law = ctx->law == NF_SOFT_PLUMMER ? 1 : 0;
    dens = (ostride == 4 && ctx->dens_b > 0.0) ? 1 : 0;
    const double ep = ctx->eps_p * ctx->prm.scale;            // eps_p in cell units
    A.addend = law ? (float)(ep * ep) : NF_TAU;
    A.close_eps = ctx->law == NF_SOFT_NEWTON ? 0.0 : ctx->prm.eps_cells;
    const double bc = ctx->dens_b * ctx->prm.scale;           // density radius in cell units
    A.b2 = (float)(bc * bc) + A.addend;
    const double cellsz = ctx->box / (double)ctx->cpd;
    A.wfac = cellsz * cellsz;
    // near cells: may hold r < eps_s (spline), r < r_c <= 0.25 (Plummer, Newton), or r < b (density)
    int nc = ctx->law == NF_SOFT_SPLINE ? ctx->prm.near_cheb : 1;
    if (dens) { const int nb = (int)ceil(bc); if (nb > nc) nc = nb; }
    if (nc > ctx->R) nc = ctx->R;
    A.near_cheb = nc;
}

// d_out: N x ostride floats (ostride 3: accelerations; 4: accelerations + density estimate)
nf_status nf_run_interact(nf_ctx *ctx, const float *d_pos, int64_t N, float *d_out, int ostride, double kfac, cudaStream_t st) {
    InteractArgs A;
    int law, dens;
    fill_interact_args(ctx, d_pos, d_out, ostride, kfac, A, law, dens);
    const int grid = ctx->sm_count * g_interact_blocks_per_sm;
    for (int flag = 1; flag >= 0; --flag) {     // the instantiation whose regime is not in force returns at once
        interact_kernel(law, dens, flag)<<<grid, NF_CTA_THREADS, sizeof(Stage) * NF_NSTAGE, st>>>(A); ctx->launches++;
    }
    NF_CUDA_OK(ctx, cudaGetLastError());
    return NF_OK;
}

// nf_debug_delivered_pairs: the COUNT instantiation over the sink blocks of the last nf_accel
nf_status nf_run_count(nf_ctx *ctx, cudaStream_t st) {
    InteractArgs A;
    int law, dens;
    fill_interact_args(ctx, nullptr, nullptr, 3, 0.f, A, law, dens);
    NF_CUDA_OK(ctx, cudaMemsetAsync(ctx->d_ctrl, 0, sizeof(uint32_t), st));             // the work counter
    NF_CUDA_OK(ctx, cudaMemsetAsync(A.count_out, 0, 2 * sizeof(unsigned long long), st));
    const int grid = ctx->sm_count * g_interact_blocks_per_sm;
    for (int flag = 1; flag >= 0; --flag) {
        count_kernel(flag)<<<grid, NF_CTA_THREADS, sizeof(Stage) * NF_NSTAGE, st>>>(A); ctx->launches++;
    }
    NF_CUDA_OK(ctx, cudaGetLastError());
    return NF_OK;
}

// ------------------------------------------------------------------------------ exports
// Neighbour list of one sink cell, enumerated exactly as the producer warp does: column images
// by nf_wrap1, z by nf_mod of the unwrapped index.
__global__ void k_neighbors(int cpd, int R, int cell, int32_t *out) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const int ck = cell % cpd, cj = (cell / cpd) % cpd, ci = cell / (cpd * cpd);
    int n = 0;
    const int w = 2 * R + 1, nn = w * w * w;
    for (int a = -R; a <= R; ++a) {
        int ia; const int sci = nf_wrap1(ci + a, cpd, ia);
        for (int b = -R; b <= R; ++b) {
            int ib; const int scj = nf_wrap1(cj + b, cpd, ib);
            const int cb = (sci * cpd + scj) * cpd;
            for (int u = ck - R; u <= ck + R; ++u, ++n) {
                const int wz = nf_mod(u, cpd);
                out[n] = cb + wz;
                out[nn + 3 * n + 0] = ia;
                out[nn + 3 * n + 1] = ib;
                out[nn + 3 * n + 2] = (u - wz) / cpd;
            }
        }
    }
}

nf_status nf_run_neighbors(nf_ctx *ctx, int cell, cudaStream_t st) {
    k_neighbors<<<1, 32, 0, st>>>(ctx->cpd, ctx->R, cell, ctx->d_nbr); ctx->launches++;
    NF_CUDA_OK(ctx, cudaGetLastError());
    return NF_OK;
}

// out[0] = sum over sink cells c of n_c * sum_{c' in N(c)} n_c', out[1] = number of sinks (the caller subtracts it)
__global__ void __launch_bounds__(256) k_paircount(int cpd, int R, int x0, int nx, const uint32_t *__restrict__ offsets, unsigned long long *__restrict__ out) {
    const int ncell = cpd * cpd * cpd;
    int c = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long v = 0, ns = 0;
    if (c < ncell) {
        const unsigned long long nc = offsets[c + 1] - offsets[c];
        if (nc && nf_sink_slab(c / (cpd * cpd), cpd, x0, nx)) {
            ns = nc;
            const int ck = c % cpd, cj = (c / cpd) % cpd, ci = c / (cpd * cpd);
            unsigned long long s = 0;
            for (int a = -R; a <= R; ++a) {
                int ia; const int sci = nf_wrap1(ci + a, cpd, ia);
                for (int b = -R; b <= R; ++b) {
                    int ib; const int scj = nf_wrap1(cj + b, cpd, ib);
                    const int cb = (sci * cpd + scj) * cpd;
                    for (int u = ck - R; u <= ck + R; ++u) {
                        const int wz = nf_mod(u, cpd);
                        s += offsets[cb + wz + 1] - offsets[cb + wz];
                    }
                }
            }
            v = nc * s;
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) { v += __shfl_xor_sync(0xffffffffu, v, d); ns += __shfl_xor_sync(0xffffffffu, ns, d); }
    if ((threadIdx.x & 31) == 0 && ns) { atomicAdd(out, v); atomicAdd(out + 1, ns); }
}

nf_status nf_run_paircount(nf_ctx *ctx, cudaStream_t st) {
    NF_CUDA_OK(ctx, cudaMemsetAsync(ctx->d_pairs, 0, 2 * sizeof(unsigned long long), st));
    const int ncell = (int)ctx->ncell;
    k_paircount<<<(ncell + 255) / 256, 256, 0, st>>>(ctx->cpd, ctx->R, ctx->slab_x0, ctx->slab_nx, ctx->d_offsets, ctx->d_pairs); ctx->launches++;
    NF_CUDA_OK(ctx, cudaGetLastError());
    return NF_OK;
}
