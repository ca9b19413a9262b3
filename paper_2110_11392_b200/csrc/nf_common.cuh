// nf_common.cuh -- shared declarations of the CUDA near-field path (sm_100a only).
// Not shared with oracle/ in any way.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include "../../include/nearfield.h"

#if defined(__CUDA_ARCH__) && (__CUDA_ARCH__ < 1000)
#error "this library is written for sm_100a (B200) only"
#endif

// ---- layout constants -------------------------------------------------------------------
#define NF_PAD_FLAG 0x80000000u   // high bit of the cell-key plane marks a padding slot
#define NF_BIG 1.0e18f            // x offset of padding sources (+BIG) and masked sinks (-BIG): r^-3 underflows to exactly 0
#define NF_TAU 1.0e-30f           // addend of the first r^2 product: self pairs give f*d = c0*0 = 0, no NaN
#define NF_SPLINE_PER_PLUMMER 2.16  // eps_s = 2.16 eps_p

// interaction kernel geometry
#ifndef NF_NW
#define NF_NW 4                   // consumer warps per CTA
#endif
#ifndef NF_REFILL_BELOW
#define NF_REFILL_BELOW 2          // a warp tries to refill when fewer than this many produced stages lie ahead of it
#endif
#define NF_CTA_THREADS (NF_NW * 32)
#ifndef NF_SINKS
#define NF_SINKS 2                // sinks per consumer thread (adjacent slots 2t, 2t+1 of the warp's range when 2)
#endif
#define NF_BS (NF_NW * 32 * NF_SINKS)   // sinks per CTA work item
#ifndef NF_QUADS_PER_TRIP
#define NF_QUADS_PER_TRIP 2     // source quads per unrolled trip of the pair loop (1 or 2)
#endif
#ifndef NF_TILE
#define NF_TILE 640               // source slots per pipeline stage (per coordinate plane)
#endif
#define NF_TABMAX 31              // source cells per segment table (32 entries = one per producer lane)
#ifndef NF_NSTAGE
#define NF_NSTAGE 5               // pipeline depth
#endif
#ifndef NF_CELL_PAD
#define NF_CELL_PAD 4             // every cell is padded to a multiple of this many slots (power of two, >= 2)
#endif
#ifndef NF_MIN_CTAS
#define NF_MIN_CTAS 4             // resident CTAs per SM the interaction kernel is compiled for
#endif

#define NF_HOST_CHUNKS 8          // nf_accel_host: ranges the H2D copy is cut into (A1 runs per range)

struct NfParams {
    int cpd, R, ncell, ncol;
    double scale;        // cpd / box
    double eps_cells;    // eps_s in cell units
    float c0, c1, c2;    // spline coefficients in cell units: 10/e^3, -15/e^4, 6/e^5, e = eps_s/cell
    int near_cheb;       // source cells at Chebyshev distance <= near_cheb may hold r < eps_s
    int kahan;
};

struct NfBlockDesc {     // one sink work item: <= NF_BS consecutive padded slots of one z-column
    uint32_t col;        // cx*cpd + cy
    uint32_t s0;         // first slot in the SINK order (cells padded to 2 slots; d_pair_slot maps a pair to its padded slot)
    uint32_t cnt;        // number of sink-order slots
    uint32_t cost;       // estimated cost (sinks x sources in the z-window of the home column), saturating
};

struct nf_ctx {
    int device, cpd, R, sm_count;
    double eps_p, box, gm;
    int law;                     // NF_SOFT_SPLINE | NF_SOFT_PLUMMER
    double dens_b;               // FoF-scale density radius (length units); 0 = off
    int slab_x0, slab_nx;        // sink slabs: x cell indices [x0, x0 + nx) periodic; nx = cpd: all
    int64_t ncell, ncol;
    NfParams prm;
    // options
    int opt_stage_timing, opt_kahan, opt_heavy_first;
    float opt_rc;                // close-pair radius in cells; < 0 = automatic
    // scratch (grow-only)
    int64_t capN, capPad, capBlk, capScan;
    uint32_t *d_key, *d_arr, *d_counts, *d_offsets, *d_poff, *d_tmp_perm, *d_chunk_sorted, *d_perm_true, *d_perm_pad;
    unsigned long long *d_scan_in, *d_scan_blk;
    // nf_rebin (allocated at its first use): the other half of the offsets / permutation double buffers,
    // the insert list, per-cell stayer counts + bucket fill counters
    uint32_t *d_offsets_alt, *d_perm_alt, *d_ins, *d_nstay;
    int64_t capRebin;
    int bin_valid;               // d_offsets / d_perm_true hold the grid order of bin_validN particles
    int64_t bin_validN;
    float *d_sorted;             // 4 planes of capPad: x, y, z (cell units), cell key (uint32 bits)
    uint32_t *d_col_nblk, *d_col_base, *d_scan32_blk, *d_blk_order;
    uint32_t *d_mp_hist;         // nf_multipoles: occupancy-class histogram of the cells (260 words)
    uint32_t *d_poff2;           // sink order: exclusive scan of the occupancies rounded up to even (A4)
    uint32_t *d_pair_slot;       // sink pair i (sink-order slots 2i, 2i+1) -> padded slot of its first sink (A4)
    NfBlockDesc *d_blk;
    uint32_t *d_ctrl;            // [0] work counter  [1] number of blocks  [2] bad-position flag  [3] npad
                                 // [4] sink-order slot count  [8] NF_DEBUG_BOUNDS: code of a failed bounds check
                                 // [5] insert-list tail (nf_rebin)  [6] dense-cell count (nf_multipoles)  [7] long-cell count (rank)
                                 // [16..79] cost histogram  [96..98] float rc^2, rc, rc^-3  [100..101] u64 sum n_c^2  [104] work counter of nf_accel_f64
    unsigned long long *d_pairs;
    int32_t *d_nbr;              // debug neighbour list
    // host staging for nf_accel_host
    float *d_pos_buf, *d_acc_buf;
    int64_t capHost;
    cudaStream_t own_stream;
    cudaStream_t copy_stream;    // nf_accel_host: H2D ranges, each followed by A1 on the compute stream
    cudaEvent_t ev_chunk[NF_HOST_CHUNKS];
    cudaEvent_t ev_order;        // orders a call after the previous one when the stream changes
    // state of the last call
    cudaStream_t last_stream;
    int64_t lastN;
    int have_last;
    int bin_pinned;              // nf_bin: the binning of (bin_pos, bin_N) is kept and reused until the particles move
    const float *bin_pos;
    int64_t bin_N;
    int have_sched;              // the sink blocks of the last nf_accel / nf_accel4 are still in d_blk (nf_debug_delivered_pairs)
    int64_t launches;            // kernels launched by this context (nf_launch_count)
    cudaEvent_t ev[8];
    char err[512];
};

// -DNF_DEBUG_BOUNDS build (python -m paper_2110_11392_b200.build --debug-bounds <out.so>): every index the
// kernels derive from the offset tables, the ring cursor and the permutations is checked against the
// bound of the array it addresses; a violation records its code in ctrl[8] (largest code wins) and
// nf_sync reports it as NF_ECUDA.  tests/test_gpu_debug_bounds.py runs the small parity cases under it
// (compute-sanitizer is not available on this pool).  Compiled out of the product library.
#ifdef NF_DEBUG_BOUNDS
#define NF_CHECK(ctrl, cond, code) do { if (!(cond)) atomicMax(const_cast<uint32_t *>(ctrl) + 8, (uint32_t)(code)); } while (0)
#else
#define NF_CHECK(ctrl, cond, code) do { } while (0)
#endif

#define NF_CUDA_OK(ctx, call)                                                                   \
    do {                                                                                        \
        cudaError_t e__ = (call);                                                               \
        if (e__ != cudaSuccess) {                                                               \
            snprintf((ctx)->err, sizeof((ctx)->err), "%s failed: %s (%s:%d)", #call,            \
                     cudaGetErrorString(e__), __FILE__, __LINE__);                              \
            return (e__ == cudaErrorMemoryAllocation) ? NF_ENOMEM : NF_ECUDA;                   \
        }                                                                                       \
    } while (0)

// stages implemented in the other translation units
nf_status nf_run_binner(nf_ctx *ctx, const float *d_pos, int64_t N, cudaStream_t st);
nf_status nf_run_binner_host(nf_ctx *ctx, const float *h_pos, float *d_pos, int64_t N, cudaStream_t st);
nf_status nf_run_rebin(nf_ctx *ctx, const float *d_pos, int64_t N, cudaStream_t st);
nf_status nf_scan_cells(nf_ctx *ctx, cudaStream_t st);
nf_status nf_run_scheduler(nf_ctx *ctx, int64_t N, cudaStream_t st);
nf_status nf_run_interact(nf_ctx *ctx, const float *d_pos, int64_t N, float *d_out, int ostride, double kfac, cudaStream_t st);
nf_status nf_run_neighbors(nf_ctx *ctx, int cell, cudaStream_t st);
nf_status nf_run_multipoles(nf_ctx *ctx, const float *d_pos, int order, double *d_M, cudaStream_t st);
nf_status nf_run_kick_drift(nf_ctx *ctx, float *d_pos, float *d_vel, const float *d_acc, int64_t N, double dt_kick, double dt_drift,
                            cudaStream_t st);
nf_status nf_run_timestep_ratio(nf_ctx *ctx, const float *d_vel, const float *d_acc, double *d_out3, cudaStream_t st);
nf_status nf_run_taylor(nf_ctx *ctx, const float *d_pos, int order, const double *d_T, float *d_acc, int accumulate, cudaStream_t st);
nf_status nf_run_f64(nf_ctx *ctx, const float *d_pos, int64_t N, double *d_acc, cudaStream_t st);
nf_status nf_run_paircount(nf_ctx *ctx, cudaStream_t st);
nf_status nf_run_count(nf_ctx *ctx, cudaStream_t st);
nf_status nf_run_cell_histogram(nf_ctx *ctx, const float *d_pos, int64_t N, int32_t *d_counts, cudaStream_t st);
nf_status nf_run_slab_pairs(nf_ctx *ctx, const int32_t *d_counts, long long *d_pairs, long long *d_npart, cudaStream_t st);
nf_status nf_run_select_slabs(nf_ctx *ctx, const float *d_pos, int64_t N, int x0, int nx, float *d_out, uint32_t *d_blk, cudaStream_t st);
nf_status nf_interact_setup(nf_ctx *ctx);
nf_status nf_binner_setup(nf_ctx *ctx);
nf_status nf_scan_pairs(nf_ctx *ctx, cudaStream_t st);
nf_status nf_scan_u32(nf_ctx *ctx, const uint32_t *in, uint32_t n, uint32_t *out, cudaStream_t st);

// ---- device helpers shared by the kernels -------------------------------------------------
// periodic wrap of a cell index that is at most one period out of range; image = floor(v/cpd)
__device__ __forceinline__ int nf_wrap1(int v, int cpd, int &image) {
    image = 0;
    if (v < 0) { v += cpd; image = -1; }
    else if (v >= cpd) { v -= cpd; image = 1; }
    return v;
}
// non-negative modulus for any int
__device__ __forceinline__ int nf_mod(int v, int cpd) {
    int m = v % cpd;
    return m < 0 ? m + cpd : m;
}
// A1's cell rule for one axis (reading S5): I = floor((double)x * CPD / box), cell = I mod CPD for
// any finite x (half-open cells, periodic wrap); a NaN/Inf position sets `bad`
__device__ __forceinline__ int nf_axis_cell(float x, double scale, int cpd, int &bad) {
    double xd = (double)x;
    if (!isfinite(xd)) { bad = 1; return 0; }
    double t = xd * scale;
    double I = floor(t);
    if (I >= 0.0 && I < (double)cpd) return (int)I;
    double m = fmod(I, (double)cpd);      // exact
    if (m < 0.0) m += (double)cpd;
    return (int)m;
}

// The sorted planes (d_sorted, NF_PLANES planes of capPad slots): 0-2 x, y, z offsets from the cell
// centre in CELL units, rounded to float32 (the hot loop's operands); 3 the cell key (uint32 bits);
// 4-6 the float32 remainders lo = (float)(offset - (double)hi), so that (double)hi + (double)lo is
// the double-precision offset to 2^-48 -- read by the exact paths (close pairs, multipoles) in place
// of a second gather through the permutation.
#define NF_PLANES 7
__device__ __forceinline__ void nf_store_offsets(float *sorted, uint32_t cap_pad, uint32_t dst, const float *p, double scale) {
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const double t = (double)p[k] * scale;
        const double off = t - floor(t) - 0.5;                 // [-0.5, 0.5), reading S5
        const float hi = (float)off;
        sorted[(size_t)k * cap_pad + dst] = hi;
        sorted[(size_t)(4 + k) * cap_pad + dst] = (float)(off - (double)hi);
    }
}
__device__ __forceinline__ void nf_store_padding(float *sorted, uint32_t cap_pad, uint32_t dst) {
    sorted[dst] = NF_BIG; sorted[(size_t)cap_pad + dst] = 0.f; sorted[2ull * cap_pad + dst] = 0.f;
#pragma unroll
    for (int k = 4; k < 7; ++k) sorted[(size_t)k * cap_pad + dst] = 0.f;
}
