// nf_api.cu -- the C ABI of include/nearfield.h: argument checks, scratch management, stage
// sequencing.  No arithmetic of the method lives here.
#include <math.h>
#include <new>
#include <stdlib.h>
#include <string.h>
#include "nf_common.cuh"

static char g_static_err[256] = "";

static void free_scratch(nf_ctx *c) {
    void *ptrs[] = {c->d_key, c->d_arr, c->d_tmp_perm, c->d_chunk_sorted, c->d_perm_true, c->d_perm_pad, c->d_sorted, c->d_blk, c->d_blk_order, c->d_perm_alt, c->d_ins,
                    c->d_pair_slot};
    for (void *p : ptrs) if (p) cudaFree(p);
    c->d_key = c->d_arr = c->d_tmp_perm = c->d_chunk_sorted = c->d_perm_true = c->d_perm_pad = c->d_perm_alt = c->d_ins = nullptr;
    c->d_sorted = nullptr; c->d_blk = nullptr; c->d_blk_order = nullptr; c->d_pair_slot = nullptr;
    c->capN = c->capPad = c->capBlk = c->capRebin = 0;
    c->bin_valid = 0; c->bin_pinned = 0; c->have_sched = 0;
}

extern "C" nf_status nf_create(nf_ctx **out, int cpd, int R, double eps_plummer, double box) {
    if (!out) { snprintf(g_static_err, sizeof g_static_err, "nf_create: out is NULL"); return NF_EINVAL; }
    *out = nullptr;
    if (R < 1 || R > NF_MAX_R || cpd < 2 * R + 1 || !(eps_plummer > 0) || !isfinite(eps_plummer) || !(box > 0) || !isfinite(box) ||
        (double)cpd * cpd * cpd >= 2147483648.0) {
        snprintf(g_static_err, sizeof g_static_err, "nf_create: bad argument (cpd=%d R=%d eps=%g box=%g)", cpd, R, eps_plummer, box);
        return NF_EINVAL;
    }
    int dev = 0, ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1 || cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        snprintf(g_static_err, sizeof g_static_err, "nf_create: no CUDA device (there is no CPU fallback)");
        return NF_ECUDA;
    }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess || prop.major < 10) {
        snprintf(g_static_err, sizeof g_static_err, "nf_create: device is not sm_100 class (compute %d.%d)", prop.major, prop.minor);
        return NF_ECUDA;
    }
    nf_ctx *c = new (std::nothrow) nf_ctx;
    if (!c) return NF_ENOMEM;
    memset(c, 0, sizeof *c);
    c->device = dev; c->cpd = cpd; c->R = R; c->eps_p = eps_plummer; c->box = box; c->gm = 0.0;
    c->sm_count = prop.multiProcessorCount;
    c->ncell = (int64_t)cpd * cpd * cpd; c->ncol = (int64_t)cpd * cpd;
    c->slab_x0 = 0; c->slab_nx = cpd;
    c->opt_kahan = 1; c->opt_heavy_first = 0; c->opt_stage_timing = 0; c->opt_rc = -1.f;
    NfParams &p = c->prm;
    p.cpd = cpd; p.R = R; p.ncell = (int)c->ncell; p.ncol = (int)c->ncol;
    p.scale = (double)cpd / box;
    const double e = NF_SPLINE_PER_PLUMMER * eps_plummer * p.scale;   // eps_s in cell units
    p.eps_cells = e;
    p.c0 = (float)(10.0 / (e * e * e));
    p.c1 = (float)(-15.0 / (e * e * e * e));
    p.c2 = (float)(6.0 / (e * e * e * e * e));
    int nc = (int)ceil(e);
    if (nc < 1) nc = 1;
    if (nc > R) nc = R;
    p.near_cheb = nc;
    p.kahan = 1;
    nf_status rc = NF_OK;
    auto fail = [&](nf_status s) { snprintf(g_static_err, sizeof g_static_err, "%s", c->err); nf_destroy(c); return s; };
#define TRY_ALLOC(ptr, bytes)                                                                  \
    if (cudaMalloc((void **)&(ptr), (bytes)) != cudaSuccess) {                                  \
        cudaGetLastError(); snprintf(c->err, sizeof c->err, "nf_create: cudaMalloc(%zu) failed", (size_t)(bytes)); \
        return fail(NF_ENOMEM);                                                                 \
    }
    const size_t nscan = (size_t)((c->ncell + 2047) / 2048 + 8);
    c->capScan = (int64_t)nscan;
    TRY_ALLOC(c->d_counts, (size_t)(c->ncell + 1) * 4);
    TRY_ALLOC(c->d_offsets, (size_t)(c->ncell + 1) * 4);
    TRY_ALLOC(c->d_poff, (size_t)(c->ncell + 1) * 4);
    TRY_ALLOC(c->d_poff2, (size_t)(c->ncell + 1) * 4);
    TRY_ALLOC(c->d_mp_hist, 2064 * 4);      // occupancy classes of nf_multipoles (NFM_NCLASS + 1 <= 2064)
    TRY_ALLOC(c->d_scan_blk, nscan * 8);
    TRY_ALLOC(c->d_col_nblk, (size_t)(c->ncol + 1) * 4);
    TRY_ALLOC(c->d_col_base, (size_t)(c->ncol + 1) * 4);
    TRY_ALLOC(c->d_ctrl, 128 * 4);
    TRY_ALLOC(c->d_pairs, 64);      // [0..1] pair counter, sink counter; [2..4] time-step reduction (doubles)
    TRY_ALLOC(c->d_nbr, (size_t)4 * 729 * 4);
#undef TRY_ALLOC
    // flags and counters start at zero (nf_cell_histogram only ever SETS the bad-position flag ctrl[2], and may be the first call)
    if (cudaMemset(c->d_ctrl, 0, 128 * 4) != cudaSuccess) { snprintf(c->err, sizeof c->err, "nf_create: cudaMemset failed"); return fail(NF_ECUDA); }
    for (int i = 0; i < 8; ++i)
        if (cudaEventCreate(&c->ev[i]) != cudaSuccess) { snprintf(c->err, sizeof c->err, "cudaEventCreate failed"); return fail(NF_ECUDA); }
    if (cudaStreamCreateWithFlags(&c->own_stream, cudaStreamNonBlocking) != cudaSuccess ||
        cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) != cudaSuccess) { snprintf(c->err, sizeof c->err, "cudaStreamCreate failed"); return fail(NF_ECUDA); }
    if (cudaEventCreateWithFlags(&c->ev_order, cudaEventDisableTiming) != cudaSuccess) { snprintf(c->err, sizeof c->err, "cudaEventCreate failed"); return fail(NF_ECUDA); }
    for (int i = 0; i < NF_HOST_CHUNKS; ++i)
        if (cudaEventCreateWithFlags(&c->ev_chunk[i], cudaEventDisableTiming) != cudaSuccess) { snprintf(c->err, sizeof c->err, "cudaEventCreate failed"); return fail(NF_ECUDA); }
    rc = nf_interact_setup(c);
    if (rc == NF_OK) rc = nf_binner_setup(c);
    if (rc != NF_OK) return fail(rc);
    *out = c;
    return NF_OK;
}

extern "C" nf_status nf_destroy(nf_ctx *c) {
    if (!c) return NF_OK;
    cudaSetDevice(c->device);
    cudaDeviceSynchronize();
    free_scratch(c);
    void *ptrs[] = {c->d_counts, c->d_offsets, c->d_poff, c->d_poff2, c->d_mp_hist, c->d_scan_blk, c->d_col_nblk, c->d_col_base, c->d_ctrl, c->d_pairs, c->d_nbr, c->d_pos_buf, c->d_acc_buf,
                    c->d_offsets_alt, c->d_nstay};
    for (void *p : ptrs) if (p) cudaFree(p);
    for (int i = 0; i < 8; ++i) if (c->ev[i]) cudaEventDestroy(c->ev[i]);
    for (int i = 0; i < NF_HOST_CHUNKS; ++i) if (c->ev_chunk[i]) cudaEventDestroy(c->ev_chunk[i]);
    if (c->ev_order) cudaEventDestroy(c->ev_order);
    if (c->own_stream) cudaStreamDestroy(c->own_stream);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    cudaGetLastError();
    delete c;
    return NF_OK;
}

extern "C" int nf_bounds_checked(void) {
#ifdef NF_DEBUG_BOUNDS
    return 1;
#else
    return 0;
#endif
}

extern "C" const char *nf_last_error(const nf_ctx *c) { return c ? c->err : g_static_err; }

extern "C" nf_status nf_set_gm(nf_ctx *c, double gm) {
    if (!c || !isfinite(gm)) return NF_EINVAL;
    c->gm = gm;
    return NF_OK;
}

extern "C" nf_status nf_set_option(nf_ctx *c, const char *name, double v) {
    if (!c || !name) return NF_EINVAL;
    const int iv = (int)v;
    if (!strcmp(name, "rc_cells")) {
        // (for the spline law a positive value below eps_s is raised to eps_s on the device: k_choose_rc)
        if (!(v <= 0.25) || !isfinite(v)) { snprintf(c->err, sizeof c->err, "nf_set_option(rc_cells): need value <= 0.25 (negative = automatic)"); return NF_EINVAL; }
        c->opt_rc = (float)v;
        return NF_OK;
    }
    if (v != 0.0 && v != 1.0) { snprintf(c->err, sizeof c->err, "nf_set_option(%s): value must be 0 or 1", name); return NF_EINVAL; }
    if (!strcmp(name, "stage_timing")) c->opt_stage_timing = iv;
    else if (!strcmp(name, "kahan")) c->opt_kahan = iv;
    else if (!strcmp(name, "heavy_first")) c->opt_heavy_first = iv;
    else { snprintf(c->err, sizeof c->err, "nf_set_option: unknown option '%s'", name); return NF_EINVAL; }
    return NF_OK;
}

// One stream at a time per context: the scratch of a context is shared by its calls.  When a call
// arrives on another stream than the previous one, its work is ordered after that call's (an event on
// the previous stream, waited on by the new one) -- calls on different streams never overlap on one context.
static void enter_stream(nf_ctx *c, cudaStream_t st) {
    if (c->have_last && c->last_stream != st) {
        if (cudaEventRecord(c->ev_order, c->last_stream) == cudaSuccess) cudaStreamWaitEvent(st, c->ev_order, 0);
        else cudaGetLastError();
    }
    c->last_stream = st; c->have_last = 1;
}

static nf_status ensure_scratch(nf_ctx *c, int64_t N) {
    if (N <= c->capN) return NF_OK;
    cudaStreamSynchronize(c->last_stream);
    free_scratch(c);
    c->bin_pinned = 0; c->have_sched = 0;
    {   // block totals of the scans: over the cells, and over N/256 selection blocks (nf_select_slabs)
        const int64_t need = ((N + 255) / 256 + 2047) / 2048 + 8;
        if (need > c->capScan) {
            cudaFree(c->d_scan_blk); c->d_scan_blk = nullptr; c->capScan = 0;
            if (cudaMalloc((void **)&c->d_scan_blk, (size_t)need * 8) != cudaSuccess) {
                cudaGetLastError();
                snprintf(c->err, sizeof c->err, "scratch allocation for N=%lld failed", (long long)N);
                return NF_ENOMEM;
            }
            c->capScan = need;
        }
    }
    const int64_t capPad = ((N + (NF_CELL_PAD - 1) * c->ncell + 8 + 3) / 4) * 4 + 8;
    const int64_t capBlk = capPad / NF_BS + c->ncol + 8;
    cudaError_t e = cudaSuccess;
    auto A = [&](void **p, size_t bytes) { if (e == cudaSuccess) e = cudaMalloc(p, bytes); };
    A((void **)&c->d_key, (size_t)(N < 8 ? 8 : N) * 4);      // (also nf_select_slabs' block counts + scan: 2 (ceil(N/256) + 1) words, more than N when N <= 3)
    A((void **)&c->d_arr, (size_t)N * 4);
    A((void **)&c->d_tmp_perm, (size_t)capPad * 4);
    A((void **)&c->d_chunk_sorted, (size_t)capPad * 4);
    A((void **)&c->d_perm_true, (size_t)N * 4);
    A((void **)&c->d_perm_pad, (size_t)capPad * 4);
    A((void **)&c->d_sorted, (size_t)capPad * 4 * NF_PLANES);
    A((void **)&c->d_blk, (size_t)capBlk * sizeof(NfBlockDesc));
    A((void **)&c->d_blk_order, (size_t)capBlk * 4);
    A((void **)&c->d_pair_slot, (size_t)(capPad / 2 + 8) * 4);
    if (e != cudaSuccess) {
        cudaGetLastError();
        free_scratch(c);
        snprintf(c->err, sizeof c->err, "nf_accel: scratch allocation for N=%lld failed: %s", (long long)N, cudaGetErrorString(e));
        return NF_ENOMEM;
    }
    c->capN = N; c->capPad = capPad; c->capBlk = capBlk;
    return NF_OK;
}

// A1..A3 for (d_pos, N), or nothing when nf_bin pinned a binning of exactly this buffer
// ("most particles stay in their cell" -- and between the force, multipole, Taylor and
// time-step calls of one step none moves at all).
static nf_status bin_for(nf_ctx *c, const float *d_pos, int64_t N, cudaStream_t st) {
    nf_status rc = ensure_scratch(c, N);
    if (rc != NF_OK) return rc;
    enter_stream(c, st); c->lastN = N;
    if (c->bin_pinned && c->bin_pos == d_pos && c->bin_N == N) return NF_OK;
    c->bin_pinned = 0; c->have_sched = 0; c->bin_valid = 0;
    rc = nf_run_binner(c, d_pos, N, st);
    if (rc == NF_OK) { c->bin_valid = 1; c->bin_validN = N; }
    return rc;
}

extern "C" nf_status nf_bin(nf_ctx *c, const float *d_pos, int64_t N, void *cuda_stream) {
    if (!c) return NF_EINVAL;
    c->err[0] = 0;
    if (N <= 0 || !d_pos || (double)N + (double)(NF_CELL_PAD - 1) * (double)c->ncell >= 2147483640.0) {
        snprintf(c->err, sizeof c->err, "nf_bin: bad argument (N=%lld)", (long long)N);
        return NF_EINVAL;
    }
    NF_CUDA_OK(c, cudaSetDevice(c->device));
    c->bin_pinned = 0;
    nf_status rc = bin_for(c, d_pos, N, (cudaStream_t)cuda_stream);
    if (rc != NF_OK) return rc;
    c->bin_pinned = 1; c->bin_pos = d_pos; c->bin_N = N;
    return NF_OK;
}

extern "C" nf_status nf_rebin(nf_ctx *c, const float *d_pos, int64_t N, void *cuda_stream) {
    if (!c) return NF_EINVAL;
    c->err[0] = 0;
    if (N <= 0 || !d_pos || (double)N + (double)(NF_CELL_PAD - 1) * (double)c->ncell >= 2147483640.0) {
        snprintf(c->err, sizeof c->err, "nf_rebin: bad argument (N=%lld)", (long long)N);
        return NF_EINVAL;
    }
    if (!c->bin_valid || c->bin_validN != N || N > c->capN) return nf_bin(c, d_pos, N, cuda_stream);   // nothing to update: sort
    cudaStream_t st = (cudaStream_t)cuda_stream;
    NF_CUDA_OK(c, cudaSetDevice(c->device));
    if (c->capRebin < N || !c->d_offsets_alt) {
        cudaStreamSynchronize(c->last_stream);
        if (c->d_perm_alt) cudaFree(c->d_perm_alt);
        if (c->d_ins) cudaFree(c->d_ins);
        c->d_perm_alt = c->d_ins = nullptr; c->capRebin = 0;
        cudaError_t e = cudaMalloc((void **)&c->d_perm_alt, (size_t)c->capN * 4);
        if (e == cudaSuccess) e = cudaMalloc((void **)&c->d_ins, (size_t)c->capN * 4);
        if (e == cudaSuccess && !c->d_offsets_alt) e = cudaMalloc((void **)&c->d_offsets_alt, (size_t)(c->ncell + 1) * 4);
        if (e == cudaSuccess && !c->d_nstay) e = cudaMalloc((void **)&c->d_nstay, (size_t)(c->ncell + 1) * 8);
        if (e != cudaSuccess) {
            cudaGetLastError();
            snprintf(c->err, sizeof c->err, "nf_rebin: scratch allocation failed: %s", cudaGetErrorString(e));
            return NF_ENOMEM;
        }
        c->capRebin = c->capN;
    }
    enter_stream(c, st); c->lastN = N;
    c->bin_pinned = 0; c->have_sched = 0; c->bin_valid = 0;
    nf_status rc = nf_run_rebin(c, d_pos, N, st);
    if (rc != NF_OK) return rc;
    c->bin_valid = 1; c->bin_validN = N;
    c->bin_pinned = 1; c->bin_pos = d_pos; c->bin_N = N;
    return NF_OK;
}

extern "C" nf_status nf_unbin(nf_ctx *c) {
    if (!c) return NF_EINVAL;
    c->bin_pinned = 0;
    return NF_OK;
}

extern "C" nf_status nf_set_softening(nf_ctx *c, int law) {
    if (!c) return NF_EINVAL;
    if (law != NF_SOFT_SPLINE && law != NF_SOFT_PLUMMER && law != NF_SOFT_NEWTON) { snprintf(c->err, sizeof c->err, "nf_set_softening: unknown law %d", law); return NF_EINVAL; }
    c->law = law;
    return NF_OK;
}

extern "C" nf_status nf_set_sink_slabs(nf_ctx *c, int x0, int nx) {
    if (!c) return NF_EINVAL;
    if (x0 < 0 || x0 >= c->cpd || nx < 1 || nx > c->cpd) {
        snprintf(c->err, sizeof c->err, "nf_set_sink_slabs: need 0 <= x0 < cpd and 1 <= nx <= cpd (x0=%d nx=%d)", x0, nx);
        return NF_EINVAL;
    }
    c->slab_x0 = x0; c->slab_nx = nx;
    return NF_OK;
}

extern "C" nf_status nf_cell_histogram(nf_ctx *c, const float *d_pos, int64_t N, int32_t *d_counts, void *cuda_stream) {
    if (!c) return NF_EINVAL;
    c->err[0] = 0;
    if (N < 0 || !d_counts || (N > 0 && !d_pos) || N >= 2147483647ll) { snprintf(c->err, sizeof c->err, "nf_cell_histogram: bad argument (N=%lld)", (long long)N); return NF_EINVAL; }
    NF_CUDA_OK(c, cudaSetDevice(c->device));
    enter_stream(c, (cudaStream_t)cuda_stream);
    return nf_run_cell_histogram(c, d_pos, N, d_counts, (cudaStream_t)cuda_stream);
}

extern "C" nf_status nf_slab_pairs(nf_ctx *c, const int32_t *d_counts, int64_t *d_pairs, int64_t *d_npart, void *cuda_stream) {
    if (!c) return NF_EINVAL;
    c->err[0] = 0;
    if (!d_counts || !d_pairs || !d_npart) { snprintf(c->err, sizeof c->err, "nf_slab_pairs: NULL argument"); return NF_EINVAL; }
    NF_CUDA_OK(c, cudaSetDevice(c->device));
    return nf_run_slab_pairs(c, d_counts, (long long *)d_pairs, (long long *)d_npart, (cudaStream_t)cuda_stream);
}

extern "C" nf_status nf_select_slabs(nf_ctx *c, const float *d_pos, int64_t N, int x0, int nx, float *d_out, int64_t *h_count, void *cuda_stream) {
    if (!c) return NF_EINVAL;
    c->err[0] = 0;
    if (N < 0 || !h_count || (N > 0 && !d_pos) || x0 < 0 || x0 >= c->cpd || nx < 0 || nx > c->cpd ||
        (double)N + (double)(NF_CELL_PAD - 1) * (double)c->ncell >= 2147483640.0) {
        snprintf(c->err, sizeof c->err, "nf_select_slabs: bad argument (N=%lld x0=%d nx=%d)", (long long)N, x0, nx);
        return NF_EINVAL;
    }
    *h_count = 0;
    if (N == 0 || nx == 0) return NF_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    NF_CUDA_OK(c, cudaSetDevice(c->device));
    nf_status rc = ensure_scratch(c, N);
    if (rc != NF_OK) return rc;
    enter_stream(c, st); c->have_sched = 0;      // (the block scan reuses ctrl[1])
    rc = nf_run_select_slabs(c, d_pos, N, x0, nx, d_out, c->d_key, st);
    if (rc != NF_OK) return rc;
    uint32_t tot = 0;
    NF_CUDA_OK(c, cudaMemcpyAsync(&tot, c->d_ctrl + 1, sizeof tot, cudaMemcpyDeviceToHost, st));
    NF_CUDA_OK(c, cudaStreamSynchronize(st));
    *h_count = (int64_t)tot;
    return NF_OK;
}

extern "C" nf_status nf_set_density_radius(nf_ctx *c, double b) {
    if (!c) return NF_EINVAL;
    if (!(b >= 0) || !isfinite(b)) { snprintf(c->err, sizeof c->err, "nf_set_density_radius: need a finite b >= 0"); return NF_EINVAL; }
    c->dens_b = b;
    return NF_OK;
}

static nf_status accel_any(nf_ctx *c, const float *d_pos, int64_t N, float *d_acc, int ostride, void *cuda_stream) {
    if (!c) return NF_EINVAL;
    c->err[0] = 0;
    if (N < 0 || (N > 0 && (!d_pos || !d_acc)) || (double)N + (double)(NF_CELL_PAD - 1) * (double)c->ncell >= 2147483640.0) {
        snprintf(c->err, sizeof c->err, "nf_accel: bad argument (N=%lld)", (long long)N);
        return NF_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (N == 0) return NF_OK;
    NF_CUDA_OK(c, cudaSetDevice(c->device));
    if (c->opt_stage_timing) { for (int i = 0; i < 4; ++i) cudaEventRecord(c->ev[i], st); cudaEventRecord(c->ev[6], st); }
    nf_status rc = bin_for(c, d_pos, N, st);
    if (rc != NF_OK) return rc;
    if (c->opt_stage_timing && c->bin_pinned) cudaEventRecord(c->ev[3], st);      // binning reused: stages A1-A3 read 0
    rc = nf_run_scheduler(c, N, st);
    if (rc != NF_OK) return rc;
    if (c->opt_stage_timing) cudaEventRecord(c->ev[4], st);
    const double gm = c->gm > 0 ? c->gm : 1.0 / (double)N;
    const double cellsz = c->box / (double)c->cpd;
    const double kfac = gm / (cellsz * cellsz);
    rc = nf_run_interact(c, d_pos, N, d_acc, ostride, kfac, st);
    if (rc != NF_OK) return rc;
    c->have_sched = 1;
    if (c->opt_stage_timing) { cudaEventRecord(c->ev[5], st); cudaEventRecord(c->ev[7], st); }
    return NF_OK;
}

extern "C" nf_status nf_accel(nf_ctx *c, const float *d_pos, int64_t N, float *d_acc, void *cuda_stream) {
    return accel_any(c, d_pos, N, d_acc, 3, cuda_stream);
}

extern "C" nf_status nf_accel4(nf_ctx *c, const float *d_pos, int64_t N, float *d_acc4, void *cuda_stream) {
    return accel_any(c, d_pos, N, d_acc4, 4, cuda_stream);
}

extern "C" nf_status nf_accel_f64(nf_ctx *c, const float *d_pos, int64_t N, double *d_acc, void *cuda_stream) {
    if (!c) return NF_EINVAL;
    c->err[0] = 0;
    if (N < 0 || (N > 0 && (!d_pos || !d_acc)) || (double)N + (double)(NF_CELL_PAD - 1) * (double)c->ncell >= 2147483640.0) {
        snprintf(c->err, sizeof c->err, "nf_accel_f64: bad argument (N=%lld)", (long long)N);
        return NF_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (N == 0) return NF_OK;
    NF_CUDA_OK(c, cudaSetDevice(c->device));
    nf_status rc = bin_for(c, d_pos, N, st);
    if (rc != NF_OK) return rc;
    return nf_run_f64(c, d_pos, N, d_acc, st);
}

extern "C" nf_status nf_multipoles(nf_ctx *c, const float *d_pos, int64_t N, int order, double *d_M, void *cuda_stream) {
    if (!c) return NF_EINVAL;
    c->err[0] = 0;
    if (N < 0 || !d_M || (N > 0 && !d_pos) || order < 0 || order > NF_MAX_MULTIPOLE_ORDER ||
        (double)N + (double)(NF_CELL_PAD - 1) * (double)c->ncell >= 2147483640.0) {
        snprintf(c->err, sizeof c->err, "nf_multipoles: bad argument (N=%lld order=%d)", (long long)N, order);
        return NF_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    NF_CUDA_OK(c, cudaSetDevice(c->device));
    if (N == 0) {
        const size_t cml = (size_t)(order + 3) * (order + 2) * (order + 1) / 6;
        NF_CUDA_OK(c, cudaMemsetAsync(d_M, 0, (size_t)c->ncell * cml * sizeof(double), st));
        return NF_OK;
    }
    nf_status rc = bin_for(c, d_pos, N, st);
    if (rc != NF_OK) return rc;
    return nf_run_multipoles(c, d_pos, order, d_M, st);
}

extern "C" nf_status nf_kick_drift(nf_ctx *c, float *d_pos, float *d_vel, const float *d_acc, int64_t N, double dt_kick, double dt_drift,
                                   void *cuda_stream) {
    if (!c) return NF_EINVAL;
    c->err[0] = 0;
    if (N < 0 || (N > 0 && (!d_pos || !d_vel || !d_acc)) || !isfinite(dt_kick) || !isfinite(dt_drift)) {
        snprintf(c->err, sizeof c->err, "nf_kick_drift: bad argument (N=%lld)", (long long)N);
        return NF_EINVAL;
    }
    if (N == 0) return NF_OK;
    NF_CUDA_OK(c, cudaSetDevice(c->device));
    if (c->bin_pinned && c->bin_pos == d_pos && dt_drift != 0.0) c->bin_pinned = 0;    // the particles move: re-sort (or nf_bin) next time
    return nf_run_kick_drift(c, d_pos, d_vel, d_acc, N, dt_kick, dt_drift, (cudaStream_t)cuda_stream);
}

extern "C" nf_status nf_timestep_ratio(nf_ctx *c, const float *d_pos, const float *d_vel, const float *d_acc, int64_t N, double *h_out,
                                       void *cuda_stream) {
    if (!c) return NF_EINVAL;
    c->err[0] = 0;
    if (N < 0 || !h_out || (N > 0 && (!d_pos || !d_vel || !d_acc)) ||
        (double)N + (double)(NF_CELL_PAD - 1) * (double)c->ncell >= 2147483640.0) {
        snprintf(c->err, sizeof c->err, "nf_timestep_ratio: bad argument (N=%lld)", (long long)N);
        return NF_EINVAL;
    }
    h_out[0] = h_out[1] = INFINITY; h_out[2] = h_out[3] = 0.0;
    if (N == 0) return NF_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    NF_CUDA_OK(c, cudaSetDevice(c->device));
    nf_status rc = bin_for(c, d_pos, N, st);
    if (rc != NF_OK) return rc;
    double *d3 = (double *)(c->d_pairs + 2);
    rc = nf_run_timestep_ratio(c, d_vel, d_acc, d3, st);
    if (rc != NF_OK) return rc;
    double r[3];
    NF_CUDA_OK(c, cudaMemcpyAsync(r, d3, sizeof r, cudaMemcpyDeviceToHost, st));
    NF_CUDA_OK(c, cudaStreamSynchronize(st));
    h_out[0] = r[0];
    h_out[2] = sqrt(r[1] / (double)N);
    h_out[3] = sqrt(r[2]);
    h_out[1] = r[2] > 0.0 ? h_out[2] / h_out[3] : INFINITY;
    return NF_OK;
}

extern "C" nf_status nf_taylor_accel(nf_ctx *c, const float *d_pos, int64_t N, int order, const double *d_T, float *d_acc, int accumulate,
                                     void *cuda_stream) {
    if (!c) return NF_EINVAL;
    c->err[0] = 0;
    if (N < 0 || (N > 0 && (!d_pos || !d_T || !d_acc)) || order < 0 || order > NF_MAX_MULTIPOLE_ORDER ||
        (double)N + (double)(NF_CELL_PAD - 1) * (double)c->ncell >= 2147483640.0) {
        snprintf(c->err, sizeof c->err, "nf_taylor_accel: bad argument (N=%lld order=%d)", (long long)N, order);
        return NF_EINVAL;
    }
    if (N == 0) return NF_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    NF_CUDA_OK(c, cudaSetDevice(c->device));
    nf_status rc = bin_for(c, d_pos, N, st);
    if (rc != NF_OK) return rc;
    return nf_run_taylor(c, d_pos, order, d_T, d_acc, accumulate ? 1 : 0, st);
}

extern "C" nf_status nf_sync(nf_ctx *c) {
    if (!c) return NF_EINVAL;
    if (!c->have_last) return NF_OK;
    NF_CUDA_OK(c, cudaStreamSynchronize(c->last_stream));
    uint32_t ctrl[16];
    NF_CUDA_OK(c, cudaMemcpy(ctrl, c->d_ctrl, sizeof ctrl, cudaMemcpyDeviceToHost));
    if (ctrl[8]) { snprintf(c->err, sizeof c->err, "bounds check %u failed in a kernel (NF_DEBUG_BOUNDS build)", ctrl[8]); return NF_ECUDA; }
    if (ctrl[2]) { snprintf(c->err, sizeof c->err, "nf_accel: a position was NaN or infinite"); return NF_EPOS; }
    return NF_OK;
}

extern "C" nf_status nf_accel_host(nf_ctx *c, const float *h_pos, int64_t N, float *h_acc) {
    if (!c) return NF_EINVAL;
    if (N < 0 || (N > 0 && (!h_pos || !h_acc)) || (double)N + (double)(NF_CELL_PAD - 1) * (double)c->ncell >= 2147483640.0) {
        snprintf(c->err, sizeof c->err, "nf_accel_host: bad argument (N=%lld)", (long long)N);
        return NF_EINVAL;
    }
    if (N == 0) return NF_OK;
    NF_CUDA_OK(c, cudaSetDevice(c->device));
    if (N > c->capHost) {
        if (c->d_pos_buf) cudaFree(c->d_pos_buf);
        if (c->d_acc_buf) cudaFree(c->d_acc_buf);
        c->d_pos_buf = c->d_acc_buf = nullptr; c->capHost = 0;
        NF_CUDA_OK(c, cudaMalloc((void **)&c->d_pos_buf, (size_t)N * 12));
        NF_CUDA_OK(c, cudaMalloc((void **)&c->d_acc_buf, (size_t)N * 12));
        c->capHost = N;
    }
    // H2D in ranges with A1 behind each (nf_run_binner_host), then the rest of the path on that binning
    cudaStream_t st = c->own_stream;
    c->err[0] = 0;
    nf_status rc = ensure_scratch(c, N);
    if (rc != NF_OK) return rc;
    enter_stream(c, st); c->lastN = N;
    c->bin_pinned = 0; c->have_sched = 0; c->bin_valid = 0;
    rc = nf_run_binner_host(c, h_pos, c->d_pos_buf, N, st);
    if (rc != NF_OK) return rc;
    c->bin_valid = 1; c->bin_validN = N;
    c->bin_pinned = 1; c->bin_pos = c->d_pos_buf; c->bin_N = N;
    rc = nf_accel(c, c->d_pos_buf, N, c->d_acc_buf, (void *)st);
    c->bin_pinned = 0;                       // the staging buffer is overwritten by the next call
    if (rc != NF_OK) return rc;
    NF_CUDA_OK(c, cudaMemcpyAsync(h_acc, c->d_acc_buf, (size_t)N * 12, cudaMemcpyDeviceToHost, st));
    return nf_sync(c);
}

extern "C" nf_status nf_stage_ms(nf_ctx *c, float *h_ms) {
    if (!c || !h_ms) return NF_EINVAL;
    for (int i = 0; i < NF_N_STAGES; ++i) h_ms[i] = 0.f;
    if (!c->have_last || !c->opt_stage_timing) { snprintf(c->err, sizeof c->err, "nf_stage_ms: enable option stage_timing and call nf_accel first"); return NF_EINVAL; }
    NF_CUDA_OK(c, cudaStreamSynchronize(c->last_stream));
    NF_CUDA_OK(c, cudaEventElapsedTime(&h_ms[0], c->ev[0], c->ev[1]));
    NF_CUDA_OK(c, cudaEventElapsedTime(&h_ms[1], c->ev[1], c->ev[2]));
    NF_CUDA_OK(c, cudaEventElapsedTime(&h_ms[2], c->ev[2], c->ev[3]));
    NF_CUDA_OK(c, cudaEventElapsedTime(&h_ms[3], c->ev[3], c->ev[4]));
    NF_CUDA_OK(c, cudaEventElapsedTime(&h_ms[4], c->ev[4], c->ev[5]));
    NF_CUDA_OK(c, cudaEventElapsedTime(&h_ms[5], c->ev[6], c->ev[7]));
    return NF_OK;
}

extern "C" nf_status nf_debug_cells(nf_ctx *c, const uint32_t **d_offsets, const uint32_t **d_perm, const float **d_sorted,
                                    const uint32_t **d_poffsets, int64_t *h_npad) {
    if (!c) return NF_EINVAL;
    if (!c->have_last) { snprintf(c->err, sizeof c->err, "nf_debug_cells: no nf_accel call yet"); return NF_EINVAL; }
    if (d_offsets) *d_offsets = c->d_offsets;
    if (d_perm) *d_perm = c->d_perm_true;
    if (d_sorted) *d_sorted = c->d_sorted;
    if (d_poffsets) *d_poffsets = c->d_poff;
    if (h_npad) *h_npad = c->capPad;   // plane stride of d_sorted
    return NF_OK;
}

extern "C" nf_status nf_close_radius(nf_ctx *c, double *h_rc_cells) {
    if (!c || !h_rc_cells) return NF_EINVAL;
    if (!c->have_last) { snprintf(c->err, sizeof c->err, "nf_close_radius: no nf_accel call yet"); return NF_EINVAL; }
    NF_CUDA_OK(c, cudaStreamSynchronize(c->last_stream));
    float dyn[2];
    NF_CUDA_OK(c, cudaMemcpy(dyn, c->d_ctrl + 96, sizeof dyn, cudaMemcpyDeviceToHost));
    *h_rc_cells = dyn[1];
    return NF_OK;
}

extern "C" nf_status nf_launch_count(nf_ctx *c, int64_t *h_count) {
    if (!c || !h_count) return NF_EINVAL;
    *h_count = c->launches;
    return NF_OK;
}

extern "C" nf_status nf_debug_read(nf_ctx *c, const void *d_src, void *h_dst, uint64_t bytes) {
    if (!c || !d_src || !h_dst) return NF_EINVAL;
    NF_CUDA_OK(c, cudaSetDevice(c->device));
    if (c->have_last) NF_CUDA_OK(c, cudaStreamSynchronize(c->last_stream));
    NF_CUDA_OK(c, cudaMemcpy(h_dst, d_src, (size_t)bytes, cudaMemcpyDeviceToHost));
    return NF_OK;
}

extern "C" nf_status nf_debug_neighbors(nf_ctx *c, int cell, int32_t *h_ids, int8_t *h_image) {
    if (!c || !h_ids || !h_image || cell < 0 || cell >= c->ncell) return NF_EINVAL;
    NF_CUDA_OK(c, cudaSetDevice(c->device));
    const int w = 2 * c->R + 1, nn = w * w * w;
    nf_status rc = nf_run_neighbors(c, cell, c->own_stream);
    if (rc != NF_OK) return rc;
    int32_t *tmp = (int32_t *)malloc((size_t)nn * 4 * sizeof(int32_t));
    if (!tmp) return NF_ENOMEM;
    cudaError_t e = cudaMemcpyAsync(tmp, c->d_nbr, (size_t)nn * 4 * sizeof(int32_t), cudaMemcpyDeviceToHost, c->own_stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->own_stream);
    if (e != cudaSuccess) { free(tmp); snprintf(c->err, sizeof c->err, "nf_debug_neighbors: %s", cudaGetErrorString(e)); return NF_ECUDA; }
    for (int n = 0; n < nn; ++n) {
        h_ids[n] = tmp[n];
        for (int k = 0; k < 3; ++k) h_image[3 * n + k] = (int8_t)tmp[nn + 3 * n + k];
    }
    free(tmp);
    return NF_OK;
}

extern "C" nf_status nf_debug_delivered_pairs(nf_ctx *c, int64_t *h_out) {
    if (!c || !h_out) return NF_EINVAL;
    if (!c->have_last || !c->have_sched) { snprintf(c->err, sizeof c->err, "nf_debug_delivered_pairs: the last call on this context was not nf_accel / nf_accel4"); return NF_EINVAL; }
    NF_CUDA_OK(c, cudaSetDevice(c->device));
    NF_CUDA_OK(c, cudaStreamSynchronize(c->last_stream));
    nf_status rc = nf_run_count(c, c->own_stream);
    if (rc != NF_OK) return rc;
    unsigned long long v[2] = {0, 0};
    NF_CUDA_OK(c, cudaMemcpyAsync(v, c->d_pairs + 6, 16, cudaMemcpyDeviceToHost, c->own_stream));
    NF_CUDA_OK(c, cudaStreamSynchronize(c->own_stream));
    h_out[0] = (int64_t)v[0]; h_out[1] = (int64_t)v[1];
    return NF_OK;
}

extern "C" nf_status nf_interaction_count(nf_ctx *c, int64_t *h_pairs) {
    if (!c || !h_pairs) return NF_EINVAL;
    if (!c->have_last) { snprintf(c->err, sizeof c->err, "nf_interaction_count: no nf_accel call yet"); return NF_EINVAL; }
    NF_CUDA_OK(c, cudaSetDevice(c->device));
    NF_CUDA_OK(c, cudaStreamSynchronize(c->last_stream));
    nf_status rc = nf_run_paircount(c, c->own_stream);
    if (rc != NF_OK) return rc;
    unsigned long long v[2] = {0, 0};
    NF_CUDA_OK(c, cudaMemcpyAsync(v, c->d_pairs, 16, cudaMemcpyDeviceToHost, c->own_stream));
    NF_CUDA_OK(c, cudaStreamSynchronize(c->own_stream));
    *h_pairs = (int64_t)v[0] - (int64_t)v[1];
    return NF_OK;
}
