/*
 * nearfield.h -- C ABI of libnearfield_b200.so: the Abacus near-field force on one B200.
 *
 * What the library computes (reference: /root/reference/PAPER.md, arXiv 2110.11392):
 *   "every cell interacting with itself and its 124 nearest neighbor cells (for near-field
 *   radius R=2) using open boundary conditions and Newtonian gravity, or a softened form
 *   thereof" (sec. 3.4.1) on a periodic grid of CPD^3 cells, with
 *   the spline softening law of Eq. 3 and eps_s = 2.16 eps_p:
 *
 *       a_i = gm * sum_{j in the (2R+1)^3 cells around cell(i), j != i} F(x_j - x_i + image)
 *       F(r) = [10 - 15u + 6u^2] r / eps_s^3   (u = |r|/eps_s < 1),   r/|r|^3 otherwise.
 *
 *   The periodic image is the whole-cell shift of the CELL PAIR, not the
 *   particle minimum image.  Steps run by nf_accel, all in CUDA kernels for sm_100a
 *   (DESIGN.md "The path"): A1 cell key + histogram, A2 exclusive scan, A3 stable scatter into
 *   grid order with cell-relative float32 offsets, A4 pencil scheduler
 *   (PAPER.md:226-236), A5 pencil-on-pencil interaction kernel, A6 un-permute to input order.
 *
 * Conventions
 *   - Plain pointers and sizes only.  "d_" = device pointer on the context's device,
 *     "h_" = host pointer.  float = IEEE binary32.  Positions/accelerations are N x 3, xyz
 *     interleaved, contiguous (three floats per particle).
 *   - The caller owns every buffer it passes in.  The library never frees, reallocates or
 *     writes d_pos / h_pos.  The context owns all scratch (grow-only).
 *   - All device work of nf_accel is enqueued on `cuda_stream` (a cudaStream_t passed as
 *     void*; NULL = the legacy default stream); the call returns without synchronising.
 *     One stream at a time per context: the context's scratch is shared by its calls, so a
 *     call on another stream than the previous call's is ordered after it (an event on the
 *     previous stream, waited on by the new one) -- two calls on one context never overlap;
 *     use one context per stream for concurrency.  A stream handed to a call must stay
 *     valid until the next call on the context or nf_sync.  Calls are not thread-safe per
 *     context (one host thread at a time).
 *   - Every function returns an nf_status and never throws or aborts; nf_last_error gives
 *     the text of the last failure on that context.
 *   - There is no CPU fallback: without a CUDA device nf_create fails with NF_ECUDA.
 */
#ifndef NEARFIELD_B200_H
#define NEARFIELD_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nf_ctx nf_ctx; /* opaque; created by nf_create, freed by nf_destroy */

typedef enum {
    NF_OK = 0,
    NF_EINVAL = 1, /* bad argument (see each function) */
    NF_ECUDA = 2,  /* a CUDA runtime call failed (text in nf_last_error) */
    NF_ENOMEM = 3, /* device or host allocation failed */
    NF_EPOS = 4    /* a position was NaN or infinite (reported by nf_sync) */
} nf_status;

#define NF_MAX_R 4          /* compiled maximum near-field radius */
#define NF_MAX_MULTIPOLE_ORDER 16   /* compiled maximum order p of nf_multipoles */
#define NF_SOFT_SPLINE 0    /* Eq. 3, the paper's "single_spline" (Fig. 19) */
#define NF_SOFT_PLUMMER 1   /* Eq. 2 */
#define NF_SOFT_NEWTON 2    /* no softening: F = r/|r|^3 ("Newtonian gravity, or a softened form thereof") */
#define NF_N_STAGES 8       /* entries of nf_stage_ms */

/*
 * nf_create -- make a context for a grid of cpd^3 cells of a periodic box of side `box`,
 * near-field radius R cells and Plummer-equivalent softening length
 * eps_plummer (same length unit as box and positions; converted internally to the spline
 * length eps_s = 2.16 eps_plummer).  Uses the current CUDA device.
 * NF_EINVAL: out == NULL, R < 1, R > NF_MAX_R, cpd < 2R+1, cpd^3 >= 2^31, eps_plummer <= 0
 * or not finite, box <= 0 or not finite.  NF_ECUDA: no usable device.
 */
nf_status nf_create(nf_ctx **out, int cpd, int R, double eps_plummer, double box);

/* nf_destroy -- synchronise the context's last stream, free all scratch.  NULL is NF_OK. */
nf_status nf_destroy(nf_ctx *ctx);

/*
 * nf_set_gm -- G*m of the (equal-mass) particles, the factor in a_i = gm * sum F
 * (kernel has no mass; equal masses 1/N with G=1 in BASELINE.json).
 * gm <= 0 (the default) means "1/N of each call".  NF_EINVAL: ctx NULL or gm not finite.
 */
nf_status nf_set_gm(nf_ctx *ctx, double gm);

/*
 * nf_accel -- near-field accelerations of N particles.
 *   d_pos  [in]  device, N*3 floats, positions; any finite value is wrapped periodically
 *                into [0, box) by the cell index (half-open cells, floor).
 *   d_acc  [out] device, N*3 floats, a_i in (length unit)/time^2 for gm in those units,
 *                in INPUT order.  Must not overlap d_pos.
 *   cuda_stream  cudaStream_t as void*.
 * Enqueues A1..A6 on the stream and returns.  N == 0 is NF_OK and does nothing.
 * NF_EINVAL: ctx/d_pos/d_acc NULL (with N > 0), N < 0, N + cpd^3 >= 2^31 - 8.
 * NF_ENOMEM / NF_ECUDA: scratch allocation or a launch failed.
 * A NaN/Inf position does not fail this call: the particle is binned into cell 0, the
 * result is unspecified, and the next nf_sync returns NF_EPOS.
 */
nf_status nf_accel(nf_ctx *ctx, const float *d_pos, int64_t N, float *d_acc, void *cuda_stream);

/*
 * nf_bin -- run the binning (A1..A3) of d_pos now and KEEP it: until the particles move, every
 * call on ctx that is given the same d_pos pointer and N (nf_accel, nf_accel4, nf_accel_f64,
 * nf_multipoles, nf_taylor_accel, nf_timestep_ratio) reuses this grid order instead of sorting
 * again -- within one time step the force, multipole, Taylor and time-step calls see the same
 * positions (Table 1).  The caller promises not to change d_pos meanwhile -- the pin
 * is keyed on the POINTER and the count only, so an in-place change made by anything but this context's
 * nf_kick_drift, or a new buffer of the same size that an allocator places at the freed address of the
 * pinned one, is silently served the OLD grid order: keep the pinned buffer alive and call nf_unbin (or
 * nf_bin again) whenever its contents change by other means.  The
 * pin ends at the next nf_bin / nf_rebin / nf_unbin, at an nf_kick_drift of that buffer with
 * dt_drift != 0, or when a call passes another buffer or count (which is then sorted as usual).
 * NF_EINVAL: ctx/d_pos NULL, N <= 0 or too large.
 */
nf_status nf_bin(nf_ctx *ctx, const float *d_pos, int64_t N, void *cuda_stream);

/*
 * nf_rebin -- drift-aware update of the grid order (the paper's insert list + merge, PAPER.md:356-395:
 * "most particles stay in their cell"): d_pos holds the positions of the SAME N particles (same input
 * order) the context last binned, moved a little (e.g. by nf_kick_drift).  Particles whose cell is
 * unchanged keep their place among their cell's stayers (no sorting: the old order is ascending in
 * input index); the others go through an insert list and are merged into their new cells by input
 * index.  The result equals a full sort (nf_bin) of the new positions bit for bit -- offsets,
 * permutation, planes -- and is pinned like nf_bin's.  How far the particles moved affects only the
 * cost.  If the context holds no binning of N particles this is nf_bin.  Errors as nf_bin.
 *
 * WHICH ONE TO CALL: nf_bin.  On a device-resident particle set the full counting sort is the faster of the
 * two: measured on the 157 M-particle configuration after a drift of 0.05 cell rms per axis (11 % of the
 * particles change cell), nf_bin 5.5 ms against nf_rebin 18.0 ms (15 GB of DRAM traffic against 40 GB;
 * DESIGN.md section 9).  The paper's insert list pays where the state streams through host memory slab by slab
 * and stayers are never touched; here every stayer is re-gathered through the old
 * permutation, and in a clustered cell the merge costs (cell occupancy) x (arrivals).  nf_rebin is kept as the
 * restatement of the paper's scheme and as a second, independently coded route to the same grid order that the
 * tests compare bit for bit with nf_bin; it is not on any timed path.
 */
nf_status nf_rebin(nf_ctx *ctx, const float *d_pos, int64_t N, void *cuda_stream);

/* nf_unbin -- drop the pin of nf_bin / nf_rebin (the next call sorts again). */
nf_status nf_unbin(nf_ctx *ctx);

/*
 * nf_set_softening -- the "near-force softening technique" the paper chooses at build time
 * (PAPER.md:620): NF_SOFT_SPLINE (default; Eq. 3 with eps_s = 2.16 eps_plummer) or
 * NF_SOFT_PLUMMER (Eq. 2, F = r/(r^2 + eps_plummer^2)^(3/2)) or NF_SOFT_NEWTON (no
 * softening, F = r/|r|^3; eps_plummer is ignored, a coincident pair contributes 0 as
 * F(0) = 0 does for the softened laws; pairs closer than the close-pair radius are evaluated in
 * double precision, see option "rc_cells").  Takes effect at the next nf_accel / nf_accel4 /
 * nf_accel_f64.  NF_EINVAL: ctx NULL or an unknown law.
 */
nf_status nf_set_softening(nf_ctx *ctx, int law);

/*
 * nf_set_density_radius -- radius b (length units of box) of the FoF-scale density estimate
 * of sec. 3.4.4 ("Compute FOF-scale density"), used by nf_accel4.
 * b = 0 (default) switches it off.  NF_EINVAL: ctx NULL, b < 0 or not finite.
 */
nf_status nf_set_density_radius(nf_ctx *ctx, double b);

/*
 * nf_set_sink_slabs -- slab decomposition (PAPER.md:80 "1-D slab decomposition", :413): only
 * particles whose x cell index lies in the periodic range [x0, x0 + nx) are SINKS of the
 * following nf_accel / nf_accel4 calls; every particle passed in is still a source.  A rank
 * that owns those slabs passes its own particles plus the ghost particles of the R slabs on
 * either side (near-field radius, Table 1) and reads back its own particles'
 * rows; rows of non-sink particles are left untouched.  nf_interaction_count then counts the
 * pairs of the sink cells only, so the counts of a complete decomposition add up to the
 * single-GPU count.  Default: x0 = 0, nx = cpd (everything).  NF_EINVAL: ctx NULL, x0 outside
 * [0, cpd), nx outside [1, cpd].
 */
nf_status nf_set_sink_slabs(nf_ctx *ctx, int x0, int nx);

/*
 * Device-side support of the slab decomposition (paper_2110_11392_b200/slabs.py is the host plumbing
 * around these; ghost slabs = near-field radius, Table 1):
 *
 * nf_cell_histogram -- occupancy histogram of N particles under step A1's cell rule (half-open cells,
 *   periodic wrap of any finite position): d_counts [out] device, cpd^3 int32, key = (cx*cpd+cy)*cpd+cz,
 *   caller-owned (so that ranks can sum their histograms with one all-reduce).  Zero-fills first;
 *   N == 0 gives zeros.  A NaN/Inf position is not counted and makes the next nf_sync return NF_EPOS.
 * nf_slab_pairs -- from a (global) histogram, per x slab i: d_npart[i] = particles in the slab and
 *   d_pairs[i] = sum over its cells c of n_c * sum_{c' in N(c)} n_c' (self pairs included: subtract
 *   d_npart for the q != p count), the integer identity P7 -- the work the slabs are balanced by.
 *   d_pairs, d_npart [out] device, cpd int64 each.
 * nf_select_slabs -- copy the particles whose x cell index lies in the periodic range [x0, x0 + nx)
 *   to d_out (device, room for N*3 floats; NULL = count only) in input order, and return their number
 *   in *h_count (synchronises the stream).  nx = 0 selects nothing.
 * NF_EINVAL: NULL arguments, N < 0 or too large, x0 outside [0, cpd), nx outside [0, cpd].
 */
nf_status nf_cell_histogram(nf_ctx *ctx, const float *d_pos, int64_t N, int32_t *d_counts, void *cuda_stream);
nf_status nf_slab_pairs(nf_ctx *ctx, const int32_t *d_counts, int64_t *d_pairs, int64_t *d_npart, void *cuda_stream);
nf_status nf_select_slabs(nf_ctx *ctx, const float *d_pos, int64_t N, int x0, int nx, float *d_out, int64_t *h_count,
                          void *cuda_stream);

/*
 * nf_cell_offsets_noalloc -- step A2 without a context and without any allocation: the exclusive scan
 * of a cell histogram into the per-cell offsets of the grid order (each cell is an
 * offset and a count into the grid-ordered arrays),
 *     d_offsets[c] = sum of d_counts[c'] over c' < c,   d_offsets[ncell] = the total.
 *
 * For callers that cannot let a library call cudaMalloc.  Everything else in this header works on an
 * nf_ctx whose scratch comes from cudaMalloc, at nf_create and again when a larger N arrives.  That
 * does not suit (a) a code that gave the whole device to its own memory pool at start-up, as a
 * simulation sized to fill the GPU does -- a later cudaMalloc can just fail; or (b) a time-step loop
 * that keeps copies and kernels in flight on several streams -- cudaMalloc and cudaFree wait for the
 * whole device and break that overlap.  This call touches only the caller's two buffers and a fixed
 * array of tile partial sums that is part of the library's device image.  It calls no cudaMalloc,
 * cudaFree or allocating library routine, and needs no context.
 *
 *   d_counts   [in]  device, ncell int32, non-negative, total below 2^32 (e.g. nf_cell_histogram's
 *                    output, key = (cx*cpd+cy)*cpd+cz).  May be NULL when ncell == 0.
 *   d_offsets  [out] device, ncell + 1 uint32.  Must not overlap d_counts.  Caller-owned, like d_counts.
 *   cuda_stream      cudaStream_t as void*; both launches are enqueued there, no synchronisation.
 *
 * Limits and rules
 *   - ncell <= NF_NOALLOC_MAX_CELLS (8 388 608 = 4096 tiles of 2048 cells, i.e. cpd <= 203; the
 *     157 M-particle configuration has 135^3 = 2 460 375).  A larger ncell is refused with NF_EINVAL
 *     and a message that names the limit; nothing is launched.  Use a context (nf_bin) there.
 *   - Cost of the fixed array: 16 KB of device memory on every GPU that loads this library, from the
 *     load until the process exits, whether or not this call is ever made.
 *   - The device that holds the buffers (and owns the stream) must be the CURRENT device.  The first
 *     call on each device looks up the array's device address (cudaGetSymbolAddress) and remembers
 *     it; make that first call before any stream capture begins on that device.
 *   - All calls on a device share the one array.  It keeps whatever the previous call left; nothing in
 *     it has to start at zero, because each call writes every word it later reads.  Two calls whose
 *     kernels can overlap on the GPU (different streams with no ordering between them) race on the
 *     array and give wrong offsets: order them (same stream, or an event).  Host threads may call
 *     concurrently (the set-up is locked); the ordering of the GPU work is still the caller's job.
 *   - Result equals the context path's offsets (nf_debug_cells after nf_bin) bit for bit.
 * Errors: NF_EINVAL -- ncell < 0 or beyond the limit, d_offsets NULL, d_counts NULL with ncell > 0;
 * NF_ECUDA -- no current device, the address look-up or a launch failed.  The text is returned by
 * nf_cell_offsets_noalloc_error (static storage, valid until the next failing call).
 */
#define NF_NOALLOC_MAX_CELLS 8388608
nf_status nf_cell_offsets_noalloc(const int32_t *d_counts, int64_t ncell, uint32_t *d_offsets, void *cuda_stream);
const char *nf_cell_offsets_noalloc_error(void);

/*
 * nf_accel4 -- nf_accel with the accelerations "promoted to 4-vectors":
 *   d_acc4 [out] device, N*4 floats (ax, ay, az, w) in INPUT order, where
 *       w_i = sum over the sources j != i of the same (2R+1)^3 cells with r_ij < b of (b^2 - r_ij^2),
 *   the paper's apodised top-hat estimate "computed as b^2 - r^2 on the GPU", unnormalised, in
 *   (length unit)^2; the particle itself is not counted, a distinct particle at r = 0 counts b^2.
 *   With b = 0 the 4th component is not written.
 * Same kernels as nf_accel (the density rides in the near-cell form of the pair loop); same
 * arguments, ordering and errors.
 */
nf_status nf_accel4(nf_ctx *ctx, const float *d_pos, int64_t N, float *d_acc4, void *cuda_stream);

/*
 * nf_accel_f64 -- the paper's "Double precision: yes" build (Fig. 19) as a second
 * entry point, for validating the float32 kernel on the GPU: the same
 * binning, then a plain direct sum in double precision (offsets recomputed in double from the
 * float32 positions, piecewise law with a branch, no packed arithmetic, no close-pair path).
 *   d_acc [out] device, N*3 DOUBLES, input order.  Honours nf_set_gm, nf_set_softening and
 *   nf_set_sink_slabs.  Some 30 times slower than nf_accel; not part of the timed path.
 * Errors as nf_accel.
 */
nf_status nf_accel_f64(nf_ctx *ctx, const float *d_pos, int64_t N, double *d_acc, void *cuda_stream);

/*
 * nf_multipoles -- the cell multipoles of Eq. 4 (sec. 3.3.2), the particle-facing
 * step of the far field that follows NearForce in the paper's pipeline, in the complete basis:
 *     M_cell^{a,b,c} = sum over the particles q of the cell of x_q^a y_q^b z_q^c,
 *     0 <= a <= order, 0 <= b <= order - a, 0 <= c <= order - a - b,
 * (x_q, y_q, z_q) = offset of q from its cell centre in length units, in double precision.
 *   d_M [out] device, cpd^3 * cml DOUBLES, cell-major (key = (cx*cpd+cy)*cpd+cz), cml =
 *       (order+3)(order+2)(order+1)/6, element order = the nesting a (outer), b, c (inner) of the
 *       paper's pseudo-code.  Empty cells get zeros.  order = 8 is the paper's choice.
 * Runs the binning (A1-A3) of d_pos and one kernel; N == 0 zero-fills.  The conversion to the
 * reduced basis, the FFTs and the convolution are not part of this library.
 * NF_EINVAL: ctx/d_M NULL, d_pos NULL with N > 0, N < 0, order outside [0, NF_MAX_MULTIPOLE_ORDER].
 */
nf_status nf_multipoles(nf_ctx *ctx, const float *d_pos, int64_t N, int order, double *d_M, void *cuda_stream);

/*
 * nf_taylor_accel -- far-field acceleration of every particle from its cell's Taylor series of
 * the potential (TaylorForce, Table 1).  The paper does not print
 * the series; this library's reading: d_T holds, per cell, the coefficients T^{a,b,c} of
 *     phi(x,y,z) = sum_{a+b+c <= order} T^{a,b,c} x^a y^b z^c,  (x,y,z) = offset from the cell centre,
 * in the complete basis and element order of nf_multipoles (factorials folded into T), and
 *     a = -grad phi.
 *   d_T   [in]  device, cpd^3 * cml doubles, cell-major;  d_acc [out] device, N*3 floats, input
 *   order: written, or added to when accumulate != 0 (e.g. onto nf_accel's near field).
 * Evaluated in double, rounded to float32 once.  Runs the binning (A1-A3) and one kernel.  Producing
 * T (reduced basis, FFTs, derivatives-tensor convolution) is not part of this library.
 * NF_EINVAL: ctx NULL, N < 0, a NULL buffer with N > 0, order outside [0, NF_MAX_MULTIPOLE_ORDER].
 */
nf_status nf_taylor_accel(nf_ctx *ctx, const float *d_pos, int64_t N, int order, const double *d_T, float *d_acc, int accumulate,
                          void *cuda_stream);

/*
 * nf_kick_drift -- Kick then Drift of the KDK leapfrog (sec. 3.1; Table 1
 * PAPER.md:379-380), in place on float32 state:
 *     v <- v + a * dt_kick ;   x <- x + v_new * dt_drift, wrapped periodically into [0, box).
 *   d_pos, d_vel [in/out] device, N*3 floats; d_acc [in] device, N*3 floats (e.g. nf_accel's output
 *   plus the caller's far field).  Each update is evaluated in double (product and sum rounded
 *   separately) and rounded to float32 once; a wrapped value that rounds to box becomes 0.
 *   dt_kick / dt_drift are plain intervals (the cosmological kick/drift factors are the caller's);
 *   a half kick is dt_drift = 0, a pure drift dt_kick = 0.
 * Ordering: the kernel is enqueued on `cuda_stream` as given.  Unlike the calls that use the context's
 *   scratch, this one is NOT ordered after the context's previous call when that ran on another stream: if
 *   d_acc is being written by an nf_accel on stream A, or d_pos is the buffer nf_bin pinned and a force call on
 *   stream A is still reading it, pass stream A here too (or order the streams with an event yourself).
 * NF_EINVAL: ctx NULL, N < 0, a NULL buffer with N > 0, a non-finite interval.
 */
nf_status nf_kick_drift(nf_ctx *ctx, float *d_pos, float *d_vel, const float *d_acc, int64_t N, double dt_kick, double dt_drift,
                        void *cuda_stream);

/*
 * nf_timestep_ratio -- the particle-dependent part of the global time-step criterion, Eq. 1
 * (PAPER.md:98-102):  max( min over cells of [v_rms / a_max]_c , v_rms,global / a_max,global ), with
 * v_rms = sqrt(mean |v|^2) (mean velocity not subtracted) and a_max = max |a| over the particles of a
 * cell of the cpd^3 grid, or of the box.  Empty cells and cells with a_max = 0 do not constrain.
 *   h_out [out] host, 4 doubles: [0] min_c v_rms/a_max (+inf if none), [1] v_rms,global / a_max,global,
 *   [2] v_rms,global, [3] a_max,global.  The caller forms
 *   da = min(eta_H a, eta_acc a H max(h_out[0], h_out[1])).
 * Runs the binning (A1-A3) of d_pos and one reduction kernel; synchronises the stream.
 * NF_EINVAL: ctx/h_out NULL, N < 0, a NULL buffer with N > 0.
 */
nf_status nf_timestep_ratio(nf_ctx *ctx, const float *d_pos, const float *d_vel, const float *d_acc, int64_t N, double *h_out,
                            void *cuda_stream);

/*
 * nf_accel_host -- the same through HOST buffers: copies h_pos to the device, runs
 * nf_accel, copies the result back into h_acc and synchronises (this is the end-to-end
 * call bench.py times; pinned host memory makes the copies asynchronous DMA).
 * The host-to-device copy is cut into 8 ranges on a second stream and A1 (key +
 * histogram) runs on each range as it lands; A2..A6 need the whole histogram and
 * follow the last range; the device-to-host copy follows the (permuted) un-permute.
 * Errors as nf_accel, plus NF_EPOS for a non-finite position.
 */
nf_status nf_accel_host(nf_ctx *ctx, const float *h_pos, int64_t N, float *h_acc);

/*
 * nf_sync -- wait for the last nf_accel on this context and report deferred errors:
 * NF_EPOS if it saw a non-finite position, NF_ECUDA if the stream failed.
 */
nf_status nf_sync(nf_ctx *ctx);

/* nf_last_error -- text of the last failure ("" if none); owned by ctx (or static if ctx
 * is NULL), valid until the next call on ctx. */
const char *nf_last_error(const nf_ctx *ctx);

/*
 * nf_set_option -- tuning / instrumentation knobs (all have working defaults):
 *   "stage_timing" (0/1)  record CUDA events between stages for nf_stage_ms
 *   "kahan"        (0/1)  compensated fold of per-segment partial sums (default 1)
 *   "heavy_first"  (0/1)  order sink blocks by descending estimated cost instead of grid order
 *                        (default 0: grid order keeps neighbouring blocks' source windows in L2; measured
 *                        no slower on the clustered configs)
 *   "rc_cells"     (<= 0.25) close-pair radius in cell units: pairs with r < rc are evaluated
 *                        exactly in double precision instead of the float32 fast path;
 *                        0 = none (Eq. 3 as a min everywhere); negative (default) = automatic,
 *                        from the particle-weighted occupancy and eps_s.
 *                        Spline law: a positive radius below eps_s is raised to eps_s (the fast
 *                        path evaluates Eq. 3's polynomial only inside the close-pair radius, so the
 *                        radius may not end inside the softened core); the value in
 *                        force is what nf_close_radius reports.  NF_SOFT_NEWTON: at least 1e-4.
 * NF_EINVAL: unknown name or value out of range.
 */
nf_status nf_set_option(nf_ctx *ctx, const char *name, double value);

/*
 * nf_stage_ms -- device time of each stage of the last nf_accel, in milliseconds
 * (needs option "stage_timing" = 1; synchronises):
 *   [0] A1 key+histogram  [1] A2 scans  [2] A3 scatter+rank+gather  [3] A4 scheduler
 *   [4] A5 interaction kernel (with fused A6 un-permute)  [5] whole call  [6],[7] reserved
 */
nf_status nf_stage_ms(nf_ctx *ctx, float *h_ms /* NF_N_STAGES */);

/* ---- exports for the bit-exact checks and for throughput accounting ------------------- */

/*
 * nf_debug_cells -- borrowed device pointers to the grid-order structures of the last
 * nf_accel (valid until the next nf_accel / nf_destroy on ctx; synchronise first):
 *   *d_offsets  uint32[cpd^3 + 1]  first grid-order slot of each cell, key = (cx*cpd+cy)*cpd+cz
 *   *d_perm     uint32[N]          input index of the particle in each grid-order slot;
 *                                  ascending input index within a cell (stable).
 *   *d_sorted   float[4][Npad]     four planes (x, y, z offsets from the cell centre in CELL
 *                                  units, then the cell key as uint32) in PADDED slot order;
 *   *d_poffsets uint32[cpd^3 + 1]  first padded slot of each cell (cells padded to a multiple of 4 slots)
 * Any out-pointer may be NULL.
 */
nf_status nf_debug_cells(nf_ctx *ctx, const uint32_t **d_offsets, const uint32_t **d_perm,
                         const float **d_sorted, const uint32_t **d_poffsets, int64_t *h_npad);

/* nf_close_radius -- the close-pair radius (cell units) the last nf_accel used; 0 = none
 * (see option "rc_cells").  Synchronises. */
nf_status nf_close_radius(nf_ctx *ctx, double *h_rc_cells);

/* nf_bounds_checked -- 1 if this library is the -DNF_DEBUG_BOUNDS build (every index the kernels derive
 * is checked against the bound of its array; nf_sync returns NF_ECUDA "bounds check <code> failed" on a
 * violation), 0 for the product build.  No context needed. */
int nf_bounds_checked(void);

/* nf_launch_count -- number of CUDA kernels this context has launched since nf_create
 * (memsets and copies are not counted).  bench.py reports the difference over its timed region. */
nf_status nf_launch_count(nf_ctx *ctx, int64_t *h_count);

/* nf_debug_read -- copy `bytes` from a device pointer handed out by nf_debug_cells to host
 * memory (synchronous).  NF_EINVAL on NULL arguments. */
nf_status nf_debug_read(nf_ctx *ctx, const void *d_src, void *h_dst, uint64_t bytes);

/*
 * nf_debug_neighbors -- the neighbour list of sink cell `cell` under the enumeration rule of the
 * interaction kernel's stage producer (column images by a single wrap, z by the modulus of the
 * unwrapped index): (2R+1)^3 entries in (a,b,c) lexicographic order, h_ids[n] = neighbour cell
 * key, h_image[3n..3n+2] = periodic image counts in {-1,0,1}.  Produced on
 * the device by a separate one-thread kernel that restates that rule -- it checks the rule, not
 * what the interaction kernel visited; nf_debug_delivered_pairs measures the latter.
 */
nf_status nf_debug_neighbors(nf_ctx *ctx, int cell, int32_t *h_ids, int8_t *h_image);

/*
 * nf_debug_delivered_pairs -- what the interaction kernel's traversal DELIVERS, measured: re-runs
 * the sink blocks of the last nf_accel / nf_accel4 through a counting instantiation of the
 * interaction kernel (same copy ring, stage cursor, z-windows and paired-cell passes; the pair
 * arithmetic replaced by a count of the non-padding sources each pass hands to each non-padding
 * sink).  h_out[0] = (sink, source) deliveries including each sink's meeting with itself,
 * h_out[1] = meetings of a sink with itself.  A correct traversal gives h_out[1] = number of
 * sinks and h_out[0] - h_out[1] = nf_interaction_count = the oracle's pair count (pin P7).
 * Synchronises.  NF_EINVAL: NULL arguments, or the last call on ctx was not nf_accel / nf_accel4.
 */
nf_status nf_debug_delivered_pairs(nf_ctx *ctx, int64_t *h_out /* 2 */);

/*
 * nf_interaction_count -- pairs (sink, source), source != sink, of the last nf_accel:
 * sum_c n_c * sum_{c' in N(c)} n_c'  -  N, computed on the device from the cell offsets (the
 * formula; nf_debug_delivered_pairs is the measurement).  Padding and masked lanes are not work.
 * Synchronises.
 */
nf_status nf_interaction_count(nf_ctx *ctx, int64_t *h_pairs);

#ifdef __cplusplus
}
#endif
#endif /* NEARFIELD_B200_H */
