// nf_multipoles.cu -- nf_multipoles: the cell multipoles of Eq. 4 (sec. 3.3.2) in the
// complete basis, the step after NearForce in the paper's pipeline that "sees" the particles.
//
//     M_{cell}^{a,b,c} = sum_q x_q^a y_q^b z_q^c,  0 <= a <= p, 0 <= b <= p-a, 0 <= c <= p-a-b,
//
// (x_q, y_q, z_q) = offset of particle q from its cell centre, in length units, in double (the
// paper computes the multipoles in double: "double M[cml]").  cml = (p+3)(p+2)(p+1)/6
// values per cell, index order = the (a, b, c) nesting of the paper's pseudo-code.
//
// Two mappings.  Order 8 (the paper's): k_multipoles_cells, a lane per cell -- or per 512-particle
// chunk of a cell denser than NFM_LANE_MAX, whose partial sums k_mp_reduce adds (below).  The other
// orders: k_multipoles, where the
// BASIS is spread across threads and the particles of the cell stream past it: one CTA per
// cell, 64 threads up to order 9 (160 above); thread t owns one (a, b) pair -- pairs sorted by
// descending element count p-a-b+1, so that the first warp holds the long ones and the second
// warp's loop is short (p = 8: 45 pairs, warp bounds 9 and 2) -- and keeps its accumulators in
// registers.  The particles of the cell are staged 32 at a time in shared memory as power
// tables x^0..p, y^0..p, z^0..p in double (offsets recomputed from the caller's float32
// positions through the grid-order permutation of A1-A3, powers by repeated multiplication as
// in the pseudo-code); per particle a thread reads x^a and y^b (conflict-free multicast), forms
// m = x^a y^b and does M[a,b,c] += m z^c as one FMA per element with z^c broadcast from shared
// memory -- the FMA form the paper itself proposes ("M[a,b,c] += mxy*Zc[c]").
// Particles are added in ascending grid order.  Bound: FP64 pipe (cml FMAs + (p+1)(p+2)/2
// multiplies + 3p table multiplies per 12-byte particle, against 3.2 GB of output at config 4).
#include <type_traits>
#include "nf_common.cuh"

#define NFM_TILE 32
#define NFM_MAX_ORDER NF_MAX_MULTIPOLE_ORDER
// threads per CTA >= (p+1)(p+2)/2 pairs (a, b): 64 up to p = 9 (55 pairs; 45 at the paper's p = 8), 160 up to p = 16 (153)
static int nfm_threads(int order) { return order <= 9 ? 64 : 160; }

struct MultipoleArgs {
    const float *pos;
    const uint32_t *offsets, *perm;   // true (unpadded) grid order
    double *M;
    double scale, cellsz;
    int ncell, order, cml;
    const uint32_t *poff;             // first padded slot of each cell
    const float *sorted;              // the NF_PLANES sorted planes (hi offsets 0-2, lo remainders 4-6)
    uint32_t cap_pad;
};

// ---- order 8, cells of up to NFM_LANE_MAX particles: ONE LANE PER CELL --------------------------
// (the paper's AVX-512 code keeps a cell's accumulators in registers and streams its particles past
// them; so does a lane here.)  A lane owns one cell: it streams the cell's particles
// from the sorted planes (hi + lo float32 = the double-precision offset to 2^-48; four particles per
// 16-byte load and plane: cells are padded to 4 slots) and accumulates M[a,b,c] += (x^a y^b) z^c as
// one DFMA per element into REGISTER accumulators -- no shared memory, no cross-lane reduction, no
// atomics.  165 accumulators do not fit in registers, so the basis is cut into two slices of whole
// (a, b) rows (88 + 77 elements) done one after the other, each re-reading the cell and re-deriving
// the particle's offsets and powers: every extra slice costs a pass (measured: 3 slices +7 %, 7
// slices 2.1x, although they allow twice the warps), so the slices are as large as 255 registers
// hold.  A warp takes as long as its longest cell, so the lanes take their cells from a list sorted
// by DESCENDING occupancy (k_mp_hist / k_mp_scan / k_mp_fill: a counting sort of the cell indices):
// the 32 cells of a warp are equally long and the longest cells start first.  At 64 +- 8 per cell
// this costs a little locality (+1 %); in the clustered configs, where neighbouring cells hold 5 and
// 500, it is worth 20-25 %.  Cells above NFM_LANE_MAX are cut into chunks that are work items of their own.
#define NFM_LANE_MAX 1024

// The basis is cut into SLICES of whole (a, b) rows, filled greedily in index order up to NFM_SLICE_CAP
// accumulators; slice_of(a, b) and the slice bounds are compile-time, so every test below folds away.
#define NFM_SLICE_CAP 90      // 2 slices (88 + 77 accumulators) at p = 8: 255 registers, no spills, 2 warps per scheduler
template <int P> struct MpSlices {
    int sid[P + 1][P + 1];     // slice of row (a, b)
    int base[64], cnt[64];     // first basis index and element count of a slice
    int amin[64], amax[64], smax[64];   // range of a, and the largest power of y and z (P - a - b + ... ) a slice needs
    int n;
    constexpr MpSlices() : sid{}, base{}, cnt{}, amin{}, amax{}, smax{}, n(0) {
        int cur = 0, fill = 0, idx = 0;
        base[0] = 0; amin[0] = 0;
        for (int a = 0; a <= P; ++a)
            for (int b = 0; b <= P - a; ++b) {
                const int len = P - a - b + 1;
                if (fill > 0 && fill + len > NFM_SLICE_CAP) { cnt[cur] = fill; ++cur; fill = 0; base[cur] = idx; amin[cur] = a; smax[cur] = 0; }
                sid[a][b] = cur;
                amax[cur] = a;
                if (b > smax[cur]) smax[cur] = b;
                if (len - 1 > smax[cur]) smax[cur] = len - 1;
                fill += len; idx += len;
            }
        cnt[cur] = fill;
        n = cur + 1;
    }
};

template <int P, int SID>
__device__ __forceinline__ void mp_slice(const MultipoleArgs &A, uint32_t p0, uint32_t n, double *__restrict__ out) {
    constexpr MpSlices<P> SL{};
    constexpr int base0 = SL.base[SID], NT = SL.cnt[SID], A0 = SL.amin[SID], A1 = SL.amax[SID], SMAX = SL.smax[SID];
    double acc[NT];
#pragma unroll
    for (int k = 0; k < NT; ++k) acc[k] = 0.0;
    const float *hx = A.sorted, *hy = A.sorted + A.cap_pad, *hz = A.sorted + 2ull * A.cap_pad;
    const float *lx = A.sorted + 4ull * A.cap_pad, *ly = A.sorted + 5ull * A.cap_pad, *lz = A.sorted + 6ull * A.cap_pad;
    // the next four particles are requested before the current four are used: the load latency has to
    // be covered by the lane's own arithmetic
    float4 HX, HY, HZ, LX, LY, LZ, nHX, nHY, nHZ, nLX, nLY, nLZ;
    auto fetch = [&](uint32_t j, float4 &a0, float4 &a1, float4 &a2, float4 &a3, float4 &a4, float4 &a5) {
        a0 = __ldg(reinterpret_cast<const float4 *>(hx + p0 + j)); a1 = __ldg(reinterpret_cast<const float4 *>(hy + p0 + j));
        a2 = __ldg(reinterpret_cast<const float4 *>(hz + p0 + j)); a3 = __ldg(reinterpret_cast<const float4 *>(lx + p0 + j));
        a4 = __ldg(reinterpret_cast<const float4 *>(ly + p0 + j)); a5 = __ldg(reinterpret_cast<const float4 *>(lz + p0 + j));
    };
    if (n > 0) fetch(0, nHX, nHY, nHZ, nLX, nLY, nLZ);
    for (uint32_t j = 0; j < n; j += 4) {
        HX = nHX; HY = nHY; HZ = nHZ; LX = nLX; LY = nLY; LZ = nLZ;
        if (j + 4 < n) fetch(j + 4, nHX, nHY, nHZ, nLX, nLY, nLZ);
#pragma unroll 1
        for (int k = 0; k < 4; ++k) {
            if (j + k >= n) break;                                       // the cell's padding slots
            auto pick = [k](const float4 &v) { return k == 0 ? v.x : (k == 1 ? v.y : (k == 2 ? v.z : v.w)); };   // selects, no local memory
            const double X = ((double)pick(HX) + (double)pick(LX)) * A.cellsz, Y = ((double)pick(HY) + (double)pick(LY)) * A.cellsz,
                         Z = ((double)pick(HZ) + (double)pick(LZ)) * A.cellsz;
            // powers by squaring (dependency depth 3 instead of P): the products x^a y^b of the rows are
            // independent of one another, so the FMAs of one row never wait for the previous row's multiply
            double zp[P + 1], yp[P + 1], xp[P + 1];
            zp[0] = 1.0; yp[0] = 1.0; xp[0] = 1.0;
            if (P >= 1) { zp[1] = Z; yp[1] = Y; xp[1] = X; }
#pragma unroll
            for (int c = 2; c <= SMAX; ++c) { zp[c] = zp[c / 2] * zp[c - c / 2]; yp[c] = yp[c / 2] * yp[c - c / 2]; }
#pragma unroll
            for (int c = 2; c <= A1; ++c) xp[c] = xp[c / 2] * xp[c - c / 2];
            int idx = 0;
#pragma unroll
            for (int a = A0; a <= A1; ++a) {
#pragma unroll
                for (int b = 0; b <= P - a; ++b) {
                    if (SL.sid[a][b] != SID) continue;
                    const double mxy = (a == 0) ? yp[b] : ((b == 0) ? xp[a] : xp[a] * yp[b]);
#pragma unroll
                    for (int c = 0; c <= P - a - b; ++c) { acc[idx] = fma(mxy, zp[c], acc[idx]); ++idx; }    // M[a,b,c] += mxy * Zc[c]
                }
            }
        }
    }
#pragma unroll
    for (int k = 0; k < NT; ++k) out[base0 + k] = acc[k];
}
template <int P, int SID>
__device__ __forceinline__ void mp_all_slices(const MultipoleArgs &A, uint32_t p0, uint32_t n, double *__restrict__ out) {
    constexpr MpSlices<P> SL{};
    if constexpr (SID < SL.n) {
        mp_slice<P, SID>(A, p0, n, out);
        mp_all_slices<P, SID + 1>(A, p0, n, out);
    }
}

// The lane kernel's WORK ITEMS are cells of up to NFM_LANE_MAX particles and, for the denser cells of a
// clustered state, CHUNKS of NFM_CHUNK consecutive particles of one cell; a chunk's result goes to a
// partial buffer and k_mp_reduce adds a cell's partials in chunk order (a fixed order: deterministic).
// The items are sorted by DESCENDING particle count (counting sort: class = NFM_LANE_MAX - count), so the
// 32 items of a warp are equally long and the longest start first.  hist[0 .. NFM_NCLASS) per class, then
// its exclusive scan (k_mp_scan), then the running cursors of k_mp_fill; hist[NFM_NCLASS] = number of items;
// hist[NFM_CTR_CHUNK] / hist[NFM_CTR_DENSE] count the chunks and the dense cells.  The order within a class
// is whatever the atomics give: which lane computes an item does not change its result.
// A dense cell (n > NFM_LANE_MAX = 2 NFM_CHUNK) has ceil(n / NFM_CHUNK) chunks; chunks per particle are most at
// n = NFM_LANE_MAX + 1 (3 chunks for 1025 particles), so the partials of any input take at most
// 3 * 165 * 8 B / 1025 = 3.87 B per particle of a dense cell -- inside the partial buffer (the binner's chunk
// scratch: 4 capPad bytes >= 4 B per particle) with 3 % to spare; the static_assert below keeps it so.
#define NFM_CHUNK 512
#define NFM_NCLASS (NFM_LANE_MAX + 1)
#define NFM_CTR_CHUNK (NFM_NCLASS + 1)
#define NFM_CTR_DENSE (NFM_NCLASS + 2)
static_assert(NFM_LANE_MAX == 2 * NFM_CHUNK, "the bound on the number of chunks assumes it");
static_assert(((NFM_LANE_MAX + 1 + NFM_CHUNK - 1) / NFM_CHUNK) * 165 * 8 <= 4 * (NFM_LANE_MAX + 1),
              "the order-8 chunk partials (165 doubles per chunk) must fit 4 bytes per particle of a dense cell");
__device__ __forceinline__ uint32_t mp_class(uint32_t cnt) { return NFM_LANE_MAX - cnt; }   // longest first
__global__ void __launch_bounds__(256) k_mp_hist(int ncell, const uint32_t *__restrict__ offsets, uint32_t *__restrict__ hist) {
    __shared__ uint32_t h[NFM_NCLASS];
    for (int i = threadIdx.x; i < NFM_NCLASS; i += blockDim.x) h[i] = 0u;
    __syncthreads();
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < ncell; c += gridDim.x * blockDim.x) {
        const uint32_t n = offsets[c + 1] - offsets[c];
        if (n <= NFM_LANE_MAX) atomicAdd(&h[mp_class(n)], 1u);
        else {
            atomicAdd(&h[mp_class(NFM_CHUNK)], n / NFM_CHUNK);
            if (n % NFM_CHUNK) atomicAdd(&h[mp_class(n % NFM_CHUNK)], 1u);
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < NFM_NCLASS; i += blockDim.x) if (h[i]) atomicAdd(&hist[i], h[i]);
}
__global__ void __launch_bounds__(256) k_mp_scan(uint32_t *hist) {      // one block: exclusive scan of the NFM_NCLASS class counts in place
    constexpr int PER = (NFM_NCLASS + 255) / 256;
    __shared__ uint32_t part[256];
    uint32_t v[PER], s = 0;
#pragma unroll
    for (int k = 0; k < PER; ++k) { const int i = threadIdx.x * PER + k; v[k] = i < NFM_NCLASS ? hist[i] : 0u; s += v[k]; }
    part[threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.x == 0) { uint32_t t = 0; for (int i = 0; i < 256; ++i) { const uint32_t x = part[i]; part[i] = t; t += x; } hist[NFM_NCLASS] = t; }
    __syncthreads();
    uint32_t e = part[threadIdx.x];
#pragma unroll
    for (int k = 0; k < PER; ++k) {
        const int i = threadIdx.x * PER + k;
        if (i < NFM_NCLASS) hist[i] = e;
        e += v[k];
    }
}
struct MpItems { uint32_t *cell, *chunk, *pidx; };     // item w: particles [chunk * NFM_CHUNK, ...) of `cell`; pidx = its partial (0xffffffff: straight to M)
struct MpDense { uint32_t cell, first, nchunk; };      // a dense cell: its partials are first .. first + nchunk - 1
#define NFM_FILL_ITEMS 8
__global__ void __launch_bounds__(256) k_mp_fill(int ncell, const uint32_t *__restrict__ offsets, uint32_t *__restrict__ hist, MpItems I,
                                                 MpDense *__restrict__ dense) {
    __shared__ uint32_t h[NFM_NCLASS];
    for (int i = threadIdx.x; i < NFM_NCLASS; i += blockDim.x) h[i] = 0u;
    __syncthreads();
    uint32_t cls[NFM_FILL_ITEMS], rank[NFM_FILL_ITEMS];
    const int c0 = blockIdx.x * (256 * NFM_FILL_ITEMS) + threadIdx.x;
#pragma unroll
    for (int k = 0; k < NFM_FILL_ITEMS; ++k) {
        const int c = c0 + k * 256;
        cls[k] = 0xffffffffu;
        if (c < ncell) {
            const uint32_t n = offsets[c + 1] - offsets[c];
            if (n <= NFM_LANE_MAX) { cls[k] = mp_class(n); rank[k] = atomicAdd(&h[cls[k]], 1u); }
            else {                                            // a dense cell (rare): its chunks take their places one by one
                const uint32_t nch = (n + NFM_CHUNK - 1) / NFM_CHUNK;
                const uint32_t first = atomicAdd(&hist[NFM_CTR_CHUNK], nch);
                MpDense d; d.cell = (uint32_t)c; d.first = first; d.nchunk = nch;
                dense[atomicAdd(&hist[NFM_CTR_DENSE], 1u)] = d;
                for (uint32_t ch = 0; ch < nch; ++ch) {
                    const uint32_t cnt = (ch + 1u) * NFM_CHUNK <= n ? NFM_CHUNK : n - ch * NFM_CHUNK;
                    const uint32_t w = atomicAdd(&hist[mp_class(cnt)], 1u);
                    I.cell[w] = (uint32_t)c; I.chunk[w] = ch; I.pidx[w] = first + ch;
                }
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < NFM_NCLASS; i += blockDim.x) if (h[i]) h[i] = atomicAdd(&hist[i], h[i]);      // the block's range in class i
    __syncthreads();
#pragma unroll
    for (int k = 0; k < NFM_FILL_ITEMS; ++k) {
        const int c = c0 + k * 256;
        if (cls[k] != 0xffffffffu) { const uint32_t w = h[cls[k]] + rank[k]; I.cell[w] = (uint32_t)c; I.chunk[w] = 0u; I.pidx[w] = 0xffffffffu; }
    }
}

template <int P>
__global__ void __launch_bounds__(128, 2) k_multipoles_cells(const MultipoleArgs A, const MpItems I, const uint32_t *__restrict__ nitems,
                                                             double *__restrict__ partial) {
    const uint32_t w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= *nitems) return;
    const int cell = (int)I.cell[w];
    const uint32_t j0 = I.chunk[w] * NFM_CHUNK, pidx = I.pidx[w];
    const uint32_t ncell_p = A.offsets[cell + 1] - A.offsets[cell];
    const uint32_t n = pidx == 0xffffffffu ? ncell_p : (j0 + NFM_CHUNK <= ncell_p ? NFM_CHUNK : ncell_p - j0);
    const uint32_t p0 = A.poff[cell] + j0;                // chunks start on multiples of 4 slots
    double *out = pidx == 0xffffffffu ? A.M + (size_t)cell * A.cml : partial + (size_t)pidx * A.cml;
    mp_all_slices<P, 0>(A, p0, n, out);
}

// M of a dense cell = its chunks' partials added in chunk order
__global__ void __launch_bounds__(192) k_mp_reduce(const uint32_t *__restrict__ hist, const MpDense *__restrict__ dense, const double *__restrict__ partial,
                                                   double *__restrict__ M, int cml) {
    const uint32_t nd = hist[NFM_CTR_DENSE];
    for (uint32_t d = blockIdx.x; d < nd; d += gridDim.x) {
        const MpDense D = dense[d];
        for (int e = threadIdx.x; e < cml; e += blockDim.x) {
            double s = 0.0;
            for (uint32_t ch = 0; ch < D.nchunk; ++ch) s += partial[(size_t)(D.first + ch) * cml + e];
            M[(size_t)D.cell * cml + e] = s;
        }
    }
}

// PMAX = compile-time bound of the order (8: the paper's choice; NFM_MAX_ORDER: any order)
template <int PMAX>
__global__ void __launch_bounds__(160) k_multipoles(const MultipoleArgs A) {
    constexpr int ZROW = (PMAX + 2) & ~1;       // z-power rows padded to an even length: read as double2 (LDS.128 broadcasts)
    __shared__ double xp[NFM_TILE][PMAX + 1], yp[NFM_TILE][PMAX + 1];
    __shared__ __align__(16) double zp[NFM_TILE][ZROW];
    const int p = A.order;
    // thread t -> the t-th (a, b) pair in order of descending element count nc = p - a - b + 1
    // (ties in basis order), and the index of the pair's first element in the basis order
    int a = 0, b = 0, base = 0, nc = 0;
    {
        int t = (int)threadIdx.x;
        for (int want = p + 1; want >= 1 && nc == 0; --want) {       // pairs with a + b = p + 1 - want
            int idx = 0;
            for (int aa = 0; aa <= p && nc == 0; ++aa)
                for (int bb = 0; bb <= p - aa; ++bb) {
                    const int n = p - aa - bb + 1;
                    if (n == want) {
                        if (t == 0) { a = aa; b = bb; base = idx; nc = n; break; }
                        --t;
                    }
                    idx += n;
                }
        }
    }
    // longest element count in this warp (warp-uniform loop bound)
    int ncw = nc;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) ncw = max(ncw, __shfl_xor_sync(0xffffffffu, ncw, d));
    for (int cell = blockIdx.x; cell < A.ncell; cell += gridDim.x) {
        const uint32_t p0 = A.offsets[cell], p1 = A.offsets[cell + 1];
        double acc[PMAX + 1];
#pragma unroll
        for (int c = 0; c <= PMAX; ++c) acc[c] = 0.0;
        for (uint32_t pb = p0; pb < p1; pb += NFM_TILE) {
            __syncthreads();
            const uint32_t q = pb + threadIdx.x;
            if (threadIdx.x < NFM_TILE && q < p1) {
                const float *s = A.pos + 3ull * A.perm[q];
                const double tx = (double)s[0] * A.scale, ty = (double)s[1] * A.scale, tz = (double)s[2] * A.scale;
                const double X = (tx - floor(tx) - 0.5) * A.cellsz;     // offset from the cell centre (reading S5)
                const double Y = (ty - floor(ty) - 0.5) * A.cellsz;
                const double Z = (tz - floor(tz) - 0.5) * A.cellsz;
                double mx = 1.0, my = 1.0, mz = 1.0;
#pragma unroll
                for (int k = 0; k <= PMAX; ++k) {
                    if (k <= p) {
                        xp[threadIdx.x][k] = mx; yp[threadIdx.x][k] = my; zp[threadIdx.x][k] = mz;
                        mx *= X; my *= Y; mz *= Z;
                    }
                }
#pragma unroll
                for (int k = 0; k < ZROW; ++k)
                    if (k > p) zp[threadIdx.x][k] = 0.0;           // unused powers read as 0: the extra FMA of a pair adds nothing
            }
            __syncthreads();
            if (ncw == 0) continue;
            const int nt = (int)min((uint32_t)NFM_TILE, p1 - pb);
            // the loop over the tile's particles, with the warp's element bound NCW as a compile-time
            // constant where it is known (p = 8: 9 for the first warp, 2 for the second): no predicates
            auto tile = [&](auto ncw_tag) {
                constexpr int NCW = decltype(ncw_tag)::value;
                const double *xr = &xp[0][a], *yr = &yp[0][b];
                for (int t = 0; t < nt; ++t) {
                    const double m = xr[t * (PMAX + 1)] * yr[t * (PMAX + 1)];
                    const double2 *zr = reinterpret_cast<const double2 *>(zp[t]);
#pragma unroll
                    for (int c = 0; c < (NCW > 0 ? NCW : PMAX + 1); c += 2) {
                        if (NCW > 0 || c < ncw) {
                            const double2 zz = zr[c >> 1];
                            acc[c] = fma(m, zz.x, acc[c]);                      // M[a,b,c] += mxy * Zc[c]
                            if (c + 1 <= PMAX) acc[c + 1 <= PMAX ? c + 1 : c] = fma(m, zz.y, acc[c + 1 <= PMAX ? c + 1 : c]);
                        }
                    }
                }
            };
            if (PMAX == 8 && ncw == 9) tile(std::integral_constant<int, 9>{});
            else if (PMAX == 8 && ncw == 2) tile(std::integral_constant<int, 2>{});
            else tile(std::integral_constant<int, 0>{});
        }
        if (nc > 0) {
            double *o = A.M + (size_t)cell * A.cml + base;
#pragma unroll
            for (int c = 0; c <= PMAX; ++c)
                if (c < nc) o[c] = acc[c];
        }
    }
}

nf_status nf_run_multipoles(nf_ctx *ctx, const float *d_pos, int order, double *d_M, cudaStream_t st) {
    MultipoleArgs A;
    A.pos = d_pos; A.offsets = ctx->d_offsets; A.perm = ctx->d_perm_true; A.M = d_M;
    A.scale = ctx->prm.scale; A.cellsz = ctx->box / (double)ctx->cpd;
    A.ncell = (int)ctx->ncell; A.order = order; A.cml = (order + 3) * (order + 2) * (order + 1) / 6;
    A.poff = ctx->d_poff; A.sorted = ctx->d_sorted; A.cap_pad = (uint32_t)ctx->capPad;
    const int64_t want = ctx->ncell;
    const int grid = (int)(want < (int64_t)ctx->sm_count * 2048 ? want : (int64_t)ctx->sm_count * 2048);
    if (order == 8) {        // the paper's order: a lane per work item (cell, or chunk of a dense cell), then the dense cells' partials are added
        uint32_t *hist = ctx->d_mp_hist;
        MpItems I;                                                       // (d_tmp_perm, d_key and d_chunk_sorted are free once the binning is done)
        const size_t icap = (size_t)ctx->capPad / 3;                     // >= ncell + N / NFM_CHUNK items
        I.cell = ctx->d_tmp_perm; I.chunk = ctx->d_tmp_perm + icap; I.pidx = ctx->d_tmp_perm + 2 * icap;
        MpDense *dense = reinterpret_cast<MpDense *>(ctx->d_key);        // <= N / NFM_LANE_MAX dense cells of 3 words
        double *partial = reinterpret_cast<double *>(ctx->d_chunk_sorted);
        NF_CUDA_OK(ctx, cudaMemsetAsync(hist, 0, (NFM_NCLASS + 4) * sizeof(uint32_t), st));
        const int hgrid = (int)(want / 256 + 1 < (int64_t)ctx->sm_count * 8 ? want / 256 + 1 : (int64_t)ctx->sm_count * 8);
        k_mp_hist<<<hgrid, 256, 0, st>>>(A.ncell, A.offsets, hist); ctx->launches++;
        k_mp_scan<<<1, 256, 0, st>>>(hist); ctx->launches++;
        k_mp_fill<<<(uint32_t)((want + 256 * NFM_FILL_ITEMS - 1) / (256 * NFM_FILL_ITEMS)), 256, 0, st>>>(A.ncell, A.offsets, hist, I, dense); ctx->launches++;
        const uint64_t items = (uint64_t)want + (uint64_t)ctx->lastN / NFM_CHUNK + 1;      // upper bound of the item count, known on the host
        k_multipoles_cells<8><<<(uint32_t)((items + 127) / 128), 128, 0, st>>>(A, I, hist + NFM_NCLASS, partial); ctx->launches++;
        k_mp_reduce<<<ctx->sm_count * 8, 192, 0, st>>>(hist, dense, partial, A.M, A.cml); ctx->launches++;
        NF_CUDA_OK(ctx, cudaGetLastError());
        return NF_OK;
    }
    if (order < 8) k_multipoles<8><<<grid, nfm_threads(order), 0, st>>>(A);
    else k_multipoles<NFM_MAX_ORDER><<<grid, nfm_threads(order), 0, st>>>(A);
    ctx->launches++;
    NF_CUDA_OK(ctx, cudaGetLastError());
    return NF_OK;
}
