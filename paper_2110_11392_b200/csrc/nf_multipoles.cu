// nf_multipoles.cu -- nf_multipoles: the cell multipoles of Eq. 4 (sec. 3.3.2) in the
// complete basis, the step after NearForce in the paper's pipeline that "sees" the particles.
//
//     M_{cell}^{a,b,c} = sum_q x_q^a y_q^b z_q^c,  0 <= a <= p, 0 <= b <= p-a, 0 <= c <= p-a-b,
//
// (x_q, y_q, z_q) = offset of particle q from its cell centre, in length units, in double (the
// paper computes the multipoles in double: "double M[cml]").  cml = (p+3)(p+2)(p+1)/6
// values per cell, index order = the (a, b, c) nesting of the paper's pseudo-code.
//
// Two mappings.  Order 8, cells of up to NFM_LANE_MAX particles: k_multipoles_cells, a lane per cell
// (below).  Everything else (other orders; dense cells): k_multipoles, where the
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
    uint32_t *dense, *ndense;         // worklist of the cells k_multipoles_cells leaves to k_multipoles (NULL: all cells)
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
// atomics; 32 consecutive cells per warp.  165 accumulators do not fit in registers, so the basis is
// cut by `a` into three slices (45 + 64 + 56 elements) done one after the other, each re-deriving
// the particle's powers (+15 operations per slice and particle on top of the 165 + 45).  Lanes whose
// cell is shorter than the warp's longest idle: fine at the paper's 30-100 per cell, which is why
// cells above NFM_LANE_MAX go to k_multipoles (one CTA per cell) instead.
#define NFM_LANE_MAX 256

template <int P, int A0, int A1>
__device__ __forceinline__ void mp_slice(const MultipoleArgs &A, uint32_t p0, uint32_t n, double *__restrict__ out) {
    constexpr int base0 = []() { int s = 0; for (int a = 0; a < A0; ++a) s += (P - a + 1) * (P - a + 2) / 2; return s; }();
    constexpr int NT = []() { int s = 0; for (int a = A0; a <= A1; ++a) s += (P - a + 1) * (P - a + 2) / 2; return s; }();
    double acc[NT];
#pragma unroll
    for (int k = 0; k < NT; ++k) acc[k] = 0.0;
    const float *hx = A.sorted, *hy = A.sorted + A.cap_pad, *hz = A.sorted + 2ull * A.cap_pad;
    const float *lx = A.sorted + 4ull * A.cap_pad, *ly = A.sorted + 5ull * A.cap_pad, *lz = A.sorted + 6ull * A.cap_pad;
    // the next four particles are requested before the current four are used: with two warps per
    // scheduler the load latency has to be covered by the lane's own arithmetic
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
            double zp[P + 1];                                            // z^c by squaring: dependency depth 3 instead of P
            zp[0] = 1.0;
            if (P >= 1) zp[1] = Z;
#pragma unroll
            for (int c = 2; c <= P; ++c) zp[c] = zp[c / 2] * zp[c - c / 2];
            double mx = 1.0;
#pragma unroll
            for (int a = 0; a < A0; ++a) mx *= X;
            int idx = 0;
#pragma unroll
            for (int a = A0; a <= A1; ++a) {
                double mxy = mx;
#pragma unroll
                for (int b = 0; b <= P - a; ++b) {
#pragma unroll
                    for (int c = 0; c <= P - a - b; ++c) { acc[idx] = fma(mxy, zp[c], acc[idx]); ++idx; }    // M[a,b,c] += mxy * Zc[c]
                    mxy *= Y;
                }
                mx *= X;
            }
        }
    }
#pragma unroll
    for (int k = 0; k < NT; ++k) out[base0 + k] = acc[k];
}

template <int P>
__global__ void __launch_bounds__(128) k_multipoles_cells(const MultipoleArgs A) {
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= A.ncell) return;
    const uint32_t n = A.offsets[cell + 1] - A.offsets[cell];
    if (n > NFM_LANE_MAX) { A.dense[atomicAdd(A.ndense, 1u)] = (uint32_t)cell; return; }     // k_multipoles takes it
    const uint32_t p0 = A.poff[cell];
    double *out = A.M + (size_t)cell * A.cml;
    mp_slice<P, 0, 0>(A, p0, n, out);
    mp_slice<P, 1, 2>(A, p0, n, out);
    mp_slice<P, 3, P>(A, p0, n, out);
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
    const int nwork = A.dense ? (int)*A.ndense : A.ncell;
    for (int w = blockIdx.x; w < nwork; w += gridDim.x) {
        const int cell = A.dense ? (int)A.dense[w] : w;
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
    A.dense = nullptr; A.ndense = nullptr; A.poff = ctx->d_poff; A.sorted = ctx->d_sorted; A.cap_pad = (uint32_t)ctx->capPad;
    const int64_t want = ctx->ncell;
    const int grid = (int)(want < (int64_t)ctx->sm_count * 2048 ? want : (int64_t)ctx->sm_count * 2048);
    if (order == 8) {        // the paper's order: a lane per cell, then the cells too dense for that by the CTA-per-cell kernel
        A.dense = ctx->d_tmp_perm; A.ndense = ctx->d_ctrl + 6;           // (d_tmp_perm is free once the binning is done)
        NF_CUDA_OK(ctx, cudaMemsetAsync(A.ndense, 0, sizeof(uint32_t), st));
        k_multipoles_cells<8><<<(uint32_t)((want + 127) / 128), 128, 0, st>>>(A); ctx->launches++;
    }
    const int dgrid = order == 8 ? ctx->sm_count * 16 : grid;           // the dense cells only: their number is on the device
    if (order == 8) k_multipoles<8><<<dgrid, nfm_threads(order), 0, st>>>(A);
    else if (order < 8) k_multipoles<8><<<grid, nfm_threads(order), 0, st>>>(A);
    else k_multipoles<NFM_MAX_ORDER><<<grid, nfm_threads(order), 0, st>>>(A);
    ctx->launches++;
    NF_CUDA_OK(ctx, cudaGetLastError());
    return NF_OK;
}
