// nf_multipoles.cu -- nf_multipoles: the cell multipoles of Eq. 4 (sec. 3.3.2) in the
// complete basis, the step after NearForce in the paper's pipeline that "sees" the particles.
//
//     M_{cell}^{a,b,c} = sum_q x_q^a y_q^b z_q^c,  0 <= a <= p, 0 <= b <= p-a, 0 <= c <= p-a-b,
//
// (x_q, y_q, z_q) = offset of particle q from its cell centre, in length units, in double (the
// paper computes the multipoles in double: "double M[cml]").  cml = (p+3)(p+2)(p+1)/6
// values per cell, index order = the (a, b, c) nesting of the paper's pseudo-code.
//
// Mapping (the paper's AVX-512 metacode interleaves particles across vector lanes; here the
// BASIS is spread across threads and the particles of the cell stream past it): one CTA per
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
};

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
    const int64_t want = ctx->ncell;
    const int grid = (int)(want < (int64_t)ctx->sm_count * 2048 ? want : (int64_t)ctx->sm_count * 2048);
    if (order <= 8) k_multipoles<8><<<grid, nfm_threads(order), 0, st>>>(A);
    else k_multipoles<NFM_MAX_ORDER><<<grid, nfm_threads(order), 0, st>>>(A);
    ctx->launches++;
    NF_CUDA_OK(ctx, cudaGetLastError());
    return NF_OK;
}
