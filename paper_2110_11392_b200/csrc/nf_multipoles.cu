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
// BASIS is spread across threads and the particles of the cell stream past it): one CTA of 64
// threads per cell (160 for orders above 9); thread t owns one (a, b) pair (45 pairs at p = 8) and keeps its p-a-b+1
// accumulators in registers; the particles of the cell are staged 32 at a time in shared memory
// as (x, y, z) in double (offsets recomputed from the caller's float32 positions through the
// grid-order permutation of A1-A3); per particle the thread forms x^a y^b z^c by the same
// repeated multiplications as the pseudo-code and adds in ascending grid order, with explicit
// __dmul_rn / __dadd_rn (no FMA contraction), so every element is the pseudo-code's value bit
// for bit.  Bound: FP64 pipe (about 2 cml = 330 flop per 12-byte particle, against 3.2 GB of
// output at config 4).
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

__global__ void __launch_bounds__(160) k_multipoles(const MultipoleArgs A) {
    __shared__ double sx[NFM_TILE], sy[NFM_TILE], sz[NFM_TILE];
    const int p = A.order;
    // thread t -> (a, b) in the nesting order of the basis, and the index of its first element
    int a = 0, b = 0, base = 0, nc = 0;
    {
        int t = (int)threadIdx.x, idx = 0;
        bool found = false;
        for (int aa = 0; aa <= p && !found; ++aa)
            for (int bb = 0; bb <= p - aa; ++bb) {
                if (t == 0) { a = aa; b = bb; base = idx; nc = p - aa - bb + 1; found = true; break; }
                --t;
                idx += p - aa - bb + 1;
            }
        if (!found) nc = 0;          // spare thread: only helps with the loads
    }
    for (int cell = blockIdx.x; cell < A.ncell; cell += gridDim.x) {
        const uint32_t p0 = A.offsets[cell], p1 = A.offsets[cell + 1];
        double acc[NFM_MAX_ORDER + 1];
#pragma unroll
        for (int c = 0; c <= NFM_MAX_ORDER; ++c) acc[c] = 0.0;
        for (uint32_t pb = p0; pb < p1; pb += NFM_TILE) {
            __syncthreads();
            const uint32_t q = pb + threadIdx.x;
            if (threadIdx.x < NFM_TILE && q < p1) {
                const float *s = A.pos + 3ull * A.perm[q];
                const double tx = (double)s[0] * A.scale, ty = (double)s[1] * A.scale, tz = (double)s[2] * A.scale;
                sx[threadIdx.x] = (tx - floor(tx) - 0.5) * A.cellsz;     // offset from the cell centre (reading S5)
                sy[threadIdx.x] = (ty - floor(ty) - 0.5) * A.cellsz;
                sz[threadIdx.x] = (tz - floor(tz) - 0.5) * A.cellsz;
            }
            __syncthreads();
            if (nc == 0) continue;
            const int nt = (int)min((uint32_t)NFM_TILE, p1 - pb);
            for (int t = 0; t < nt; ++t) {
                const double X = sx[t], Y = sy[t], Z = sz[t];
                double m = 1.0;
                for (int i = 0; i < a; ++i) m = __dmul_rn(m, X);      // mx   = x^a   (mx *= X)
                for (int i = 0; i < b; ++i) m = __dmul_rn(m, Y);      // mxy  = mx y^b (mxy *= Y)
#pragma unroll
                for (int c = 0; c <= NFM_MAX_ORDER; ++c) {
                    if (c < nc) {
                        acc[c] = __dadd_rn(acc[c], m);                 // M[a,b,c] += mxyz
                        m = __dmul_rn(m, Z);                           // mxyz *= Z
                    }
                }
            }
        }
        if (nc > 0) {
            double *o = A.M + (size_t)cell * A.cml + base;
#pragma unroll
            for (int c = 0; c <= NFM_MAX_ORDER; ++c)
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
    k_multipoles<<<grid, nfm_threads(order), 0, st>>>(A); ctx->launches++;
    NF_CUDA_OK(ctx, cudaGetLastError());
    return NF_OK;
}
