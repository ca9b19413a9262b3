// nf_f64.cu -- nf_accel_f64: the near-field sum in double precision on the GPU.
//
// The paper's build has a "Double precision" switch (Fig. 19) and suggests
// validating the float32 kernel against a double one.  This is that build as
// a second entry point: same binning (A1-A3), then a plain tiled direct sum in double --
// offsets recomputed in double from the caller's float32 positions (not the float32 planes),
// integer cell shift added last, piecewise Eq. 3, Eq. 2 or the
// unsoftened r/|r|^3 with a branch, one accumulator per sink, sources of a cell in ascending input order.  No packed
// arithmetic, no clamping, no close-pair path: it is the reference the fast kernel can be held
// against on EVERY particle of a full-size input (tests/test_gpu_f64.py), where the CPU oracle
// only reaches samples.  Not on the timed path.
#include "nf_common.cuh"

#define NF64_THREADS 128

struct F64Args {
    const float *pos;
    const uint32_t *offsets, *perm;      // true (unpadded) grid order
    double *acc;                          // N x 3, input order
    double scale, cellsz, eps_s, eps_p, gm;
    int cpd, R, law, x0, nx;
    uint32_t *counter;                    // work counter over sink cells
};

__device__ __forceinline__ double off64(float x, double scale, double cellsz) {
    const double t = (double)x * scale;
    return (t - floor(t) - 0.5) * cellsz;          // offset from the cell centre, length units (reading S5)
}

__global__ void __launch_bounds__(NF64_THREADS) k_direct_f64(const F64Args A) {
    __shared__ double sx[NF64_THREADS], sy[NF64_THREADS], sz[NF64_THREADS];
    __shared__ uint32_t s_cell;
    const int cpd = A.cpd, R = A.R, ncell = cpd * cpd * cpd;
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) s_cell = atomicAdd(A.counter, 1u);
        __syncthreads();
        const int C = (int)s_cell;
        if (C >= ncell) return;
        const uint32_t p0 = A.offsets[C], p1 = A.offsets[C + 1];
        if (p0 == p1) continue;
        const int ck = C % cpd, cj = (C / cpd) % cpd, ci = C / (cpd * cpd);
        { int d = ci - A.x0; if (d < 0) d += cpd; if (d >= A.nx) continue; }      // not a sink slab
        for (uint32_t pb = p0; pb < p1; pb += NF64_THREADS) {
            const uint32_t p = pb + threadIdx.x;
            const bool live = p < p1;
            uint32_t pi = 0;
            double px = 0, py = 0, pz = 0, ax = 0, ay = 0, az = 0;
            if (live) {
                pi = A.perm[p];
                const float *q = A.pos + 3ull * pi;
                px = off64(q[0], A.scale, A.cellsz); py = off64(q[1], A.scale, A.cellsz); pz = off64(q[2], A.scale, A.cellsz);
            }
            for (int a = -R; a <= R; ++a) {
                int ia; const int sci = nf_wrap1(ci + a, cpd, ia);
                for (int b = -R; b <= R; ++b) {
                    int ib; const int scj = nf_wrap1(cj + b, cpd, ib);
                    for (int c = -R; c <= R; ++c) {
                        const int sck = nf_mod(ck + c, cpd);
                        const int S = (sci * cpd + scj) * cpd + sck;
                        const uint32_t q0 = A.offsets[S], q1 = A.offsets[S + 1];
                        const double shx = a * A.cellsz, shy = b * A.cellsz, shz = c * A.cellsz;
                        for (uint32_t qb = q0; qb < q1; qb += NF64_THREADS) {
                            __syncthreads();
                            const uint32_t qq = qb + threadIdx.x;
                            if (qq < q1) {
                                const float *s = A.pos + 3ull * A.perm[qq];
                                sx[threadIdx.x] = off64(s[0], A.scale, A.cellsz);
                                sy[threadIdx.x] = off64(s[1], A.scale, A.cellsz);
                                sz[threadIdx.x] = off64(s[2], A.scale, A.cellsz);
                            }
                            __syncthreads();
                            if (!live) continue;
                            const int nt = (int)min((uint32_t)NF64_THREADS, q1 - qb);
                            for (int t = 0; t < nt; ++t) {
                                if (qb + t == p) continue;                       // the particle itself
                                const double dx = (sx[t] - px) + shx, dy = (sy[t] - py) + shy, dz = (sz[t] - pz) + shz;
                                const double r2 = dx * dx + dy * dy + dz * dz;
                                if (r2 == 0.0) continue;                         // F(0) = 0 (reading S4)
                                double f;
                                if (A.law == NF_SOFT_PLUMMER) {
                                    const double s2 = r2 + A.eps_p * A.eps_p;
                                    f = 1.0 / (s2 * sqrt(s2));
                                } else if (A.law == NF_SOFT_NEWTON) {
                                    f = 1.0 / (r2 * sqrt(r2));                  // no softening
                                } else {
                                    const double r = sqrt(r2);
                                    if (r < A.eps_s) {
                                        const double u = r / A.eps_s;
                                        f = (10.0 - 15.0 * u + 6.0 * u * u) / (A.eps_s * A.eps_s * A.eps_s);
                                    } else {
                                        f = 1.0 / (r2 * r);
                                    }
                                }
                                ax += A.gm * f * dx; ay += A.gm * f * dy; az += A.gm * f * dz;
                            }
                        }
                    }
                }
            }
            if (live) {
                double *o = A.acc + 3ull * pi;
                o[0] = ax; o[1] = ay; o[2] = az;
            }
        }
    }
}

nf_status nf_run_f64(nf_ctx *ctx, const float *d_pos, int64_t N, double *d_acc, cudaStream_t st) {
    F64Args A;
    A.pos = d_pos; A.offsets = ctx->d_offsets; A.perm = ctx->d_perm_true; A.acc = d_acc;
    A.scale = ctx->prm.scale; A.cellsz = ctx->box / (double)ctx->cpd;
    A.eps_p = ctx->eps_p; A.eps_s = NF_SPLINE_PER_PLUMMER * ctx->eps_p;
    A.gm = ctx->gm > 0 ? ctx->gm : 1.0 / (double)N;
    A.cpd = ctx->cpd; A.R = ctx->R; A.law = ctx->law; A.x0 = ctx->slab_x0; A.nx = ctx->slab_nx;
    A.counter = ctx->d_ctrl + 104;
    NF_CUDA_OK(ctx, cudaMemsetAsync(A.counter, 0, 4, st));
    const int grid = ctx->sm_count * 8;
    k_direct_f64<<<grid, NF64_THREADS, 0, st>>>(A); ctx->launches++;
    NF_CUDA_OK(ctx, cudaGetLastError());
    return NF_OK;
}
