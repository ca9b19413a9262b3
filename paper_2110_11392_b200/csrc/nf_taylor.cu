// nf_taylor.cu -- nf_taylor_accel: the far-field acceleration of every particle from its cell's
// Taylor series of the potential, the step before NearForce in the paper's
// pipeline (TaylorForce, Table 1).  Reading F1: coefficients T^{a,b,c} of
//     phi(x,y,z) = sum_{a+b+c <= p} T^{a,b,c} x^a y^b z^c,   (x,y,z) = offset from the cell centre,
// in the complete basis and index order of nf_multipoles;  a = -grad phi.
//
// Mapping (orders other than 8; order 8 runs k_taylor_slots below): one CTA of 64 threads per cell; the cell's cml coefficients are staged once in shared
// memory (all threads then read the same coefficient: broadcast), one particle per thread (more
// in turn for fuller cells) with its power tables x^k, y^k, z^k in registers, in double.  Per
// (a, b) the z-polynomial and its derivative come from one Horner pass over c; the sums over b and
// a use the power tables.  About 4 FMA per coefficient: FP64-pipe bound, 3.2 GB of coefficients
// read once at config 4.  The result is rounded to float32 once and written (or added) in input order.
#include "nf_common.cuh"

#define NFT_THREADS 64

struct TaylorArgs {
    const float *pos;
    const uint32_t *offsets, *perm;
    const double *T;
    float *acc;
    double scale, cellsz;
    int ncell, order, cml, accumulate;
};

// EXACT: the order equals PMAX, so every loop bound is a compile-time constant and the (p+1)(p+2)/2
// Horner chains of a particle are unrolled side by side (instruction-level parallelism for the FP64 pipe).
template <int PMAX, bool EXACT>
__global__ void __launch_bounds__(NFT_THREADS, 12) k_taylor(const TaylorArgs A) {
    extern __shared__ double sT[];
    const int p = EXACT ? PMAX : A.order;
    for (int cell = blockIdx.x; cell < A.ncell; cell += gridDim.x) {
        const uint32_t p0 = A.offsets[cell], p1 = A.offsets[cell + 1];
        if (p0 == p1) continue;
        __syncthreads();
        for (int i = threadIdx.x; i < A.cml; i += NFT_THREADS) sT[i] = A.T[(size_t)cell * A.cml + i];
        __syncthreads();
        for (uint32_t q = p0 + threadIdx.x; q < p1; q += NFT_THREADS) {
            const uint32_t pi = A.perm[q];
            const float *s = A.pos + 3ull * pi;
            const double tx = (double)s[0] * A.scale, ty = (double)s[1] * A.scale, tz = (double)s[2] * A.scale;
            const double X = (tx - floor(tx) - 0.5) * A.cellsz, Y = (ty - floor(ty) - 0.5) * A.cellsz, Z = (tz - floor(tz) - 0.5) * A.cellsz;
            double xp[PMAX + 1], yp[PMAX + 1];
            xp[0] = 1.0; yp[0] = 1.0;
#pragma unroll
            for (int k = 1; k <= PMAX; ++k) { xp[k] = xp[k - 1] * X; yp[k] = yp[k - 1] * Y; }
            double gx = 0.0, gy = 0.0, gz = 0.0;
            int idx = 0;
#pragma unroll
            for (int a = 0; a <= PMAX; ++a) {
                if (a > p) break;
                double s0 = 0.0, s1 = 0.0, sq = 0.0;      // sum_b P y^b, sum_b b P y^(b-1), sum_b Q y^b
#pragma unroll
                for (int b = 0; b <= PMAX - a; ++b) {
                    if (b > p - a) break;
                    const int nc = p - a - b + 1;
                    // Horner over c from the top: P = sum_c T z^c, Q = dP/dz
                    double P = 0.0, Q = 0.0;
#pragma unroll
                    for (int c = nc - 1; c >= 0; --c) {
                        Q = fma(Q, Z, P);
                        P = fma(P, Z, sT[idx + c]);
                    }
                    idx += nc;
                    s0 = fma(P, yp[b], s0);
                    if (b > 0) s1 = fma(P * (double)b, yp[b - 1], s1);
                    sq = fma(Q, yp[b], sq);
                }
                if (a > 0) gx = fma(s0 * (double)a, xp[a - 1], gx);
                gy = fma(s1, xp[a], gy);
                gz = fma(sq, xp[a], gz);
            }
            float *o = A.acc + 3ull * pi;
            if (A.accumulate) { o[0] += (float)(-gx); o[1] += (float)(-gy); o[2] += (float)(-gz); }
            else { o[0] = (float)(-gx); o[1] = (float)(-gy); o[2] = (float)(-gz); }
        }
    }
}

// ---- order 8 (the paper's choice): one thread per PADDED grid-order slot, everything unrolled ----
// A warp takes 32 consecutive slots whatever cells they belong to (1-3 cells at 64 per cell), so no
// lane idles but on the 2 % padding slots; each lane reads its own cell's coefficients straight from
// global memory through the read-only path -- lanes of one cell read the same address (one sector),
// and the cell's 1.3 KB stay in L1 for the warps that share it -- at compile-time offsets.  The
// polynomial is evaluated as a nested Horner scheme (z innermost, then y, then x) that carries the value
// and the three partial derivatives: 2 DFMA per coefficient + 3 per (a,b) + 4 per a = 501 DFMA per
// particle and nothing but those and the 165 loads in the instruction stream: FP64-pipe bound.
template <int P>
__global__ void __launch_bounds__(128) k_taylor_slots(const TaylorArgs A, const uint32_t *__restrict__ skey,
                                                      const uint32_t *__restrict__ perm_pad, const uint32_t *__restrict__ ctrl) {
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= ctrl[3]) return;                       // npad
    const uint32_t key = skey[s];
    if (key & NF_PAD_FLAG) return;
    const uint32_t pi = perm_pad[s];
    const float *q = A.pos + 3ull * pi;
    const double tx = (double)q[0] * A.scale, ty = (double)q[1] * A.scale, tz = (double)q[2] * A.scale;
    const double X = (tx - floor(tx) - 0.5) * A.cellsz, Y = (ty - floor(ty) - 0.5) * A.cellsz, Z = (tz - floor(tz) - 0.5) * A.cellsz;
    constexpr int CML = (P + 3) * (P + 2) * (P + 1) / 6;
    const double *__restrict__ T = A.T + (size_t)key * CML;
    // phi = sum_a x^a F_a(y,z), F_a = sum_b y^b P_ab(z): Horner from the top in every variable.
    // G = phi, Gx = dphi/dx, Gy, Gz accumulate over a; S, Sy, Sz over b; Pz, Qz (= dP/dz) over c.
    double G = 0.0, Gx = 0.0, Gy = 0.0, Gz = 0.0;
#pragma unroll
    for (int a = P; a >= 0; --a) {
        // first coefficient of this a in the basis order (a outer, b, c inner)
        int base_a = 0;
#pragma unroll
        for (int aa = 0; aa < a; ++aa) base_a += (P - aa + 1) * (P - aa + 2) / 2;
        double S = 0.0, Sy = 0.0, Sz = 0.0;
#pragma unroll
        for (int b = P - a; b >= 0; --b) {
            int base_b = base_a;
#pragma unroll
            for (int bb = 0; bb < b; ++bb) base_b += P - a - bb + 1;
            const int nc = P - a - b + 1;
            double Pz = 0.0, Qz = 0.0;
#pragma unroll
            for (int c = nc - 1; c >= 0; --c) {
                Qz = fma(Qz, Z, Pz);
                Pz = fma(Pz, Z, __ldg(T + base_b + c));
            }
            Sy = fma(Sy, Y, S);
            S = fma(S, Y, Pz);
            Sz = fma(Sz, Y, Qz);
        }
        Gx = fma(Gx, X, G);
        G = fma(G, X, S);
        Gy = fma(Gy, X, Sy);
        Gz = fma(Gz, X, Sz);
    }
    float *o = A.acc + 3ull * pi;
    if (A.accumulate) { o[0] += (float)(-Gx); o[1] += (float)(-Gy); o[2] += (float)(-Gz); }
    else { o[0] = (float)(-Gx); o[1] = (float)(-Gy); o[2] = (float)(-Gz); }
}

nf_status nf_run_taylor(nf_ctx *ctx, const float *d_pos, int order, const double *d_T, float *d_acc, int accumulate, cudaStream_t st) {
    TaylorArgs A;
    A.pos = d_pos; A.offsets = ctx->d_offsets; A.perm = ctx->d_perm_true; A.T = d_T; A.acc = d_acc;
    A.scale = ctx->prm.scale; A.cellsz = ctx->box / (double)ctx->cpd;
    A.ncell = (int)ctx->ncell; A.order = order; A.cml = (order + 3) * (order + 2) * (order + 1) / 6; A.accumulate = accumulate;
    const int64_t want = ctx->ncell;
    const int grid = (int)(want < (int64_t)ctx->sm_count * 2048 ? want : (int64_t)ctx->sm_count * 2048);
    const size_t smem = (size_t)A.cml * sizeof(double);
    if (order == 8) {
        const uint64_t bound = (uint64_t)ctx->lastN + (uint64_t)(NF_CELL_PAD - 1) * (uint64_t)ctx->ncell;     // >= npad, known on the host
        k_taylor_slots<8><<<(uint32_t)((bound + 127) / 128), 128, 0, st>>>(A, (const uint32_t *)(ctx->d_sorted + 3ull * ctx->capPad), ctx->d_perm_pad, ctx->d_ctrl);
    } else if (order < 8) k_taylor<8, false><<<grid, NFT_THREADS, smem, st>>>(A);
    else k_taylor<NF_MAX_MULTIPOLE_ORDER, false><<<grid, NFT_THREADS, smem, st>>>(A);
    ctx->launches++;
    NF_CUDA_OK(ctx, cudaGetLastError());
    return NF_OK;
}
