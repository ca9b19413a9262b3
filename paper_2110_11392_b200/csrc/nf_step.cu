// nf_step.cu -- the pipeline steps either side of NearForce that touch every particle once:
// Kick and Drift of the KDK leapfrog (sec. 3.1; Table 1) and the
// particle part of the time-step criterion, Eq. 1.  HBM-bound elementwise /
// per-cell reductions; no tensor cores, no shared-memory staging needed.
#include "nf_common.cuh"

// v <- v + a dt_kick ; x <- x + v_new dt_drift wrapped into [0, box).  Each update in double from the
// float32 state, product and sum rounded separately (no FMA), rounded to float32 once
// (readings K1-K3) -- the same arithmetic as the oracle, bit for bit.
__global__ void __launch_bounds__(256) k_kick_drift(float *__restrict__ pos, float *__restrict__ vel, const float *__restrict__ acc,
                                                    uint64_t n3, double dt_kick, double dt_drift, double box) {
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    const float fbox = (float)box;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n3; i += stride) {
        const float v = (float)__dadd_rn((double)vel[i], __dmul_rn((double)acc[i], dt_kick));
        vel[i] = v;
        double x = __dadd_rn((double)pos[i], __dmul_rn((double)v, dt_drift));
        const double k = floor(__ddiv_rn(x, box));
        x = __dadd_rn(x, -__dmul_rn(k, box));
        if (x < 0.0) x = 0.0;
        float xf = (float)x;
        if (!(xf < fbox)) xf = 0.0f;
        pos[i] = xf;
    }
}

nf_status nf_run_kick_drift(nf_ctx *ctx, float *d_pos, float *d_vel, const float *d_acc, int64_t N, double dt_kick, double dt_drift,
                            cudaStream_t st) {
    const uint64_t n3 = 3ull * (uint64_t)N;
    const int grid = ctx->sm_count * 16;
    k_kick_drift<<<grid, 256, 0, st>>>(d_pos, d_vel, d_acc, n3, dt_kick, dt_drift, ctx->box); ctx->launches++;
    NF_CUDA_OK(ctx, cudaGetLastError());
    return NF_OK;
}

// ---- Eq. 1: per-cell v_rms / a_max, one warp per cell over the grid-order permutation ------------
__device__ __forceinline__ void atomic_min_pos_double(double *addr, double v) {   // v >= 0: bit patterns order like the values
    atomicMin((unsigned long long *)addr, (unsigned long long)__double_as_longlong(v));
}
__device__ __forceinline__ void atomic_max_pos_double(double *addr, double v) {
    atomicMax((unsigned long long *)addr, (unsigned long long)__double_as_longlong(v));
}

// out[0] = min over cells of v_rms/a_max (as bits, initialised to +inf), out[1] = sum |v|^2, out[2] = max |a|^2
__global__ void __launch_bounds__(256) k_cell_ratio(int ncell, const uint32_t *__restrict__ offsets, const uint32_t *__restrict__ perm,
                                                    const float *__restrict__ vel, const float *__restrict__ acc, double *__restrict__ out) {
    const int lane = threadIdx.x & 31;
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarp = (gridDim.x * blockDim.x) >> 5;
    double gv2 = 0.0, ga2 = 0.0, best = __longlong_as_double(0x7ff0000000000000ll);
    for (int c = warp; c < ncell; c += nwarp) {
        const uint32_t p0 = offsets[c], p1 = offsets[c + 1];
        if (p0 == p1) continue;
        double v2 = 0.0, a2 = 0.0;
        for (uint32_t p = p0 + lane; p < p1; p += 32) {
            const size_t i = 3ull * perm[p];
            const double vx = vel[i], vy = vel[i + 1], vz = vel[i + 2], ax = acc[i], ay = acc[i + 1], az = acc[i + 2];
            v2 += vx * vx + vy * vy + vz * vz;
            a2 = fmax(a2, ax * ax + ay * ay + az * az);
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) { v2 += __shfl_xor_sync(0xffffffffu, v2, d); a2 = fmax(a2, __shfl_xor_sync(0xffffffffu, a2, d)); }
        gv2 += v2;                       // the same on every lane
        ga2 = fmax(ga2, a2);
        if (a2 > 0.0) best = fmin(best, sqrt(v2 / (double)(p1 - p0)) / sqrt(a2));
    }
    if (lane == 0) {
        atomic_min_pos_double(&out[0], best);
        if (gv2 > 0.0) atomicAdd(&out[1], gv2);
        atomic_max_pos_double(&out[2], ga2);
    }
}

nf_status nf_run_timestep_ratio(nf_ctx *ctx, const float *d_vel, const float *d_acc, double *d_out3, cudaStream_t st) {
    const double init[3] = {__builtin_inf(), 0.0, 0.0};
    NF_CUDA_OK(ctx, cudaMemcpyAsync(d_out3, init, sizeof init, cudaMemcpyHostToDevice, st));
    const int grid = ctx->sm_count * 8;
    k_cell_ratio<<<grid, 256, 0, st>>>((int)ctx->ncell, ctx->d_offsets, ctx->d_perm_true, d_vel, d_acc, d_out3); ctx->launches++;
    NF_CUDA_OK(ctx, cudaGetLastError());
    return NF_OK;
}
