// nf_opbench.cu -- libnf_opbench.so, a BENCH-ONLY helper (not part of the product's C ABI, not in csrc/):
// the microbenchmarks behind DESIGN.md section 6 ("what actually bounds the loop").
//   (1) how long one warp-instruction holds a scheduler's pipe, by number of VARYING 64-bit register
//       operands, for packed f32x2 (FFMA2 / FADD2 / FMUL2), scalar FFMA and DFMA;
//   (2) a register-and-shared-memory replica of k_interact's trip loop (two sinks per thread, two
//       LDS.128 quads per plane and trip, 4 CTAs x 4 warps per SM) with the pair arithmetic all packed
//       (the kernel's), with the accumulates un-packed, and all scalar.
// Geometry everywhere: 4 CTAs of 128 threads per SM (the interaction kernel's occupancy).
#include <cuda_runtime.h>
#define NCH 8

template <int MODE>
__global__ void __launch_bounds__(128) k_ops(float *out, int iters, float seed) {
    float2 a[NCH], e[NCH], g[NCH];
#pragma unroll
    for (int i = 0; i < NCH; ++i) {
        a[i] = make_float2(seed + threadIdx.x * 1e-3f + i, seed - i);
        e[i] = make_float2(1.f + 1e-6f * i + 1e-8f * threadIdx.x, 1.f - 1e-6f * i);
        g[i] = make_float2(1e-7f * i + seed * 1e-9f, -1e-7f * i + 1e-9f * threadIdx.x);
    }
    const float2 b = make_float2(seed * 0.5f + 0.5f, seed * 0.51f + 0.49f), c = make_float2(seed * 1e-8f, seed * 1.1e-8f);
    const float sb = seed * 0.999f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 2; ++r)
#pragma unroll
            for (int i = 0; i < NCH; ++i) {
                if (MODE == 0) a[i] = __ffma2_rn(a[i], b, c);                       // FFMA2, 1 varying
                if (MODE == 1) a[i] = __ffma2_rn(a[i], e[i], c);                    // FFMA2, 2 varying
                if (MODE == 2) a[i] = __ffma2_rn(e[i], g[i], a[i]);                 // FFMA2, 3 varying (accumulate form)
                if (MODE == 3) a[i] = __fadd2_rn(a[i], make_float2(sb, sb));        // FADD2, 1 varying + broadcast scalar
                if (MODE == 4) a[i] = __fadd2_rn(a[i], e[i]);                       // FADD2, 2 varying
                if (MODE == 5) a[i] = __fmul2_rn(a[i], a[i]);                       // FMUL2, 1 varying
                if (MODE == 6) a[i] = __fmul2_rn(a[i], e[i]);                       // FMUL2, 2 varying
                if (MODE == 7) { a[i].x = __fmaf_rn(e[i].x, g[i].x, a[i].x); a[i].y = __fmaf_rn(e[i].y, g[i].y, a[i].y); }   // 2 scalar FFMA, 3 varying
            }
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < NCH; ++i) s += a[i].x + a[i].y + e[i].x + g[i].y;
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <int MODE>
__global__ void __launch_bounds__(128) k_ops64(float *out, int iters, double seed) {
    double a[NCH], e[NCH], g[NCH];
#pragma unroll
    for (int i = 0; i < NCH; ++i) { a[i] = seed + threadIdx.x * 1e-3 + i; e[i] = 1.0 + 1e-9 * i + 1e-12 * threadIdx.x; g[i] = 1e-9 * i + 1e-12 * threadIdx.x; }
    const double b = seed * 0.5 + 0.5, c = seed * 1e-9;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 2; ++r)
#pragma unroll
            for (int i = 0; i < NCH; ++i) {
                if (MODE == 0) a[i] = fma(a[i], b, c);          // DFMA, 1 varying
                if (MODE == 1) a[i] = fma(b, g[i], a[i]);       // DFMA, 2 varying (accumulate with a reused multiplicand: the multipoles' form)
                if (MODE == 2) a[i] = fma(e[i], g[i], a[i]);    // DFMA, 3 varying
            }
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < NCH; ++i) s += a[i] + e[i] + g[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = (float)s;
}

__device__ __forceinline__ float rsq(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
template <int V>
__device__ __forceinline__ void pair2(const float2 X, const float2 Y, const float2 Z, const float nx, const float ny, const float nz,
                                      float2 &ax, float2 &ay, float2 &az) {
    const float2 tau = make_float2(1e-30f, 1e-30f);
    if (V == 0 || V == 1) {
        const float2 dx = __fadd2_rn(X, make_float2(nx, nx)), dy = __fadd2_rn(Y, make_float2(ny, ny)), dz = __fadd2_rn(Z, make_float2(nz, nz));
        float2 r2 = __ffma2_rn(dx, dx, tau); r2 = __ffma2_rn(dy, dy, r2); r2 = __ffma2_rn(dz, dz, r2);
        const float2 ri = make_float2(rsq(r2.x), rsq(r2.y));
        const float2 f = __fmul2_rn(__fmul2_rn(ri, ri), ri);
        if (V == 0) { ax = __ffma2_rn(f, dx, ax); ay = __ffma2_rn(f, dy, ay); az = __ffma2_rn(f, dz, az); }
        else {
            ax.x = __fmaf_rn(f.x, dx.x, ax.x); ax.y = __fmaf_rn(f.y, dx.y, ax.y);
            ay.x = __fmaf_rn(f.x, dy.x, ay.x); ay.y = __fmaf_rn(f.y, dy.y, ay.y);
            az.x = __fmaf_rn(f.x, dz.x, az.x); az.y = __fmaf_rn(f.y, dz.y, az.y);
        }
    } else {
        const float dx0 = X.x + nx, dx1 = X.y + nx, dy0 = Y.x + ny, dy1 = Y.y + ny, dz0 = Z.x + nz, dz1 = Z.y + nz;
        float r0 = __fmaf_rn(dx0, dx0, 1e-30f), r1 = __fmaf_rn(dx1, dx1, 1e-30f);
        r0 = __fmaf_rn(dy0, dy0, r0); r1 = __fmaf_rn(dy1, dy1, r1); r0 = __fmaf_rn(dz0, dz0, r0); r1 = __fmaf_rn(dz1, dz1, r1);
        const float i0 = rsq(r0), i1 = rsq(r1);
        const float f0 = i0 * i0 * i0, f1 = i1 * i1 * i1;
        ax.x = __fmaf_rn(f0, dx0, ax.x); ax.y = __fmaf_rn(f1, dx1, ax.y);
        ay.x = __fmaf_rn(f0, dy0, ay.x); ay.y = __fmaf_rn(f1, dy1, ay.y);
        az.x = __fmaf_rn(f0, dz0, az.x); az.y = __fmaf_rn(f1, dz1, az.y);
    }
}
template <int V>
__global__ void __launch_bounds__(128, 4) k_trips(float *out, int ntrips, int reps, float seed) {
    extern __shared__ __align__(16) float sm[];       // xs | ys | zs, 640 slots each (one stage of the kernel's ring)
    float *xs = sm, *ys = sm + 640, *zs = sm + 1280;
    for (int i = threadIdx.x; i < 640; i += 128) { xs[i] = seed * 1e-3f * i; ys[i] = 0.3f + seed * 2e-3f * i; zs[i] = -0.2f + 1e-3f * i; }
    __syncthreads();
    float nx[2], ny[2], nz[2];
    float2 ax[2], ay[2], az[2];
    for (int j = 0; j < 2; ++j) { nx[j] = -(3.f + threadIdx.x * 1e-2f + j); ny[j] = -(2.f + j * 0.1f); nz[j] = -1.f - threadIdx.x * 1e-3f; ax[j] = ay[j] = az[j] = make_float2(0.f, 0.f); }
    for (int r = 0; r < reps; ++r) {
        const int lo = (r * 8) & 63;
        for (int trip = 0; trip < ntrips; ++trip) {
            const int t = lo + trip * 8;
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                const float4 X = *reinterpret_cast<const float4 *>(xs + t + 4 * q);
                const float4 Y = *reinterpret_cast<const float4 *>(ys + t + 4 * q);
                const float4 Z = *reinterpret_cast<const float4 *>(zs + t + 4 * q);
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    pair2<V>(make_float2(X.x, X.y), make_float2(Y.x, Y.y), make_float2(Z.x, Z.y), nx[j], ny[j], nz[j], ax[j], ay[j], az[j]);
                    pair2<V>(make_float2(X.z, X.w), make_float2(Y.z, Y.w), make_float2(Z.z, Z.w), nx[j], ny[j], nz[j], ax[j], ay[j], az[j]);
                }
            }
        }
    }
    float s = 0;
    for (int j = 0; j < 2; ++j) s += ax[j].x + ax[j].y + ay[j].x + ay[j].y + az[j].x + az[j].y;
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

static const size_t kSmem = 52 * 1024;      // as much as a CTA of the interaction kernel holds: 4 CTAs per SM
template <typename K, typename... Args>
static double time_ms(K kern, int grid, size_t smem, Args... args) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    for (int r = 0; r < 4; ++r) {
        cudaEventRecord(e0); kern<<<grid, 128, smem>>>(args...); cudaEventRecord(e1); cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    return best;
}

// h_out[0..7]  cycles per warp-instruction per scheduler: FFMA2 with 1 / 2 / 3 varying 64-bit register operands, FADD2 1 / 2,
//              FMUL2 1 / 2, scalar FFMA (3 varying)
// h_out[8..10] DFMA with 1 / 2 / 3 varying operands
// h_out[11..13] cycles per trip (16 pairs per lane-pair... 8 sources x 2 sinks) of the trip-loop replica: all packed, accumulates scalar, all scalar
// h_out[14..16] the same as pairs per second on the whole device
// clock_mhz: the SM clock to convert times into cycles (MEASURED_PEAKS.json: sm_max_mhz).  Returns 0, 1 (bad argument), 2 (CUDA failure).
extern "C" int nfo_opbench(double clock_mhz, double *h_out /* 17 */) {
    if (!h_out || !(clock_mhz > 0)) return 1;
    int dev = 0; cudaDeviceProp p;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&p, dev) != cudaSuccess) { cudaGetLastError(); return 2; }
    const int nsm = p.multiProcessorCount, grid = nsm * 4, iters = 4000;
    float *d = nullptr;
    if (cudaMalloc(&d, (size_t)grid * 128 * 4) != cudaSuccess) { cudaGetLastError(); return 2; }
    const double clk = clock_mhz * 1e6;
    auto cyc = [&](double ms, double instr_per_thread_iter) { return ms * 1e-3 * clk * nsm * 4 / ((double)iters * 2 * NCH * instr_per_thread_iter * grid * 4.0); };
    h_out[0] = cyc(time_ms(k_ops<0>, grid, kSmem, d, iters, 1.f), 1); h_out[1] = cyc(time_ms(k_ops<1>, grid, kSmem, d, iters, 1.f), 1);
    h_out[2] = cyc(time_ms(k_ops<2>, grid, kSmem, d, iters, 1.f), 1); h_out[3] = cyc(time_ms(k_ops<3>, grid, kSmem, d, iters, 1.f), 1);
    h_out[4] = cyc(time_ms(k_ops<4>, grid, kSmem, d, iters, 1.f), 1); h_out[5] = cyc(time_ms(k_ops<5>, grid, kSmem, d, iters, 1.f), 1);
    h_out[6] = cyc(time_ms(k_ops<6>, grid, kSmem, d, iters, 1.f), 1); h_out[7] = cyc(time_ms(k_ops<7>, grid, kSmem, d, iters, 1.f), 2);
    h_out[8] = cyc(time_ms(k_ops64<0>, grid, kSmem, d, iters, 1.0), 1); h_out[9] = cyc(time_ms(k_ops64<1>, grid, kSmem, d, iters, 1.0), 1);
    h_out[10] = cyc(time_ms(k_ops64<2>, grid, kSmem, d, iters, 1.0), 1);
    const int ntrips = 64, reps = 300;
    const double trips = (double)ntrips * reps * grid * 4.0;
    const double t0 = time_ms(k_trips<0>, grid, kSmem, d, ntrips, reps, 1.f), t1 = time_ms(k_trips<1>, grid, kSmem, d, ntrips, reps, 1.f),
                 t2 = time_ms(k_trips<2>, grid, kSmem, d, ntrips, reps, 1.f);
    const double tt[3] = {t0, t1, t2};
    for (int v = 0; v < 3; ++v) { h_out[11 + v] = tt[v] * 1e-3 * clk * nsm * 4 / trips; h_out[14 + v] = trips * 16 * 32 / (tt[v] * 1e-3); }
    cudaFree(d);
    return cudaGetLastError() == cudaSuccess ? 0 : 2;
}
