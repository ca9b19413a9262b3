// nf_pipeprobe.cu -- libnf_pipeprobe.so, a BENCH-ONLY helper (not part of the product's C ABI):
// pipe microbenchmarks that give bench.py the live roofline denominators of the device it runs on --
// FP32 FMA-pipe lane rate with scalar FFMA and with packed fma.rn.f32x2, MUFU.RSQ rate, and the
// FP64 DFMA lane rate (the bound of nf_multipoles / nf_taylor_accel).  DESIGN.md "Roofline" states
// how these relate to 148 SMs x 128 (FP32) / 64 (FP64) lanes x clock.
#include <cuda_runtime.h>

template <int MODE>
__global__ void __launch_bounds__(256) k_probe(float *out, int iters, float seed) {
    float a[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = seed + threadIdx.x * 1e-3f + i;
    const float b = seed * 0.5f + 1.0f, c = seed * 0.25f;
    const float2 bb = make_float2(b, b * 1.01f), cc = make_float2(c, c * 0.99f);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            if (MODE == 0) {
#pragma unroll
                for (int i = 0; i < 16; ++i) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[i]) : "f"(b), "f"(c));
            } else if (MODE == 1) {
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    float2 v = make_float2(a[2 * i], a[2 * i + 1]);
                    v = __ffma2_rn(v, bb, cc);
                    a[2 * i] = v.x; a[2 * i + 1] = v.y;
                }
            } else if (MODE == 2) {
#pragma unroll
                for (int i = 0; i < 16; ++i) asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(a[i]));
            }
        }
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += a[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// FP64: 16 independent DFMA chains per thread
__global__ void __launch_bounds__(256) k_probe_f64(float *out, int iters, double seed) {
    double a[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = seed + threadIdx.x * 1e-3 + i;
    const double b = seed * 0.5 + 1.0, c = seed * 0.25;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
#pragma unroll
            for (int i = 0; i < 16; ++i) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(a[i]) : "d"(b), "d"(c));
        }
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += a[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = (float)s;
}

template <int MODE>
static double probe_rate(float *d_out, int grid, int iters) {
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    if (MODE == 3) k_probe_f64<<<grid, 256>>>(d_out, 64, 1.0); else k_probe<MODE><<<grid, 256>>>(d_out, 64, 1.0f);
    float best = 1e30f;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(e0);
        if (MODE == 3) k_probe_f64<<<grid, 256>>>(d_out, iters, 1.0); else k_probe<MODE><<<grid, 256>>>(d_out, iters, 1.0f);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
        if (ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    return 64.0 * iters * (double)grid * 256.0 / (best * 1e-3);   // 64 lane-operations per thread per iteration
}

// h_out[0] FP32 FMA-pipe lane-operations per second, scalar FFMA stream
// h_out[1] the same for packed fma.rn.f32x2 (two lanes per thread-instruction)
// h_out[2] MUFU.RSQ lane-operations per second        h_out[3] SM count
// h_out[4] SM clock (MHz) reported by the runtime      h_out[5] FP64 DFMA lane-operations per second
// Runs on the current device, synchronises.  Returns 0, or 1 (bad argument), 2 (CUDA failure), 3 (no memory).
extern "C" int nfp_probe_pipes(double *h_out /* 6 */) {
    if (!h_out) return 1;
    int dev = 0;
    cudaDeviceProp p;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&p, dev) != cudaSuccess) { cudaGetLastError(); return 2; }
    const int grid = p.multiProcessorCount * 8;
    float *d_out = nullptr;
    if (cudaMalloc((void **)&d_out, (size_t)grid * 256 * 4) != cudaSuccess) { cudaGetLastError(); return 3; }
    h_out[0] = probe_rate<0>(d_out, grid, 8000);
    h_out[1] = probe_rate<1>(d_out, grid, 8000);
    h_out[2] = probe_rate<2>(d_out, grid, 1500);
    h_out[3] = p.multiProcessorCount;
    h_out[4] = p.clockRate / 1000.0;
    h_out[5] = probe_rate<3>(d_out, grid, 2000);
    cudaFree(d_out);
    return cudaGetLastError() == cudaSuccess ? 0 : 2;
}
