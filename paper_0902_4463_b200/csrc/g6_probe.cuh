// g6_probe.cuh -- a measurement aid, not part of the path: what the FP32 pipes of this chip sustain
// for register-sourced instructions, so that the force kernel's roofline fraction (DESIGN.md
// section 6) can be read against a MEASURED issue ceiling beside the nominal
// SMs x 128 lanes x clock.  Independent accumulator chains, no memory traffic.
//   mode 0  scalar FFMA   acc = acc * x + y          (x, y loop constants)
//   mode 1  packed FFMA2  acc = acc * x + y          (x, y loop constants: two reusable operands)
//   mode 2  FADD2 / FMUL2 / FFMA2 in turn            (the instruction kinds of the pair kernel)
//   mode 3  packed FFMA2 with three distinct, changing source registers
#pragma once
#include <cuda_runtime.h>

namespace g6 {

constexpr int PROBE_NACC = 12;
constexpr int PROBE_THREADS = 128;

template <int MODE>
__global__ void __launch_bounds__(PROBE_THREADS)
k_probe_fp32(float *out, int iters, float a, float b)
{
    float2 acc[PROBE_NACC];
    const float2 x = make_float2(a + 1e-7f * threadIdx.x, a - 1e-7f * threadIdx.x), y = make_float2(b, 0.5f * b);
#pragma unroll
    for (int k = 0; k < PROBE_NACC; ++k) acc[k] = make_float2(0.1f * k, 0.2f * k);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < PROBE_NACC; ++k) {
            if (MODE == 0) { acc[k].x = __fmaf_rn(acc[k].x, x.x, y.x); acc[k].y = __fmaf_rn(acc[k].y, x.y, y.y); }
            if (MODE == 1) acc[k] = __ffma2_rn(acc[k], x, y);
            if (MODE == 2) {
                if (k % 3 == 0) acc[k] = __fadd2_rn(acc[k], y);
                else if (k % 3 == 1) acc[k] = __fmul2_rn(acc[k], x);
                else acc[k] = __ffma2_rn(acc[k], x, y);
            }
            if (MODE == 3) acc[k] = __ffma2_rn(acc[(k + 1) % PROBE_NACC], acc[(k + 2) % PROBE_NACC], acc[k]);
        }
    }
    float s = 0.0f;
#pragma unroll
    for (int k = 0; k < PROBE_NACC; ++k) s += acc[k].x + acc[k].y;
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// FP32 lane-instructions per second (an FMA counts once) sustained by `mode`; < 0: a CUDA error code
inline double probe_fp32(int mode, int n_sm, cudaStream_t st, float *d_out, int ctas_per_sm)
{
    const int grid = n_sm * ctas_per_sm, iters = 60000;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return -1.0;
    double best = 0.0;
    for (int rep = 0; rep < 3; ++rep) {          // the first repetition also brings the clocks up
        cudaEventRecord(e0, st);
        switch (mode) {
            case 0: k_probe_fp32<0><<<grid, PROBE_THREADS, 0, st>>>(d_out, iters, 1.0f, 1e-3f); break;
            case 1: k_probe_fp32<1><<<grid, PROBE_THREADS, 0, st>>>(d_out, iters, 1.0f, 1e-3f); break;
            case 2: k_probe_fp32<2><<<grid, PROBE_THREADS, 0, st>>>(d_out, iters, 1.0f, 1e-3f); break;
            default: k_probe_fp32<3><<<grid, PROBE_THREADS, 0, st>>>(d_out, iters, 1.0f, 1e-3f); break;
        }
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { best = -1.0; break; }
        float ms = 0.0f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double rate = (double)grid * PROBE_THREADS * (double)iters * PROBE_NACC * 2.0 / (ms * 1e-3);
        if (rep > 0 && rate > best) best = rate;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return best;
}

// the cheapest possible pass over `n16` 16-byte words: what a kernel that only READS the j-store costs
__global__ void __launch_bounds__(256)
k_probe_read(const float4 *__restrict__ p, size_t n16, float *out)
{
    float s = 0.0f;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t st = (size_t)gridDim.x * blockDim.x;
    for (; i + 3 * st < n16; i += 4 * st) {
        const float4 a = __ldcs(p + i), b = __ldcs(p + i + st), c = __ldcs(p + i + 2 * st), d = __ldcs(p + i + 3 * st);
        s += a.x + b.y + c.z + d.w;
    }
    for (; i < n16; i += st) s += __ldcs(p + i).x;
    if (s == 123.456f) out[0] = s;          // keeps the loads alive
}

}  // namespace g6
