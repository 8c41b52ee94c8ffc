// g6_bench_probe.cu -- measurement aids of bench.py, built as their own library (libg6b200_probe.so); NOT part of
// libg6b200 and not on the path.  Three kinds of probe, all timed with CUDA events on the caller's stream:
//   g6p_fp32_rate   what the FP32 pipes of this chip sustain for register-sourced instruction streams that differ
//                   only in how many distinct register operands an instruction reads (the
//                   force kernel is bound by register-file operand bandwidth, not by the FMA pipe itself)
//   g6p_pair_rate   the PRODUCTION pair code (pair2 of g6_force_fast.cuh) in a loop over a shared-memory tile with
//                   no TMA, no fp64 work outside the tile fold -- and ablated copies of it in which the eleven
//                   three-operand FFMA2 read only two distinct register pairs (wrong numbers, same instruction mix)
//   g6p_read_pass   a kernel that only READS a buffer once: the floor of one small-n_i block step, which must make
//                   the same pass over the j-store (76 B per particle)
#include <cuda_runtime.h>

#include "../g6_force_fast.cuh"

using namespace g6;

namespace {

constexpr int NACC = 12;
constexpr int PROBE_THREADS = 128;

// independent accumulator chains, no memory traffic; MODE picks the operand pattern
//  0 scalar FFMA   acc = x * d[k] + acc         (x shared -> operand reuse cache; 2 fresh 32-bit reads)
//  1 scalar FFMA   three changing 32-bit sources
//  2 FFMA2         acc = acc * acc + d[k]       (2 distinct 64-bit register pairs)
//  3 FFMA2         acc = x * d[k] + acc         (x shared, reuse flag; 2 fresh pairs + 1 reused)
//  4 FFMA2         acc = d[k] * d[k+1] + acc    (3 distinct pairs)
//  5 FFMA2         acc = d[k] * dup(s[k]) + acc (2 pairs + one 32-bit broadcast operand)
//  6 FMUL2 acc*acc alternating with mode-4 FFMA2 (1 and 3 distinct pairs: averages to 2)
//  7 FADD2 / FMUL2 / FFMA2 in rotation, one changing source each
template <int MODE>
__global__ void __launch_bounds__(PROBE_THREADS) k_probe(float *out, int iters, float a, float b)
{
    float2 acc[NACC], d[NACC];
    float sc[NACC];
    const float2 x = make_float2(a + 1e-7f * threadIdx.x, a - 1e-7f * threadIdx.x), y = make_float2(b, 0.5f * b);
#pragma unroll
    for (int k = 0; k < NACC; ++k) {
        acc[k] = make_float2(0.1f * k, 0.2f * k);
        d[k] = make_float2(1e-3f * (k + threadIdx.x), 2e-3f * k + b);
        sc[k] = 1.0f + 1e-6f * (k + threadIdx.x);
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < NACC; ++k) {
            if (MODE == 0) { acc[k].x = __fmaf_rn(x.x, d[k].x, acc[k].x); acc[k].y = __fmaf_rn(x.y, d[k].y, acc[k].y); }
            if (MODE == 1) { acc[k].x = __fmaf_rn(acc[(k + 1) % NACC].x, acc[(k + 2) % NACC].y, acc[k].x); acc[k].y = __fmaf_rn(acc[(k + 1) % NACC].y, acc[(k + 3) % NACC].x, acc[k].y); }
            if (MODE == 2) acc[k] = __ffma2_rn(acc[k], acc[k], d[k]);
            if (MODE == 3) acc[k] = __ffma2_rn(x, d[k], acc[k]);
            if (MODE == 4) acc[k] = __ffma2_rn(d[k], d[(k + 1) % NACC], acc[k]);
            if (MODE == 5) acc[k] = __ffma2_rn(d[k], make_float2(sc[k], sc[k]), acc[k]);
            if (MODE == 6) { if (k & 1) acc[k] = __ffma2_rn(d[k], d[(k + 1) % NACC], acc[k]); else acc[k] = __fmul2_rn(acc[k], acc[k]); }
            if (MODE == 7) {
                if (k % 3 == 0) acc[k] = __fadd2_rn(acc[k], y);
                else if (k % 3 == 1) acc[k] = __fmul2_rn(acc[k], x);
                else acc[k] = __ffma2_rn(acc[k], x, y);
            }
        }
    }
    float s = 0.0f;
#pragma unroll
    for (int k = 0; k < NACC; ++k) s += acc[k].x + acc[k].y + d[k].x + sc[k];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// ---- the pair loop: AB = 0 is the production pair2<true> (double-single, Newton step); other values are ablations
//   1 pure-FP32 separations (production pair2<true, false>: 3 packed adds instead of 9 -- the cost of double-single)
//   2 the eleven three-operand FFMA2 (a, jerk, dx.dv) read two distinct register pairs  (numbers are wrong on purpose)
//   3 no nearest-neighbour tracking (the FMNMX3 reads three registers per two pairs)
template <int AB>
__device__ __forceinline__ void probe_pair2(IPart &I, const float2 xh, const float2 yh, const float2 zh, const float2 xl,
                                            const float2 yl, const float2 zl, const float2 vx, const float2 vy, const float2 vz,
                                            const float2 m, const float2 eps2_3, float2 &r2_out)
{
    if (AB != 2) {
        if (AB == 1) pair2<true, false>(I, xh, yh, zh, xl, yl, zl, vx, vy, vz, m, eps2_3, r2_out);
        else pair2<true, true>(I, xh, yh, zh, xl, yl, zl, vx, vy, vz, m, eps2_3, r2_out);
        return;
    }
    const float2 dx = add2(add2(xh, I.nxh[0]), add2(xl, I.nxl[0]));
    const float2 dy = add2(add2(yh, I.nxh[1]), add2(yl, I.nxl[1]));
    const float2 dz = add2(add2(zh, I.nxh[2]), add2(zl, I.nxl[2]));
    const float2 dvx = add2(vx, I.nv[0]), dvy = add2(vy, I.nv[1]), dvz = add2(vz, I.nv[2]);
    const float2 r2 = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));
    const float2 s2 = fma2(r2, dup(FOUR_THIRDS), eps2_3);
    float2 rinv = make_float2(rsqrt_approx(s2.x), rsqrt_approx(s2.y));
    const float2 u = fma2(make_float2(-s2.x, -s2.y), mul2(rinv, rinv), dup(3.0f));
    rinv = mul2(rinv, u);
    const float2 rinv2 = mul2(rinv, rinv), mrinv = mul2(m, rinv), mrinv3 = mul2(mrinv, rinv2);
    const float2 rv = add2(fma2(dz, dz, fma2(dy, dy, mul2(dx, dvx))), mul2(dvy, dvz));      // one instruction more (37 per pair evaluation), two-operand reads
    const float2 w = mul2(rv, rinv2);
    const float2 alpha = make_float2(-w.x, -w.y);
    I.p = add2(I.p, mrinv);
    I.a[0] = fma2(mrinv3, mrinv3, I.a[0]); I.a[1] = fma2(dy, dy, I.a[1]); I.a[2] = fma2(dz, dz, I.a[2]);
    const float2 tx = fma2(alpha, dx, dx), ty = fma2(alpha, dy, dy), tz = fma2(alpha, dz, dz);
    I.j[0] = fma2(tx, tx, I.j[0]); I.j[1] = fma2(ty, ty, I.j[1]); I.j[2] = fma2(tz, tz, I.j[2]);
    r2_out = r2;
}

template <int AB, int THREADS, int IT>
__global__ void __launch_bounds__(THREADS) k_pair_probe(const float *__restrict__ tile_g, float *__restrict__ out, int reps, float eps2f)
{
    __shared__ __align__(16) float tile[2][TILE_FLOATS];
    for (int k = threadIdx.x; k < 2 * TILE_FLOATS; k += THREADS) (&tile[0][0])[k] = tile_g[k];
    __syncthreads();
    IPart I[IT];
    double acc[IT][3], jrk[IT][3], pot[IT];
    int bstep[IT];
#pragma unroll
    for (int q = 0; q < IT; ++q) {
        const float f = 0.001f * (threadIdx.x + 128 * q + blockIdx.x);
        for (int k = 0; k < 3; ++k) {
            I[q].nxh[k] = dup(-(0.3f + f * (k + 1))); I[q].nxl[k] = dup(-1e-9f * f); I[q].nv[k] = dup(0.1f * f);
            acc[q][k] = 0; jrk[q][k] = 0;
        }
        pot[q] = 0; I[q].rmin = 1e30f; bstep[q] = -1;
    }
    const float2 eps2 = dup(FOUR_THIRDS * eps2f);
    for (int t = 0; t < reps; ++t) {
        const float4 *T = reinterpret_cast<const float4 *>(tile[t & 1]);
#pragma unroll
        for (int q = 0; q < IT; ++q) {
#pragma unroll
            for (int k = 0; k < 3; ++k) { I[q].a[k] = dup(0.0f); I[q].j[k] = dup(0.0f); }
            I[q].p = dup(0.0f);
        }
#pragma unroll 1
        for (int s8 = 0; s8 < JT / 8; ++s8) {
            float before[IT];
#pragma unroll
            for (int q = 0; q < IT; ++q) before[q] = I[q].rmin;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                float4 f[NF];
#pragma unroll
                for (int k = 0; k < NF; ++k) f[k] = T[k * (JT / 4) + 2 * s8 + h];
#pragma unroll
                for (int q = 0; q < IT; ++q) {
                    float2 ra, rb;
                    probe_pair2<AB>(I[q], make_float2(f[0].x, f[0].y), make_float2(f[1].x, f[1].y), make_float2(f[2].x, f[2].y),
                                    make_float2(f[3].x, f[3].y), make_float2(f[4].x, f[4].y), make_float2(f[5].x, f[5].y),
                                    make_float2(f[6].x, f[6].y), make_float2(f[7].x, f[7].y), make_float2(f[8].x, f[8].y),
                                    make_float2(f[9].x, f[9].y), eps2, ra);
                    probe_pair2<AB>(I[q], make_float2(f[0].z, f[0].w), make_float2(f[1].z, f[1].w), make_float2(f[2].z, f[2].w),
                                    make_float2(f[3].z, f[3].w), make_float2(f[4].z, f[4].w), make_float2(f[5].z, f[5].w),
                                    make_float2(f[6].z, f[6].w), make_float2(f[7].z, f[7].w), make_float2(f[8].z, f[8].w),
                                    make_float2(f[9].z, f[9].w), eps2, rb);
                    if (AB != 3) {
                        I[q].rmin = fminf(fminf(ra.x, ra.y), I[q].rmin);
                        I[q].rmin = fminf(fminf(rb.x, rb.y), I[q].rmin);
                    } else {
                        I[q].p = add2(I[q].p, mul2(ra, rb));      // keeps r2 alive: one FMUL2 + one FADD2 per two pair evaluations
                    }
                }
            }
            if (AB != 3) {
#pragma unroll
                for (int q = 0; q < IT; ++q) if (I[q].rmin < before[q]) bstep[q] = t * (JT / 8) + s8;
            }
        }
#pragma unroll
        for (int q = 0; q < IT; ++q) {
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                acc[q][k] += (double)I[q].a[k].x + (double)I[q].a[k].y;
                jrk[q][k] += (double)I[q].j[k].x + (double)I[q].j[k].y;
            }
            pot[q] -= (double)I[q].p.x + (double)I[q].p.y;
        }
    }
    double s = 0;
#pragma unroll
    for (int q = 0; q < IT; ++q) s += acc[q][0] + acc[q][1] + acc[q][2] + jrk[q][0] + jrk[q][1] + jrk[q][2] + pot[q] + I[q].rmin + bstep[q];
    out[blockIdx.x * THREADS + threadIdx.x] = (float)s;
}

__global__ void __launch_bounds__(256) k_read_pass(const float4 *__restrict__ p, size_t n16, float *out)
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

float *g_out = nullptr, *g_tile = nullptr;
int g_sm = 0;

int probe_init()
{
    if (g_out) return 0;
    cudaDeviceProp prop;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) return (int)e;
    g_sm = prop.multiProcessorCount;
    e = cudaMalloc((void **)&g_out, (size_t)g_sm * 16 * 256 * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc((void **)&g_tile, 2 * TILE_FLOATS * sizeof(float));
    if (e != cudaSuccess) return (int)e;
    // a synthetic tile: positions O(1), lo words ~1e-9, masses 1e-6
    static float h[2 * TILE_FLOATS];
    unsigned s = 12345u;
    for (int t = 0; t < 2; ++t)
        for (int k = 0; k < NF; ++k)
            for (int l = 0; l < JT; ++l) {
                s = s * 1664525u + 1013904223u;
                const float r = (float)(s >> 8) / 16777216.0f;
                h[t * TILE_FLOATS + k * JT + l] = (k >= F_XL && k < F_V) ? 1e-9f * r : (k == F_M ? 1e-6f : r);
            }
    return (int)cudaMemcpy(g_tile, h, sizeof(h), cudaMemcpyHostToDevice);
}

template <int MODE>
double fp32_rate_t(int ctas_per_sm, cudaStream_t st)
{
    const int grid = g_sm * ctas_per_sm, iters = 40000;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return -1.0;
    double best = 0.0;
    for (int rep = 0; rep < 3; ++rep) {                      // the first repetition also brings the clocks up
        cudaEventRecord(e0, st);
        k_probe<MODE><<<grid, PROBE_THREADS, 0, st>>>(g_out, iters, 1.0f, 1e-3f);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { best = -1.0; break; }
        float ms = 0.0f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double rate = (double)grid * PROBE_THREADS * (double)iters * NACC * 2.0 / (ms * 1e-3);
        if (rep > 0 && rate > best) best = rate;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return best;
}

template <int AB, int THREADS, int IT>
double pair_rate_t(cudaStream_t st)
{
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_pair_probe<AB, THREADS, IT>, THREADS, 0) != cudaSuccess || occ < 1) return -1.0;
    const int grid = g_sm * occ, reps = 600;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return -1.0;
    double best_ms = 1e30;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0, st);
        k_pair_probe<AB, THREADS, IT><<<grid, THREADS, 0, st>>>(g_tile, g_out, reps, 1e-8f);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { best_ms = -1.0; break; }
        float ms = 0.0f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best_ms) best_ms = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (best_ms <= 0) return -1.0;
    return (double)grid * THREADS * IT * (double)reps * JT / (best_ms * 1e-3);
}

}  // namespace

extern "C" {

// FP32 lane-instructions per second (an FMA counts once) of instruction stream `mode` (see k_probe), `ctas_per_sm` CTAs of
// 128 threads per SM (1 .. 16), on `cuda_stream` (a cudaStream_t cast to void*, NULL = default).  Returns 0 or a cudaError_t.
int g6p_fp32_rate(int mode, int ctas_per_sm, void *cuda_stream, double *lane_instr_per_s)
{
    if (mode < 0 || mode > 7 || ctas_per_sm < 1 || ctas_per_sm > 16 || !lane_instr_per_s) return (int)cudaErrorInvalidValue;
    int rc = probe_init();
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double r = -1.0;
    switch (mode) {
        case 0: r = fp32_rate_t<0>(ctas_per_sm, st); break;
        case 1: r = fp32_rate_t<1>(ctas_per_sm, st); break;
        case 2: r = fp32_rate_t<2>(ctas_per_sm, st); break;
        case 3: r = fp32_rate_t<3>(ctas_per_sm, st); break;
        case 4: r = fp32_rate_t<4>(ctas_per_sm, st); break;
        case 5: r = fp32_rate_t<5>(ctas_per_sm, st); break;
        case 6: r = fp32_rate_t<6>(ctas_per_sm, st); break;
        default: r = fp32_rate_t<7>(ctas_per_sm, st); break;
    }
    if (r < 0) return (int)cudaGetLastError();
    *lane_instr_per_s = r;
    return 0;
}

// pair evaluations (interactions) per second of the pair loop, variant `ab` (see probe_pair2), shape 0 = 128 threads x 2
// i-particles, 1 = 256 x 1; all resident CTAs of every SM.  Returns 0 or a cudaError_t.
int g6p_pair_rate(int ab, int shape, void *cuda_stream, double *interactions_per_s)
{
    if (ab < 0 || ab > 3 || shape < 0 || shape > 1 || !interactions_per_s) return (int)cudaErrorInvalidValue;
    int rc = probe_init();
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double r = -1.0;
    switch (ab * 2 + shape) {
        case 0: r = pair_rate_t<0, 128, 2>(st); break;
        case 1: r = pair_rate_t<0, 256, 1>(st); break;
        case 2: r = pair_rate_t<1, 128, 2>(st); break;
        case 3: r = pair_rate_t<1, 256, 1>(st); break;
        case 4: r = pair_rate_t<2, 128, 2>(st); break;
        case 5: r = pair_rate_t<2, 256, 1>(st); break;
        case 6: r = pair_rate_t<3, 128, 2>(st); break;
        default: r = pair_rate_t<3, 256, 1>(st); break;
    }
    if (r < 0) return (int)cudaGetLastError();
    *interactions_per_s = r;
    return 0;
}

// enqueue on `cuda_stream` a kernel that reads `bytes` (a multiple of 16) of device memory at `d_ptr` once
int g6p_read_pass(const void *d_ptr, unsigned long long bytes, void *cuda_stream)
{
    if (!d_ptr || bytes < 16) return (int)cudaErrorInvalidValue;
    int rc = probe_init();
    if (rc) return rc;
    k_read_pass<<<g_sm * 8, 256, 0, (cudaStream_t)cuda_stream>>>(reinterpret_cast<const float4 *>(d_ptr), (size_t)(bytes / 16), g_out);
    return (int)cudaGetLastError();
}

}  // extern "C"
