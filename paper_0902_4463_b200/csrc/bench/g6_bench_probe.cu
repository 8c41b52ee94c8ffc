// g6_bench_probe.cu -- measurement aids of bench.py, built as their own library (libg6b200_probe.so); NOT part of
// libg6b200 and not on the path.  Three kinds of probe, all timed with CUDA events on the caller's stream:
//   g6p_fp32_rate   what the FP32 pipes of this chip sustain for register-sourced instruction streams that differ
//                   only in how many distinct register operands an instruction reads (the
//                   force kernel is bound by register-file operand bandwidth, not by the FMA pipe itself)
//   g6p_pair_rate   the PRODUCTION pair code (pair2 of g6_force_fast.cuh) in a loop over a shared-memory tile with
//                   no TMA, no fp64 work outside the tile fold -- and ablated copies of it in which the eleven
//                   three-operand FFMA2 read only two distinct register pairs (wrong numbers, same instruction mix)
//   g6p_mix_cycles  what ONE non-FMA instruction costs next to a saturated stream of two-operand FFMA2 (LDS, MOV, IADD, LOP, FMNMX,
//                   FMNMX3, VIMNMX3, scalar FFMA, MUFU.RSQ): cycles per 12 FFMA2 of a stream with k extra instructions
//   g6p_operand_rate packed FFMA2 / FADD2 whose third / second operand is a 32-bit broadcast register, a reused pair, or a
//                   UNIFORM-register pair (kernel parameter -> LDCU -> UR): which operand forms cost no vector-register read
//   g6p_pair_rate_cbank  the production pair loop with the j-tile in the CONSTANT BANK (operands = uniform-register pairs, no
//                   shared memory at all): the prototype that showed the pipe stays throttled wherever the j operands come from
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

// ---- a saturated stream of two-operand FFMA2 (12 chains) plus `extra` instructions of one kind per 12:
//  0 none | 1 LDS | 2 MOV imm | 3 IADD | 4 LOP3 (two register reads) | 5 FMNMX (two reads) | 6 FMNMX3 | 7 VIMNMX3 | 8 scalar FFMA | 9 MUFU.RSQ
template <int KIND, int EXTRA>
__global__ void __launch_bounds__(PROBE_THREADS) k_mix(float *out, int iters, float a, float b)
{
    __shared__ float sh[1024];
    for (int i = threadIdx.x; i < 1024; i += PROBE_THREADS) sh[i] = a * i;
    __syncthreads();
    const unsigned shbase = (unsigned)__cvta_generic_to_shared(sh);
    float2 acc[NACC], d[NACC];
    int x[NACC];
    float f[NACC];
#pragma unroll
    for (int k = 0; k < NACC; ++k) {
        acc[k] = make_float2(0.1f * k + a, 0.2f * k);
        d[k] = make_float2(1e-3f * (k + threadIdx.x) + a, 2e-3f * k + b);
        x[k] = threadIdx.x + k;
        f[k] = 1.0f + k * a;
    }
    constexpr int EVERY = EXTRA > 0 ? NACC / EXTRA : NACC + 1;
#pragma unroll 4
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < NACC; ++k) {
            acc[k] = __ffma2_rn(acc[k], acc[k], d[k]);
            if (EXTRA > 0 && k % EVERY == 0) {
                if (KIND == 1) { float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(shbase + (unsigned)((it * NACC + k) & 1023) * 4)); f[k] = v; }
                if (KIND == 2) asm volatile("mov.b32 %0, %1;" : "=r"(x[k]) : "n"(12345));
                if (KIND == 3) asm volatile("add.s32 %0, %0, 3;" : "+r"(x[k]));
                if (KIND == 4) asm volatile("xor.b32 %0, %0, %1;" : "+r"(x[k]) : "r"(x[(k + 1) % NACC]));
                if (KIND == 5) asm volatile("min.f32 %0, %0, %1;" : "+f"(f[k]) : "f"(acc[k].x));
                if (KIND == 6) f[k] = fminf(fminf(acc[k].x, acc[k].y), f[k]);
                if (KIND == 7) x[k] = __vimin3_s32(x[k], __float_as_int(acc[k].x), __float_as_int(acc[k].y));
                if (KIND == 8) asm volatile("fma.rn.f32 %0, %0, %0, %1;" : "+f"(f[k]) : "f"(a));
                if (KIND == 9) f[k] = rsqrt_approx(f[k]);
            }
        }
    }
    float r = 0.0f;
#pragma unroll
    for (int k = 0; k < NACC; ++k) r += acc[k].x + acc[k].y + d[k].x + x[k] + f[k];
    out[blockIdx.x * blockDim.x + threadIdx.x] = r;
}

// ---- operand forms: four accumulators share the operand d[k] / sc[k] / P.c[k] for four consecutive instructions
//  0 FFMA2 acc, x, PAIR (shared vector pair, .reuse)   1 FFMA2 acc, x, UR pair   2 FFMA2 acc, x, 32-bit broadcast
//  3 FADD2 acc, PAIR                                   4 FADD2 acc, UR pair      5 FFMA2 three distinct vector pairs
struct ProbeParams { float2 c[NACC]; };
template <int MODE>
__global__ void __launch_bounds__(PROBE_THREADS) k_operand(float *out, int iters, float a, float b, const __grid_constant__ ProbeParams P)
{
    float2 acc[4], x[4], d[NACC], e[NACC];
    float sc[NACC];
#pragma unroll
    for (int q = 0; q < 4; ++q) { acc[q] = make_float2(0.1f * q + a, threadIdx.x); x[q] = make_float2(1.0f + 1e-7f * threadIdx.x * (q + 1), 1.0f - 1e-7f * q * b); }
#pragma unroll
    for (int k = 0; k < NACC; ++k) { d[k] = make_float2(1e-3f * (k + threadIdx.x) + a, 2e-3f * k + b); e[k] = make_float2(d[k].y, d[k].x + 1.f); sc[k] = 1e-3f * k + b * threadIdx.x; }
#pragma unroll 4
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < NACC; ++k) {
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                if (MODE == 0) acc[q] = __ffma2_rn(acc[q], x[q], d[k]);
                if (MODE == 1) acc[q] = __ffma2_rn(acc[q], x[q], P.c[k]);
                if (MODE == 2) acc[q] = __ffma2_rn(acc[q], x[q], make_float2(sc[k], sc[k]));
                if (MODE == 3) acc[q] = __fadd2_rn(acc[q], d[k]);
                if (MODE == 4) acc[q] = __fadd2_rn(acc[q], P.c[k]);
                if (MODE == 5) acc[q] = __ffma2_rn(d[(k + q) % NACC], e[(k + 2 * q + 1) % NACC], acc[q]);
            }
        }
    }
    float r = 0.0f;
#pragma unroll
    for (int q = 0; q < 4; ++q) r += acc[q].x + acc[q].y + x[q].x;
#pragma unroll
    for (int k = 0; k < NACC; ++k) r += d[k].x + e[k].y + sc[k];
    out[blockIdx.x * blockDim.x + threadIdx.x] = r;
}

// ---- the production pair loop with the j-tiles in the constant bank: j operands reach the packed instructions as uniform-register
// pairs (LDCU.64), the i operands as 32-bit broadcast registers; no shared memory, no LDS
constexpr int CB_TILES = 6;                                   // 6 x 256 j = 60 KiB of the 64 KiB bank
__constant__ float4 c_tiles[CB_TILES * NF * (JT / 4)];

template <int THREADS, int IT>
__global__ void __launch_bounds__(THREADS) k_pair_cbank(float *out, int reps, float eps2f)
{
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
    for (int r = 0; r < reps; ++r) {
#pragma unroll 1
        for (int t = 0; t < CB_TILES; ++t) {
#pragma unroll
            for (int q = 0; q < IT; ++q) {
#pragma unroll
                for (int k = 0; k < 3; ++k) { I[q].a[k] = dup(0.0f); I[q].j[k] = dup(0.0f); }
                I[q].p = dup(0.0f);
            }
            const float4 *T = c_tiles + t * NF * (JT / 4);
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
                        pair2<true>(I[q], make_float2(f[0].x, f[0].y), make_float2(f[1].x, f[1].y), make_float2(f[2].x, f[2].y),
                                    make_float2(f[3].x, f[3].y), make_float2(f[4].x, f[4].y), make_float2(f[5].x, f[5].y),
                                    make_float2(f[6].x, f[6].y), make_float2(f[7].x, f[7].y), make_float2(f[8].x, f[8].y),
                                    make_float2(f[9].x, f[9].y), eps2, ra);
                        pair2<true>(I[q], make_float2(f[0].z, f[0].w), make_float2(f[1].z, f[1].w), make_float2(f[2].z, f[2].w),
                                    make_float2(f[3].z, f[3].w), make_float2(f[4].z, f[4].w), make_float2(f[5].z, f[5].w),
                                    make_float2(f[6].z, f[6].w), make_float2(f[7].z, f[7].w), make_float2(f[8].z, f[8].w),
                                    make_float2(f[9].z, f[9].w), eps2, rb);
                        I[q].rmin = fminf(fminf(ra.x, ra.y), I[q].rmin);
                        I[q].rmin = fminf(fminf(rb.x, rb.y), I[q].rmin);
                    }
                }
#pragma unroll
                for (int q = 0; q < IT; ++q) if (I[q].rmin < before[q]) bstep[q] = t * (JT / 8) + s8;
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
    }
    double s = 0;
#pragma unroll
    for (int q = 0; q < IT; ++q) s += acc[q][0] + acc[q][1] + acc[q][2] + jrk[q][0] + jrk[q][1] + jrk[q][2] + pot[q] + bstep[q] + I[q].rmin;
    out[(size_t)blockIdx.x * THREADS + threadIdx.x] = (float)s;
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

template <typename Launch>
double time_best_ms(cudaStream_t st, int reps, Launch launch)
{
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return -1.0;
    double best_ms = 1e30;
    for (int rep = 0; rep < reps; ++rep) {
        cudaEventRecord(e0, st);
        launch();
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { best_ms = -1.0; break; }
        float ms = 0.0f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best_ms) best_ms = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return best_ms;
}

// cycles (at `sm_hz`) per 12 FFMA2 of the mixed stream, best of 2 / 4 / 8 CTAs per SM
template <int KIND, int EXTRA>
double mix_cycles_t(cudaStream_t st, double sm_hz)
{
    const int iters = 100000;
    double best = 1e30;
    for (int c : {2, 4, 8}) {
        const int grid = g_sm * c;
        const double ms = time_best_ms(st, 3, [&] { k_mix<KIND, EXTRA><<<grid, PROBE_THREADS, 0, st>>>(g_out, iters, 0.5f, 0.25f); });
        if (ms <= 0) return -1.0;
        // one sub-partition issues for grid * warps / (SMs * 4) warps; a 12-FFMA2 group is 24 pipe cycles at full rate
        const double warps_per_smsp = (double)c * (PROBE_THREADS / 32) / 4.0;
        const double cyc = ms * 1e-3 * sm_hz / ((double)iters * warps_per_smsp);
        if (cyc < best) best = cyc;
    }
    return best;
}

template <int MODE>
double operand_rate_t(cudaStream_t st)
{
    ProbeParams P;
    for (int k = 0; k < NACC; ++k) P.c[k] = make_float2(1e-3f * k, 2e-3f * k);
    const int iters = 50000;
    double best = 0.0;
    for (int c : {1, 2, 4}) {
        const int grid = g_sm * c;
        const double ms = time_best_ms(st, 3, [&] { k_operand<MODE><<<grid, PROBE_THREADS, 0, st>>>(g_out, iters, 0.5f, 0.25f, P); });
        if (ms <= 0) return -1.0;
        const double rate = (double)grid * PROBE_THREADS * (double)iters * NACC * 4 * 2.0 / (ms * 1e-3);
        if (rate > best) best = rate;
    }
    return best;
}

template <int THREADS, int IT>
double pair_cbank_t(cudaStream_t st)
{
    static bool loaded = false;
    if (!loaded) {
        static float h[CB_TILES * TILE_FLOATS];
        unsigned s = 4321u;
        for (int t = 0; t < CB_TILES; ++t)
            for (int k = 0; k < NF; ++k)
                for (int l = 0; l < JT; ++l) {
                    s = s * 1664525u + 1013904223u;
                    const float r = (float)(s >> 8) / 16777216.0f;
                    h[t * TILE_FLOATS + k * JT + l] = (k >= F_XL && k < F_V) ? 1e-9f * r : (k == F_M ? 1e-6f : r);
                }
        if (cudaMemcpyToSymbol(c_tiles, h, sizeof(h)) != cudaSuccess) return -1.0;
        loaded = true;
    }
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_pair_cbank<THREADS, IT>, THREADS, 0) != cudaSuccess || occ < 1) return -1.0;
    const int grid = g_sm * occ, reps = 300;
    const double ms = time_best_ms(st, 4, [&] { k_pair_cbank<THREADS, IT><<<grid, THREADS, 0, st>>>(g_out, reps, 1e-8f); });
    if (ms <= 0) return -1.0;
    return (double)grid * THREADS * IT * (double)reps * CB_TILES * JT / (ms * 1e-3);
}

}  // namespace

extern "C" {

// SM cycles (at sm_hz) that 12 two-operand FFMA2 plus `extra` (0, 1, 2, 4 or 12) instructions of `kind` (see k_mix) take on one
// sub-partition when the FMA pipe is the only limit (24 at full rate).  Returns 0 or a cudaError_t.
int g6p_mix_cycles(int kind, int extra, double sm_hz, void *cuda_stream, double *cycles_per_12_ffma2)
{
    if (kind < 0 || kind > 9 || !cycles_per_12_ffma2 || !(sm_hz > 0)) return (int)cudaErrorInvalidValue;
    int rc = probe_init();
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double r = -1.0;
#define MIXCASE(K) case K: r = extra == 0 ? mix_cycles_t<K, 0>(st, sm_hz) : extra == 1 ? mix_cycles_t<K, 1>(st, sm_hz) : extra == 2 ? mix_cycles_t<K, 2>(st, sm_hz) \
                              : extra == 4 ? mix_cycles_t<K, 4>(st, sm_hz) : extra == 12 ? mix_cycles_t<K, 12>(st, sm_hz) : -2.0; break;
    switch (kind) { MIXCASE(0) MIXCASE(1) MIXCASE(2) MIXCASE(3) MIXCASE(4) MIXCASE(5) MIXCASE(6) MIXCASE(7) MIXCASE(8) MIXCASE(9) }
#undef MIXCASE
    if (r == -2.0) return (int)cudaErrorInvalidValue;
    if (r < 0) return (int)cudaGetLastError();
    *cycles_per_12_ffma2 = r;
    return 0;
}

// FP32 lane-instructions per second of the operand-form stream `mode` (see k_operand).  Returns 0 or a cudaError_t.
int g6p_operand_rate(int mode, void *cuda_stream, double *lane_instr_per_s)
{
    if (mode < 0 || mode > 5 || !lane_instr_per_s) return (int)cudaErrorInvalidValue;
    int rc = probe_init();
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double r = -1.0;
    switch (mode) {
        case 0: r = operand_rate_t<0>(st); break;
        case 1: r = operand_rate_t<1>(st); break;
        case 2: r = operand_rate_t<2>(st); break;
        case 3: r = operand_rate_t<3>(st); break;
        case 4: r = operand_rate_t<4>(st); break;
        default: r = operand_rate_t<5>(st); break;
    }
    if (r < 0) return (int)cudaGetLastError();
    *lane_instr_per_s = r;
    return 0;
}

// pair evaluations per second of the production pair loop with its j-tiles in the constant bank; shape 0 = 128 threads x 2
// i-particles, 1 = 128 x 1 (LDCU-bound).  Returns 0 or a cudaError_t.
int g6p_pair_rate_cbank(int shape, void *cuda_stream, double *interactions_per_s)
{
    if (shape < 0 || shape > 1 || !interactions_per_s) return (int)cudaErrorInvalidValue;
    int rc = probe_init();
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const double r = shape == 0 ? pair_cbank_t<128, 2>(st) : pair_cbank_t<128, 1>(st);
    if (r < 0) return (int)cudaGetLastError();
    *interactions_per_s = r;
    return 0;
}


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
