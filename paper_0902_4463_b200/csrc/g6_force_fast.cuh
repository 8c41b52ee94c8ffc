// g6_force_fast.cuh -- the production force kernel for sm_100a (step a-4 of the path).
//
// What it computes is what k_force_ref computes (section 2.3, Eq. 3); how differs from the
// paper's G80 kernel because the B200 bound is the FP32 issue slot, not shared
// memory latency:
//
//  * i-particles live in registers, IT per thread ("one i-particle per thread",
//    generalised).  Every FP32 operation of a pair is issued as a PACKED two-wide instruction
//    (FADD2 / FMUL2 / FFMA2, new in sm_100) over TWO CONSECUTIVE j-particles: the i operand is
//    duplicated once outside the loop, the j operands arrive already paired from shared memory
//    (LDS.128 = four consecutive j of one field).  One issue slot then carries two pairs' worth
//    of FMA-pipe work, which leaves slots for the MUFU.RSQ, the nearest-neighbour FMNMX3 and the
//    shared-memory loads.  IEEE round-to-nearest per lane, so Eq. 3 stays bit-exact.
//  * j-tiles (JT particles, 10 KiB, field-major) are staged global -> shared by ONE 1-D TMA bulk
//    copy each (cp.async.bulk ... mbarrier::complete_tx::bytes) into a ring of NSTAGE buffers
//    guarded by full/empty mbarriers; consumer warps drift by up to NSTAGE-2 tiles, no
//    __syncthreads in the loop.  (PAPER.md:102 loads one j per thread and synchronises.)
//  * self-exclusion is hoisted to tile level: the predictor recorded [min,max] of the j indices of
//    every tile, and a warp takes the checked path (per-pair index compare, address < nj) only on
//    tiles whose index range contains one of its i-particles, or on the ragged last tile.
//    All other tiles run without any per-pair test (needs eps2 > 0 so that s2 > 0).
//  * nearest neighbour: the loop keeps only min r2 (one FMNMX3 per two pairs) and the 8-j step in
//    which it last improved; the j address is recovered afterwards by re-evaluating those 8 j
//    with the same arithmetic (first j that reproduces the minimum: ties -> smallest address).
//  * FP32 partial sums run over one tile (two chains of JT/2 terms per component, even and odd j)
//    and are folded into fp64 accumulators per tile (reading 9).
//  * the grid is (i-tiles) x (S j-splits); S is chosen by the host scheduler so that the SMs are
//    full at any n_i (PAPER.md:82, :104 generalised); partials go to k_combine.
#pragma once
#include "g6_force_ref.cuh"

namespace g6 {

// ---------------------------------------------------------------- PTX helpers (mbarrier + TMA)
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
// bounded wait: a protocol error traps (the launch fails) instead of hanging the device
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t spins = 0;
    while (!mbar_try_wait(bar, parity)) {
        if (++spins > (1u << 24)) __trap();
    }
}
// 1-D TMA bulk copy global -> shared, completion signalled on an mbarrier (bytes % 16 == 0)
__device__ __forceinline__ void tma_load_1d(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// ---------------------------------------------------------------- packed FP32 helpers
__device__ __forceinline__ float2 dup(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }

constexpr float THIRD = 0.333333343267440796f;     // RN32(1/3)
constexpr float FOUR_THIRDS = 1.33333337306976318f; // RN32(4/3)
// pair2 works on sigma = SC s2 (s2 = r2 + eps2) so that the y it ends up with satisfies y^2 = 3 / s2 (see pair2)
template <bool NEWTON> __host__ __device__ constexpr float pair_scale() { return NEWTON ? FOUR_THIRDS : THIRD; }

// per-i-particle register state
struct IPart {
    float2 nxh[3], nxl[3], nv[3];   // NEGATED hi/lo position words and velocity, duplicated
    float2 a[3], j[3], p;           // FP32 tile accumulators: .x even j, .y odd j
    float rmin;                     // min unsoftened r2 so far (over this CTA's j-range)
};

// One i-particle against two consecutive j-particles (packed lanes).  33 FMA-pipe packed
// instructions (+3 with the Newton step), 2 MUFU, 1 FMNMX3.  MASKED: m and r2 already masked.
//   DS = false: pure-FP32 separations, dx = xj_hi - xi_hi (3 packed adds instead of Eq. 3's 9): the variant the
//               paper's "DS costs <~ 20 %" is measured against; bit-identical to DS with zero lo words.
//   DBG       : also hand the separations of the two pairs to the caller (parity pin P11: Eq. 3 bit for bit)
template <bool NEWTON, bool DS = true, bool DBG = false>
__device__ __forceinline__ void pair2(IPart &I, const float2 xh, const float2 yh, const float2 zh, const float2 xl,
                                      const float2 yl, const float2 zl, const float2 vx, const float2 vy, const float2 vz,
                                      const float2 m, const float2 eps2_3, float2 &r2_out, float2 *dbg = nullptr)
{
    // Eq. 3: dx = (xj_hi - xi_hi) + (xj_lo - xi_lo)
    const float2 dx = DS ? add2(add2(xh, I.nxh[0]), add2(xl, I.nxl[0])) : add2(xh, I.nxh[0]);
    const float2 dy = DS ? add2(add2(yh, I.nxh[1]), add2(yl, I.nxl[1])) : add2(yh, I.nxh[1]);
    const float2 dz = DS ? add2(add2(zh, I.nxh[2]), add2(zl, I.nxl[2])) : add2(zh, I.nxh[2]);
    if (DBG) { dbg[0] = dx; dbg[1] = dy; dbg[2] = dz; }
    const float2 dvx = add2(vx, I.nv[0]);
    const float2 dvy = add2(vy, I.nv[1]);
    const float2 dvz = add2(vz, I.nv[2]);
    const float2 r2 = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));
    // sigma = SC s2 instead of s2 (one FFMA2 either way), SC chosen so that the y used below has y^2 = 3 / s2:
    // y^2 then already carries the factor 3 of the jerk's radial term and alpha = -(dx.dv) y^2 needs no separate
    // multiply.  The sums come out scaled by y s (pot) and (y s)^3 (acc, jerk); k_force_fast undoes that exactly
    // (with the binary32 value of SC) in fp64 when it writes its partials.  3 - y^2 s2 = 3e-8 only touches alpha.
    //   no Newton step: SC = 1/3,  y = rsqrt(sigma) = sqrt(3) / s
    //   Newton step   : SC = 4/3,  y0 = rsqrt(sigma);  y = y0 (3 - sigma y0^2) = TWICE the Newton-Raphson iterate
    //                   y0 (3 - sigma y0^2) / 2, i.e. 2 / sqrt(sigma) = sqrt(3) / s: the halving is never done,
    //                   the step costs 3 packed instructions (FMUL2, FFMA2, FMUL2) instead of 4.
    const float2 s2 = fma2(r2, dup(pair_scale<NEWTON>()), eps2_3);          // eps2_3 = SC * eps^2
    float2 rinv = make_float2(rsqrt_approx(s2.x), rsqrt_approx(s2.y));
    if (NEWTON) {
        const float2 ns2 = make_float2(-s2.x, -s2.y);       // folded into the FFMA2 operand modifier
        const float2 u = fma2(ns2, mul2(rinv, rinv), dup(3.0f));
        rinv = mul2(rinv, u);
    }
    const float2 rinv2 = mul2(rinv, rinv);
    const float2 mrinv = mul2(m, rinv);
    const float2 mrinv3 = mul2(mrinv, rinv2);
    const float2 rv = fma2(dz, dvz, fma2(dy, dvy, mul2(dx, dvx)));
    const float2 w = mul2(rv, rinv2);
    const float2 alpha = make_float2(-w.x, -w.y);           // folded into the FFMA2 operand modifier
    I.p = add2(I.p, mrinv);                       // +m/s; the sign is applied at the flush
    I.a[0] = fma2(mrinv3, dx, I.a[0]);
    I.a[1] = fma2(mrinv3, dy, I.a[1]);
    I.a[2] = fma2(mrinv3, dz, I.a[2]);
    I.j[0] = fma2(mrinv3, fma2(alpha, dx, dvx), I.j[0]);
    I.j[1] = fma2(mrinv3, fma2(alpha, dy, dvy), I.j[1]);
    I.j[2] = fma2(mrinv3, fma2(alpha, dz, dvz), I.j[2]);
    r2_out = r2;
}

// DBG: store the separations of j addresses (ja, ja + 1) against i-particle i into A.dbg_dx[i][j][3]
__device__ __forceinline__ void dbg_store(const ForceArgs &A, int i, int ja, const float2 *d)
{
    if (i >= A.ni) return;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        if (ja < A.nj) A.dbg_dx[((size_t)i * A.nj + ja) * 3 + k] = d[k].x;
        if (ja + 1 < A.nj) A.dbg_dx[((size_t)i * A.nj + ja + 1) * 3 + k] = d[k].y;
    }
}

constexpr int FAST_NSTAGE = 4;

template <int THREADS, int IT>
struct FastSmem {
    alignas(128) float tile[FAST_NSTAGE][TILE_FLOATS];
    alignas(8) uint64_t full[FAST_NSTAGE];
    alignas(8) uint64_t empty[FAST_NSTAGE];
};

// NB = true: also build the neighbour lists (r2 < h2_i, reading 20).  The
// unchecked loop then keeps the minimum r2 of each 8-j step (as many FMNMX as before) and compares
// it with max(h2_i, rmin): only a step that holds a neighbour or a new nearest neighbour leaves
// the packed code, re-evaluates its 8 separations from shared memory and appends to the list.
// DS = false: the pure-FP32 variant of pair2 (option "ds" = 0).  DBG: every pair's Eq.-3 separation goes to A.dbg_dx
// (only instantiated by the parity-test hook csrc/debug/g6_debug_dx.cu, never by the library).
template <int THREADS, int IT, bool NEWTON, bool NB = false, bool DS = true, bool DBG = false>
__global__ void __launch_bounds__(THREADS, (NB && THREADS * IT == 256) ? 3 : 0)
k_force_fast(ForceArgs A)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    FastSmem<THREADS, IT> &sm = *reinterpret_cast<FastSmem<THREADS, IT> *>(smem_raw);
    constexpr int NWARP = THREADS / 32;
    constexpr float INF = __builtin_huge_valf();

    const int tid = threadIdx.x;
    const int s = blockIdx.y;
    const int t0 = (int)(((long long)A.ntiles * s) / A.S);
    const int t1 = (int)(((long long)A.ntiles * (s + 1)) / A.S);
    const int nt = t1 - t0;

    if (tid == 0) {
#pragma unroll
        for (int k = 0; k < FAST_NSTAGE; ++k) { mbar_init(&sm.full[k], 1); mbar_init(&sm.empty[k], NWARP); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // prologue: prefetch distance PD = NSTAGE-2 tiles (one tile of slack between warps, see below)
    constexpr int PD = FAST_NSTAGE - 2;
    if (tid == 0) {
#pragma unroll
        for (int k = 0; k < PD; ++k)
            if (k < nt) {
                mbar_expect_tx(&sm.full[k], TILE_BYTES);
                tma_load_1d(sm.tile[k], A.pred + (size_t)(t0 + k) * TILE_FLOATS, TILE_BYTES, &sm.full[k]);
            }
    }

    // ---- my IT i-particles -> registers (fp64 -> double-single / FP32, negated and duplicated)
    IPart I[IT];
    int my[IT];
    double acc[IT][3], jrk[IT][3], pot[IT];
    int bstep[IT];          // the 8-j step (global numbering: address / 8) in which rmin last improved
    float h2f[IT], thr[IT]; // NB: neighbour radius^2 and max(h2, rmin), the step-minimum that needs a look
    int nbc[IT];            // NB: neighbours found so far in this CTA's j-range
#pragma unroll
    for (int q = 0; q < IT; ++q) {
        const int i = (blockIdx.x * IT + q) * THREADS + tid;
        my[q] = i < A.ni ? A.i_index[i] : -1;
        bstep[q] = -1;
        pot[q] = 0;
        I[q].rmin = INF;
        h2f[q] = (NB && i < A.ni) ? (float)A.h2[i] : 0.0f;
        thr[q] = INF;
        nbc[q] = 0;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            float hi = 0.0f, lo = 0.0f, vv = 0.0f;
            if (i < A.ni) {
                ds_split(A.xi[3 * (size_t)i + k], hi, lo);
                if (!A.ds) lo = 0.0f;
                vv = (float)A.vi[3 * (size_t)i + k];
            }
            I[q].nxh[k] = dup(-hi);
            I[q].nxl[k] = dup(-lo);
            I[q].nv[k] = dup(-vv);
            acc[q][k] = 0;
            jrk[q][k] = 0;
        }
    }
    const float2 eps2 = dup(pair_scale<NEWTON>() * A.eps2);  // pair2 works on sigma = SC s2
    // y s = 1 / kP: sqrt(3) nominally; exactly 1 / sqrt(SC) without and 2 / sqrt(SC) with the Newton step
    const double kP = NEWTON ? 0.5 * sqrt((double)FOUR_THIRDS) : sqrt((double)THIRD), kA = kP * kP * kP;

    for (int it = 0; it < nt; ++it) {
        const int t = t0 + it;
        const int st = it % FAST_NSTAGE;
        const uint32_t ph = (uint32_t)(it / FAST_NSTAGE) & 1u;

        // producer: tile it+PD goes into the stage tile it-2 occupied; every warp must have released
        // that one, so this thread never waits on a warp that is less than a tile behind it
        if (tid == 0) {
            const int nx = it + PD;
            if (nx < nt) {
                const int sx = nx % FAST_NSTAGE;
                if (it >= 2) mbar_wait(&sm.empty[sx], (uint32_t)((it - 2) / FAST_NSTAGE) & 1u);
                mbar_expect_tx(&sm.full[sx], TILE_BYTES);
                tma_load_1d(sm.tile[sx], A.pred + (size_t)(t0 + nx) * TILE_FLOATS, TILE_BYTES, &sm.full[sx]);
            }
        }
        // does this warp need the checked path on this tile?
        const int imin = __ldg(A.tile_imin + t), imax = __ldg(A.tile_imax + t);
        bool hit = false;
#pragma unroll
        for (int q = 0; q < IT; ++q) hit |= (my[q] >= imin) & (my[q] <= imax);
        const bool checked = __any_sync(0xffffffffu, hit) || (t * JT + JT > A.nj);

        mbar_wait(&sm.full[st], ph);
        const float4 *T = reinterpret_cast<const float4 *>(sm.tile[st]);

#pragma unroll
        for (int q = 0; q < IT; ++q) {
#pragma unroll
            for (int k = 0; k < 3; ++k) { I[q].a[k] = dup(0.0f); I[q].j[k] = dup(0.0f); }
            I[q].p = dup(0.0f);
        }

        if (!checked) {
            // a step = 8 consecutive j: two LDS.128 per field, four packed pair-evaluations per i
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
                        float2 ra, rb, da[3], db[3];
                        pair2<NEWTON, DS, DBG>(I[q], make_float2(f[0].x, f[0].y), make_float2(f[1].x, f[1].y), make_float2(f[2].x, f[2].y),
                                      make_float2(f[3].x, f[3].y), make_float2(f[4].x, f[4].y), make_float2(f[5].x, f[5].y),
                                      make_float2(f[6].x, f[6].y), make_float2(f[7].x, f[7].y), make_float2(f[8].x, f[8].y),
                                      make_float2(f[9].x, f[9].y), eps2, ra, da);
                        pair2<NEWTON, DS, DBG>(I[q], make_float2(f[0].z, f[0].w), make_float2(f[1].z, f[1].w), make_float2(f[2].z, f[2].w),
                                      make_float2(f[3].z, f[3].w), make_float2(f[4].z, f[4].w), make_float2(f[5].z, f[5].w),
                                      make_float2(f[6].z, f[6].w), make_float2(f[7].z, f[7].w), make_float2(f[8].z, f[8].w),
                                      make_float2(f[9].z, f[9].w), eps2, rb, db);
                        if (DBG) {
                            const int i = (blockIdx.x * IT + q) * THREADS + tid, ja = t * JT + 8 * s8 + 4 * h;
                            dbg_store(A, i, ja, da);
                            dbg_store(A, i, ja + 2, db);
                        }
                        if (NB) {
                            // before[] is reused as the running minimum of this step
                            if (h == 0) before[q] = fminf(fminf(ra.x, ra.y), fminf(rb.x, rb.y));
                            else before[q] = fminf(fminf(fminf(ra.x, ra.y), before[q]), fminf(rb.x, rb.y));
                        } else {
                            I[q].rmin = fminf(fminf(ra.x, ra.y), I[q].rmin);
                            I[q].rmin = fminf(fminf(rb.x, rb.y), I[q].rmin);
                        }
                    }
                }
#pragma unroll
                for (int q = 0; q < IT; ++q) {
                    if (!NB) {
                        if (I[q].rmin < before[q]) bstep[q] = t * (JT / 8) + s8;
                    } else if (before[q] < thr[q]) {
                        // rare: this step holds a neighbour or a new nearest neighbour
                        if (before[q] < I[q].rmin) { I[q].rmin = before[q]; bstep[q] = t * (JT / 8) + s8; }
                        if (before[q] < h2f[q]) {
                            const float *Tf = sm.tile[st] + 8 * s8;
                            const int i = (blockIdx.x * IT + q) * THREADS + tid;
#pragma unroll
                            for (int l = 0; l < 8; ++l) {
                                const float dx = __fadd_rn(__fadd_rn(Tf[(F_XH + 0) * JT + l], I[q].nxh[0].x), __fadd_rn(Tf[(F_XL + 0) * JT + l], I[q].nxl[0].x));
                                const float dy = __fadd_rn(__fadd_rn(Tf[(F_XH + 1) * JT + l], I[q].nxh[1].x), __fadd_rn(Tf[(F_XL + 1) * JT + l], I[q].nxl[1].x));
                                const float dz = __fadd_rn(__fadd_rn(Tf[(F_XH + 2) * JT + l], I[q].nxh[2].x), __fadd_rn(Tf[(F_XL + 2) * JT + l], I[q].nxl[2].x));
                                const float r2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
                                if (r2 < h2f[q]) nb_append(A, s, i, nbc[q], t * JT + 8 * s8 + l);
                            }
                        }
                        thr[q] = fmaxf(h2f[q], I[q].rmin);
                    }
                }
            }
        } else {
            // checked tile: mask out j >= nj and index_j == index_i (mass -> 0, r2 -> +inf)
            const int *JI = tile_indices(A.jraw, t);
            const int4 *JX = reinterpret_cast<const int4 *>(JI);
#pragma unroll 1
            for (int l4 = 0; l4 < JT / 4; ++l4) {
                float4 f[NF];
#pragma unroll
                for (int k = 0; k < NF; ++k) f[k] = T[k * (JT / 4) + l4];
                const int j0 = t * JT + 4 * l4;
                int4 jx = make_int4(0, 0, 0, 0);
                if (j0 + 3 < A.nj) jx = __ldg(JX + l4);
                else {
                    if (j0 + 0 < A.nj) jx.x = __ldg(JI + 4 * l4 + 0);
                    if (j0 + 1 < A.nj) jx.y = __ldg(JI + 4 * l4 + 1);
                    if (j0 + 2 < A.nj) jx.z = __ldg(JI + 4 * l4 + 2);
                }
#pragma unroll
                for (int q = 0; q < IT; ++q) {
                    const bool o0 = (j0 + 0 < A.nj) && (jx.x != my[q]);
                    const bool o1 = (j0 + 1 < A.nj) && (jx.y != my[q]);
                    const bool o2 = (j0 + 2 < A.nj) && (jx.z != my[q]);
                    const bool o3 = (j0 + 3 < A.nj) && (jx.w != my[q]);
                    const float before = I[q].rmin;
                    float2 ra, rb, da[3], db[3];
                    pair2<NEWTON, DS, DBG>(I[q], make_float2(f[0].x, f[0].y), make_float2(f[1].x, f[1].y), make_float2(f[2].x, f[2].y),
                                  make_float2(f[3].x, f[3].y), make_float2(f[4].x, f[4].y), make_float2(f[5].x, f[5].y),
                                  make_float2(f[6].x, f[6].y), make_float2(f[7].x, f[7].y), make_float2(f[8].x, f[8].y),
                                  make_float2(o0 ? f[9].x : 0.0f, o1 ? f[9].y : 0.0f), eps2, ra, da);
                    pair2<NEWTON, DS, DBG>(I[q], make_float2(f[0].z, f[0].w), make_float2(f[1].z, f[1].w), make_float2(f[2].z, f[2].w),
                                  make_float2(f[3].z, f[3].w), make_float2(f[4].z, f[4].w), make_float2(f[5].z, f[5].w),
                                  make_float2(f[6].z, f[6].w), make_float2(f[7].z, f[7].w), make_float2(f[8].z, f[8].w),
                                  make_float2(o2 ? f[9].z : 0.0f, o3 ? f[9].w : 0.0f), eps2, rb, db);
                    if (DBG) {
                        const int i = (blockIdx.x * IT + q) * THREADS + tid;
                        dbg_store(A, i, j0, da);
                        dbg_store(A, i, j0 + 2, db);
                    }
                    I[q].rmin = fminf(fminf(o0 ? ra.x : INF, o1 ? ra.y : INF), I[q].rmin);
                    I[q].rmin = fminf(fminf(o2 ? rb.x : INF, o3 ? rb.y : INF), I[q].rmin);
                    if (I[q].rmin < before) bstep[q] = j0 >> 3;
                    if (NB) {
                        const int i = (blockIdx.x * IT + q) * THREADS + tid;
                        if (o0 && ra.x < h2f[q]) nb_append(A, s, i, nbc[q], j0 + 0);
                        if (o1 && ra.y < h2f[q]) nb_append(A, s, i, nbc[q], j0 + 1);
                        if (o2 && rb.x < h2f[q]) nb_append(A, s, i, nbc[q], j0 + 2);
                        if (o3 && rb.y < h2f[q]) nb_append(A, s, i, nbc[q], j0 + 3);
                        thr[q] = fmaxf(h2f[q], I[q].rmin);
                    }
                }
            }
        }
        // release the stage (one arrival per warp)
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(&sm.empty[st]);

        // fold the tile's FP32 sums into fp64 (chains of JT/2 terms, reading 9)
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

    // ---- recover the nearest neighbour's address: re-evaluate the 8 j of the step that set the
    // minimum with the same arithmetic (packed and scalar IEEE ops round identically); the first j
    // that reproduces rmin wins, so ties go to the smallest address (reading 7)
#pragma unroll
    for (int q = 0; q < IT; ++q) {
        const int i = (blockIdx.x * IT + q) * THREADS + tid;
        if (i >= A.ni) continue;
        int baddr = -1;
        if (bstep[q] >= 0) {
            const int j0 = bstep[q] * 8;
            const float *g = A.pred + (size_t)(j0 / JT) * TILE_FLOATS + (j0 % JT);
            float r2[8];
            int jx[8];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                float4 c[6];
#pragma unroll
                for (int k = 0; k < 6; ++k) c[k] = __ldg(reinterpret_cast<const float4 *>(g + k * JT) + h);
                const float xs[6][4] = {{c[0].x, c[0].y, c[0].z, c[0].w}, {c[1].x, c[1].y, c[1].z, c[1].w}, {c[2].x, c[2].y, c[2].z, c[2].w},
                                        {c[3].x, c[3].y, c[3].z, c[3].w}, {c[4].x, c[4].y, c[4].z, c[4].w}, {c[5].x, c[5].y, c[5].z, c[5].w}};
#pragma unroll
                for (int l = 0; l < 4; ++l) {
                    const float dx = __fadd_rn(__fadd_rn(xs[0][l], I[q].nxh[0].x), __fadd_rn(xs[3][l], I[q].nxl[0].x));
                    const float dy = __fadd_rn(__fadd_rn(xs[1][l], I[q].nxh[1].x), __fadd_rn(xs[4][l], I[q].nxl[1].x));
                    const float dz = __fadd_rn(__fadd_rn(xs[2][l], I[q].nxh[2].x), __fadd_rn(xs[5][l], I[q].nxl[2].x));
                    r2[4 * h + l] = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
                    const int ja = j0 + 4 * h + l;
                    jx[4 * h + l] = ja < A.nj ? j_index(A.jraw, ja) : my[q];
                }
            }
#pragma unroll
            for (int l = 7; l >= 0; --l)
                if (r2[l] == I[q].rmin && jx[l] != my[q]) baddr = j0 + l;
        }
        const size_t o = (size_t)s * A.P.stride_s + (size_t)i * A.P.stride_i;
#pragma unroll
        for (int k = 0; k < 3; ++k) { A.P.acc[k][o] = kA * acc[q][k]; A.P.jrk[k][o] = kA * jrk[q][k]; }
        A.P.pot[o] = kP * pot[q];
        A.P.nn_r2[o] = baddr >= 0 ? I[q].rmin : INF;
        A.P.nn_addr[o] = baddr;
        if (NB) A.nb_cnt[(size_t)s * A.ni + i] = nbc[q];
    }
}

// ---------------------------------------------------------------- host side: shapes + launch
struct FastVariant { int threads, it; };

// The shapes the library builds: (threads, i-particles per thread).  Each exists with and without the Newton step,
// with neighbour lists (NB) and as the pure-FP32 variant (option "ds" = 0; without lists).  128 x 4 and 64 x 2 are
// reachable only through option "variant" (experiments); fast_pick chooses among the first five.
#define G6_FAST_SHAPES(X) X(128, 2) X(128, 1) X(64, 1) X(32, 1) X(256, 1)
#define G6_FAST_EXTRA_SHAPES(X) X(128, 4) X(64, 2)

inline int fast_key(FastVariant v) { return v.threads * 8 + v.it; }

// is (threads, it) a built shape?  `extra`: also the experiment-only shapes (no lists, no pure-FP32 variant)
inline bool fast_is_built(FastVariant v, bool extra)
{
    if (v.threads < 32 || v.it < 1 || v.it > 7) return false;
    switch (fast_key(v)) {
#define X(T, I) case T * 8 + I:
        G6_FAST_SHAPES(X)
        return true;
        G6_FAST_EXTRA_SHAPES(X)
        return extra;
#undef X
        default: return false;
    }
}

template <int THREADS, int IT, bool NB, bool DS>
inline int fast_attr()
{
    const int bytes = (int)sizeof(FastSmem<THREADS, IT>);
    cudaError_t e = cudaFuncSetAttribute(k_force_fast<THREADS, IT, true, NB, DS>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e != cudaSuccess) return (int)e;
    e = cudaFuncSetAttribute(k_force_fast<THREADS, IT, false, NB, DS>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    return (int)e;
}

inline int fast_kernel_init()
{
    int r;
#define X(T, I) if ((r = fast_attr<T, I, false, true>())) return r; if ((r = fast_attr<T, I, true, true>())) return r; if ((r = fast_attr<T, I, false, false>())) return r;
    G6_FAST_SHAPES(X)
#undef X
#define X(T, I) if ((r = fast_attr<T, I, false, true>())) return r;
    G6_FAST_EXTRA_SHAPES(X)
#undef X
    return 0;
}

// pick the (threads, i-per-thread) shape for a block of ni particles.  `force` (option
// "variant" = threads * 8 + it) overrides for experiments.
inline FastVariant fast_pick(int ni, int n_sm, int force)
{
    if (force > 0) return FastVariant{force / 8, force % 8};
    if (ni <= 32) return FastVariant{32, 1};
    if (ni <= 64) return FastVariant{64, 1};
    if (ni < 256) return FastVariant{128, 1};
    // measured at N_j = 2^20: 8 warps sharing one staged j-tile beat 4 by 6-7 % for
    // blocks of 256 .. 4096; on full sweeps 128 x 2 and 256 x 1 are equal
    if (ni <= 128 * n_sm) return FastVariant{256, 1};
    return FastVariant{128, 2};
}

template <int THREADS, int IT, bool NB, bool DS>
inline int fast_launch_t(const ForceArgs &A, bool newton, int n_itiles, int S, cudaStream_t st)
{
    dim3 grid(n_itiles, S);
    const size_t bytes = sizeof(FastSmem<THREADS, IT>);
    if (newton) k_force_fast<THREADS, IT, true, NB, DS><<<grid, THREADS, bytes, st>>>(A);
    else k_force_fast<THREADS, IT, false, NB, DS><<<grid, THREADS, bytes, st>>>(A);
    return (int)cudaGetLastError();
}

// neighbour lists exist for the automatic shapes only
inline bool fast_has_nb(FastVariant v) { return fast_is_built(v, false); }

// A.h2 != nullptr: with neighbour lists (double-single arithmetic; with ds = 0 the lo words are zero, which is the same
// numbers).  A.ds == 0 without lists: the pure-FP32 variant (3 packed adds per separation instead of 9).
inline int launch_force_fast(const ForceArgs &A, bool newton, FastVariant v, int n_itiles, int S, cudaStream_t st)
{
    switch (fast_key(v)) {
#define X(T, I) case T * 8 + I: \
            if (A.h2) return fast_launch_t<T, I, true, true>(A, newton, n_itiles, S, st); \
            if (!A.ds) return fast_launch_t<T, I, false, false>(A, newton, n_itiles, S, st); \
            return fast_launch_t<T, I, false, true>(A, newton, n_itiles, S, st);
        G6_FAST_SHAPES(X)
#undef X
#define X(T, I) case T * 8 + I: \
            if (A.h2) return (int)cudaErrorInvalidValue; \
            return fast_launch_t<T, I, false, true>(A, newton, n_itiles, S, st);
        G6_FAST_EXTRA_SHAPES(X)
#undef X
        default: return (int)cudaErrorInvalidValue;
    }
}

// resident CTAs per SM of a shape (for the j-split scheduler); nb: the neighbour-list build (more registers)
template <int THREADS, int IT, bool NB>
inline int fast_occ_t()
{
    static int n = 0;
    if (!n) {
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_force_fast<THREADS, IT, true, NB, true>, THREADS, sizeof(FastSmem<THREADS, IT>)) != cudaSuccess || n < 1) n = 1;
    }
    return n;
}
inline int fast_ctas_per_sm(FastVariant v, bool nb = false)
{
    switch (fast_key(v)) {
#define X(T, I) case T * 8 + I: return nb ? fast_occ_t<T, I, true>() : fast_occ_t<T, I, false>();
        G6_FAST_SHAPES(X)
#undef X
#define X(T, I) case T * 8 + I: return fast_occ_t<T, I, false>();
        G6_FAST_EXTRA_SHAPES(X)
#undef X
        default: return 1;
    }
}
inline int fast_ctas_per_sm_nb(FastVariant v) { return fast_ctas_per_sm(v, true); }

}  // namespace g6
