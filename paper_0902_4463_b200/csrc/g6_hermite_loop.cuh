// g6_hermite_loop.cuh -- the block-step LOOP on the device (SURVEY.md 8(f) NEXT-3 "CUDA-graph step loop", built as a
// persistent cooperative kernel because the shape of a block step depends on n_i, which a captured graph cannot follow).
//
// "Block sizes are typically small on average": in the 32k Hermite run three quarters of the block steps
// have fewer than 32 active particles, and such a step costs launches and host round trips, not arithmetic.  Here ONE
// cooperative kernel runs block step after block step -- select, predict i, predict j, force, combine, correct, j-store
// update -- and returns to the host only for a block larger than `max_i`, at t_end, or after `max_steps`:
//
//  * CTA c (one per SM, all co-resident) OWNS the raw j-tiles c, c + G, ... (at most HL_KMAX) and keeps them IN SHARED MEMORY
//    for the whole run, together with t + dt of their particles: per block step no j-particle is read from HBM or L2 at all;
//    the owner patches the staged record of a particle it has just corrected and writes it through to the j-store.
//  * a block step has three grid-wide barriers (one atomic arrival + a generation word, ~1.5 us each):
//      A  every CTA publishes (min, count at the min) of t + dt per owned tile          -> barrier 1
//         everybody derives t_next = global min, n_i and each tile's offset in the active list (increasing address);
//         owners predict their active particles in fp64 (Eq. 1-2) into the shared i-block     -> barrier 2
//      B  every CTA: i-block -> double-single in shared memory, Eq. 1-2 of its resident j-particles (same routine as
//         k_predict), then all pairs with the packed, checked pair code of the block-step kernel (pair2_checked; Eq. 3).
//         Lanes of a warp = (i-particle, j-sub-range): "several threads share an i and split the j";
//         the lanes of one i are summed by a fixed shuffle tree ONCE per step, the warps and the CTAs in fixed order in fp64
//         (reading 9): bit-reproducible.  One partial per (i, CTA)                                  -> barrier 3
//      C  the owner of each active particle sums its G partials (a warp per particle, the order of k_combine_wide), runs
//         the corrector, the Aarseth step and the power-of-two rule (hd_correct_one), and updates its resident tile.
//  * a block with n_i > max_i is selected and predicted (phase A) and handed to the host, which runs the library's sweep path
//    on it (hd_force) and re-enters the loop.
// The nearest neighbour is not tracked (the Hermite driver does not use it).
#pragma once
#include "g6_block_step.cuh"
#include "g6_hermite_dev.cuh"

namespace g6 {

constexpr int HL_THREADS = 256;
constexpr int HL_NW = HL_THREADS / 32;
constexpr int HL_KMAX = 4;                    // resident raw tiles per CTA
constexpr int HL_MAX_I = 1024;                // largest block the loop can step itself
constexpr int HL_MAX_G = 160;                 // CTAs (one per SM)
constexpr int HL_MAX_TILES = HL_MAX_G * HL_KMAX;

enum { HL_END = 0, HL_BIG = 1, HL_STEPS = 2 };

struct HlStatus {
    double t;              // system time reached
    double tnext;          // HL_BIG: time of the block handed over
    long long steps;       // block steps taken by this launch
    long long npart;       // particle steps
    int reason;            // HL_END: t >= t_end; HL_BIG: the next block (ni_next particles) is selected and predicted; HL_STEPS: max_steps taken
    int ni_next;
    int ni_last;           // size of the last block stepped (0: none)
    int pad;
    long long hist[64];    // block steps by log2(n_i)
    long long ns[64];      // device time (globaltimer, ns) spent in the block steps of each bin, as seen by CTA 0
    long long phase_ns[8]; // PROFILING: time between the phase boundaries of steps with n_i < 32 (CTA 0)
};

struct HlArgs {
    HdState S;
    HdBlock B;
    HdCorr C;
    double *a1, *ad1, *pot;        // forces of the current block (= C.a1, C.ad1), writable
    int ntiles, K, nj;
    double t_sys, t_end;
    long long max_steps;
    int max_i;
    float eps2;
    int ds;
    Partials P;                    // [k][G]: stride_s = 1, stride_i = G
    double *tile_min;              // [ntiles] per-tile minimum of t + dt
    int *tile_cnt;                 // [ntiles] particles of the tile at that minimum
    unsigned int *bar;             // [2] arrival count, generation
    HlStatus *status;              // device-visible (mapped host memory)
};

struct HlSmem {
    alignas(16) char raw[HL_KMAX][RAW_TILE_BYTES];      // the CTA's own raw j-tiles, resident
    alignas(16) float pred[HL_KMAX][TILE_FLOATS];       // their Eq. 1-2 predictions at the block time
    double tnext[HL_KMAX][JT];                          // t + dt of the own particles (+inf past the end)
    float ipart[HL_MAX_I][9];                           // i-block: hi[3], lo[3], v[3]
    int iidx[HL_MAX_I];
    double wsum[HL_NW][32][8];                          // per-warp sums of one i-chunk
    double s_tm[HL_MAX_TILES];
    int s_tc[HL_MAX_TILES];
    int s_off[HL_MAX_TILES];
    int own_k[HL_KMAX * JT], own_l[HL_KMAX * JT];       // my active particles: position in the active list, slot kk * JT + l
    double red[HL_NW][HL_KMAX];
    int redc[HL_NW][HL_KMAX];
    double gmin;
    int ni, nown;
};
static_assert(sizeof(HlSmem) <= 232448, "loop kernel shared memory");

// grid-wide barrier: sense by generation; every CTA of the (cooperative) launch must call it
__device__ __forceinline__ void hl_grid_barrier(unsigned int *bar, unsigned int G)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned int gen;
        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(gen) : "l"(bar + 1) : "memory");
        __threadfence();
        if (atomicAdd(bar, 1u) == G - 1u) {
            bar[0] = 0u;
            __threadfence();
            asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(bar + 1), "r"(gen + 1u) : "memory");
        } else {
            unsigned int now, spins = 0;
            do {
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(now) : "l"(bar + 1) : "memory");
                if (++spins > (1u << 28)) __trap();          // a protocol error fails the launch instead of hanging the device
            } while (now == gen);
        }
        __threadfence();
    }
    __syncthreads();
}

// particle p's Hermite state -> slot l of a raw tile in shared memory (what hd_store_j writes to the j-store)
__device__ __forceinline__ void hl_store_tile(char *T, int l, const HdState &S, int p)
{
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        raw_x(T, k, l) = S.x[3 * (size_t)p + k];
        raw_v(T, k, l) = (float)S.v[3 * (size_t)p + k];
        raw_a2(T, k, l) = (float)(S.a[3 * (size_t)p + k] / 2);
        raw_j6(T, k, l) = (float)(S.ad[3 * (size_t)p + k] / 6);
    }
    raw_t(T, l) = S.t[p];
    raw_m(T, l) = (float)S.m[p];
    raw_idx(T, l) = p;
}

template <bool NEWTON>
__global__ void __launch_bounds__(HL_THREADS, 1)
k_hd_loop(const HlArgs A)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    HlSmem &sm = *reinterpret_cast<HlSmem *>(smem_raw);
    const unsigned FULL = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int G = gridDim.x, cta = blockIdx.x;
    const double INF = __longlong_as_double(0x7ff0000000000000LL);
    const int Kc = cta < A.ntiles ? (A.ntiles - cta + G - 1) / G : 0;       // my tiles: cta, cta + G, ...

    // ---- load my tiles and the t + dt of their particles
    for (int kk = 0; kk < Kc; ++kk) {
        const int4 *src = reinterpret_cast<const int4 *>(A.C.raw + (size_t)(cta + kk * G) * RAW_TILE_BYTES);
        int4 *dst = reinterpret_cast<int4 *>(sm.raw[kk]);
        for (int q = tid; q < RAW_TILE_BYTES / 16; q += HL_THREADS) dst[q] = __ldcg(src + q);
        const int p = (cta + kk * G) * JT + tid;
        sm.tnext[kk][tid] = p < A.S.n ? A.S.t[p] + A.S.dt[p] : INF;
    }
    __syncthreads();

    double t_sys = A.t_sys;
    long long steps = 0, npart = 0;
    long long hist = 0, hist_ns = 0;       // thread b < 64 of CTA 0 counts bin b
    unsigned long long t_step = 0;
    if (cta == 0) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_step));
    long long ph[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    unsigned long long stamp[8];
#define HL_STAMP(k) do { if (cta == 0 && tid == 0) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(stamp[k])); } while (0)
    int reason = HL_END, ni_next = 0, ni_last = 0;
    double t_big = 0.0;
    const float2 eps2 = dup(A.eps2);

    for (;;) {
        if (!(t_sys < A.t_end)) { reason = HL_END; break; }
        if (A.max_steps > 0 && steps >= A.max_steps) { reason = HL_STEPS; break; }

        HL_STAMP(0);
        // ================= phase A: (min, count) of t + dt per own tile
        {
            double v[HL_KMAX];
#pragma unroll
            for (int kk = 0; kk < HL_KMAX; ++kk) {
                v[kk] = kk < Kc ? sm.tnext[kk][tid] : INF;
                double m = v[kk];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) m = fmin(m, __shfl_xor_sync(FULL, m, o));
                if (lane == 0) sm.red[w][kk] = m;
            }
            __syncthreads();
#pragma unroll
            for (int kk = 0; kk < HL_KMAX; ++kk) {
                double m = sm.red[0][kk];
#pragma unroll
                for (int q = 1; q < HL_NW; ++q) m = fmin(m, sm.red[q][kk]);
                const unsigned bal = __ballot_sync(FULL, kk < Kc && v[kk] == m);
                if (lane == 0) sm.redc[w][kk] = __popc(bal);
                v[kk] = m;
            }
            __syncthreads();
            if (tid < Kc) {
                int c = 0;
                double m = sm.red[0][tid];
#pragma unroll
                for (int q = 0; q < HL_NW; ++q) { c += sm.redc[q][tid]; m = fmin(m, sm.red[q][tid]); }
                __stcg(A.tile_min + cta + tid * G, m);
                __stcg(A.tile_cnt + cta + tid * G, c);
            }
        }
        HL_STAMP(1);
        hl_grid_barrier(A.bar, G);
        HL_STAMP(2);

        // everybody: t_next, n_i, offsets of the tiles in the active list (tile order = increasing address)
        {
            double m = INF;
            for (int T = tid; T < A.ntiles; T += HL_THREADS) {
                const double tm = __ldcg(A.tile_min + T);
                sm.s_tm[T] = tm;
                sm.s_tc[T] = __ldcg(A.tile_cnt + T);
                m = fmin(m, tm);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) m = fmin(m, __shfl_xor_sync(FULL, m, o));
            if (lane == 0) sm.red[w][0] = m;
            __syncthreads();
            m = sm.red[0][0];
#pragma unroll
            for (int q = 1; q < HL_NW; ++q) m = fmin(m, sm.red[q][0]);
            if (w == 0) {
                int run = 0;
                for (int T0 = 0; T0 < A.ntiles; T0 += 32) {
                    const int T = T0 + lane;
                    const bool hit = T < A.ntiles && sm.s_tm[T] == m;
                    const int c = hit ? sm.s_tc[T] : 0;
                    int inc = c;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const int u = __shfl_up_sync(FULL, inc, o);
                        if (lane >= o) inc += u;
                    }
                    if (T < A.ntiles) sm.s_off[T] = hit ? run + inc - c : -1;
                    run += __shfl_sync(FULL, inc, 31);
                }
                if (lane == 0) { sm.ni = run; sm.gmin = m; }
            }
            __syncthreads();
        }
        const double tn = sm.gmin;
        const int ni = sm.ni;
        const bool big = ni > A.max_i;

        // owners: active particles of my tiles, in address order, predicted in fp64 into the shared i-block
        {
            int nown = 0;
            for (int kk = 0; kk < Kc; ++kk) {
                const int T = cta + kk * G;
                const int base = sm.s_off[T];
                if (base < 0) continue;                                     // uniform over the CTA
                const bool on = sm.tnext[kk][tid] == tn;
                const unsigned bal = __ballot_sync(FULL, on);
                if (lane == 0) sm.redc[w][0] = __popc(bal);
                __syncthreads();
                int before = 0, total = 0;
#pragma unroll
                for (int q = 0; q < HL_NW; ++q) { const int cw = sm.redc[q][0]; before += q < w ? cw : 0; total += cw; }
                if (on) {
                    const int r = before + __popc(bal & ((1u << lane) - 1u));
                    const int k = base + r, p = T * JT + tid;
                    A.B.act[k] = p;
                    hd_predict(A.S, p, tn, A.B.xi + 3 * (size_t)k, A.B.vi + 3 * (size_t)k);
                    if (!big) { sm.own_k[nown + r] = k; sm.own_l[nown + r] = kk * JT + tid; }
                }
                nown += total;
                __syncthreads();
            }
            if (tid == 0) sm.nown = nown;
        }
        HL_STAMP(3);
        hl_grid_barrier(A.bar, G);
        HL_STAMP(4);
        if (big) { reason = HL_BIG; ni_next = ni; t_big = tn; break; }

        // ================= phase B: i-block -> double-single, my j-particles -> Eq. 1-2 at tn, all pairs
        for (int q = tid; q < ni * 3; q += HL_THREADS) {
            const int i = q / 3, c = q % 3;
            float hi, lo;
            ds_split(__ldcg(A.B.xi + q), hi, lo);
            sm.ipart[i][c] = hi;
            sm.ipart[i][3 + c] = A.ds ? lo : 0.0f;
            sm.ipart[i][6 + c] = (float)__ldcg(A.B.vi + q);
        }
        for (int i = tid; i < ni; i += HL_THREADS) sm.iidx[i] = __ldcg(A.B.act + i);
        for (int kk = 0; kk < Kc; ++kk) {
            char *R = sm.raw[kk];
            float *Pj = sm.pred[kk];
            const float dt = (float)(tn - raw_t(R, tid));
#pragma unroll
            for (int k = 0; k < 3; ++k)
                predict_coord(dt, raw_x(R, k, tid), raw_v(R, k, tid), raw_a2(R, k, tid), raw_j6(R, k, tid), A.ds,
                              Pj[(F_XH + k) * JT + tid], Pj[(F_XL + k) * JT + tid], Pj[(F_V + k) * JT + tid]);
            Pj[F_M * JT + tid] = raw_m(R, tid);
        }
        __syncthreads();

        for (int c0 = 0; c0 < ni; c0 += 32) {
            const int nic = min(32, ni - c0);
            int lg = 1;                                   // lanes per warp = 2^lg i-particles x 2^(5-lg) j-sub-ranges of 2^lg j each
            while ((1 << lg) < nic) ++lg;
            const int pw = 1 << lg;
            const int ii = lane & (pw - 1), jsub = lane >> lg;
            const bool act = ii < nic;
            IPart I;
            int my = -1;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                I.nxh[k] = dup(act ? -sm.ipart[c0 + ii][k] : 0.0f);
                I.nxl[k] = dup(act ? -sm.ipart[c0 + ii][3 + k] : 0.0f);
                I.nv[k] = dup(act ? -sm.ipart[c0 + ii][6 + k] : 0.0f);
                I.a[k] = dup(0.0f);
                I.j[k] = dup(0.0f);
            }
            I.p = dup(0.0f);
            if (act) my = sm.iidx[c0 + ii];
            if (act) {
                for (int kk = 0; kk < Kc; ++kk) {
                    const float *Pj = sm.pred[kk];
                    const int *JX = reinterpret_cast<const int *>(sm.raw[kk] + RAW_IDX);
                    const int jl0 = 32 * w + jsub * pw;
                    const int ja0 = (cta + kk * G) * JT + jl0;
                    for (int q = 0; q < pw; q += 2) {
                        const int jl = jl0 + q, ja = ja0 + q;
                        float2 f[NF];
#pragma unroll
                        for (int k = 0; k < NF; ++k) f[k] = *reinterpret_cast<const float2 *>(Pj + k * JT + jl);
                        const int2 jx = *reinterpret_cast<const int2 *>(JX + jl);
                        float2 r2;
                        pair2_checked<NEWTON>(I, f[0], f[1], f[2], f[3], f[4], f[5], f[6], f[7], f[8], f[9], eps2,
                                              (ja < A.nj) && (jx.x != my), (ja + 1 < A.nj) && (jx.y != my), r2);
                    }
                }
            }
            // the lanes of one i-particle (its j-sub-ranges): fixed shuffle tree, FP32 (chains of <= 256 pairs, reading 9)
            float v7[7] = {__fadd_rn(I.a[0].x, I.a[0].y), __fadd_rn(I.a[1].x, I.a[1].y), __fadd_rn(I.a[2].x, I.a[2].y),
                           __fadd_rn(I.j[0].x, I.j[0].y), __fadd_rn(I.j[1].x, I.j[1].y), __fadd_rn(I.j[2].x, I.j[2].y),
                           __fadd_rn(I.p.x, I.p.y)};
            for (int o = pw; o < 32; o <<= 1) {
#pragma unroll
                for (int k = 0; k < 7; ++k) v7[k] = __fadd_rn(v7[k], __shfl_xor_sync(FULL, v7[k], o));
            }
            if (lane < pw) {
#pragma unroll
                for (int k = 0; k < 7; ++k) sm.wsum[w][lane][k] = (double)v7[k];
            }
            __syncthreads();
            if (tid < nic) {                              // the warps in warp order, fp64: one partial per (i, CTA)
                double s7[7];
#pragma unroll
                for (int k = 0; k < 7; ++k) s7[k] = sm.wsum[0][tid][k];
#pragma unroll
                for (int q = 1; q < HL_NW; ++q) {
#pragma unroll
                    for (int k = 0; k < 7; ++k) s7[k] += sm.wsum[q][tid][k];
                }
                const size_t o = (size_t)cta * A.P.stride_s + (size_t)(c0 + tid) * A.P.stride_i;
#pragma unroll
                for (int k = 0; k < 3; ++k) { __stcg(A.P.acc[k] + o, s7[k]); __stcg(A.P.jrk[k] + o, s7[3 + k]); }
                __stcg(A.P.pot + o, -s7[6]);
            }
            __syncthreads();
        }
        HL_STAMP(5);
        hl_grid_barrier(A.bar, G);
        HL_STAMP(6);

        // ================= phase C: owners combine (fixed order) and correct their particles
        const int nown = sm.nown;
        for (int q = w; q < nown; q += HL_NW) {
            const int k = sm.own_k[q], slot = sm.own_l[q];
            double v[7] = {0, 0, 0, 0, 0, 0, 0};
            for (int s = lane; s < G; s += 32) {
                const size_t o = (size_t)s * A.P.stride_s + (size_t)k * A.P.stride_i;
#pragma unroll
                for (int c = 0; c < 3; ++c) { v[c] += __ldcg(A.P.acc[c] + o); v[3 + c] += __ldcg(A.P.jrk[c] + o); }
                v[6] += __ldcg(A.P.pot + o);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
                for (int c = 0; c < 7; ++c) v[c] += __shfl_xor_sync(FULL, v[c], o);
            }
            if (lane == 0) {
#pragma unroll
                for (int c = 0; c < 3; ++c) { A.a1[3 * (size_t)k + c] = v[c]; A.ad1[3 * (size_t)k + c] = v[3 + c]; }
                A.pot[k] = v[6];
                hd_correct_one(A.S, A.B, A.C, k, tn);      // corrector, new step, j-store record (global)
                const int kk = slot / JT, l = slot % JT;
                const int p = (cta + kk * G) * JT + l;
                hl_store_tile(sm.raw[kk], l, A.S, p);       // ... and my resident copy
                sm.tnext[kk][l] = tn + A.S.dt[p];
            }
        }
        HL_STAMP(7);
        if (cta == 0 && tid == 0 && ni < 32) { for (int k = 0; k < 7; ++k) ph[k] += (long long)(stamp[k + 1] - stamp[k]); ph[7] += 1; }
        t_sys = tn;
        ++steps;
        npart += ni;
        ni_last = ni;
        if (cta == 0) {
            unsigned long long now;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(now));
            if (tid < 30 && ni >= (1 << tid) && ni < (2 << tid)) { ++hist; hist_ns += (long long)(now - t_step); }
            t_step = now;
        }
        __syncthreads();
    }

    if (cta == 0) {
        if (tid < 64) { A.status->hist[tid] = hist; A.status->ns[tid] = hist_ns; }
        if (tid == 0) {
            A.status->t = t_sys;
            A.status->tnext = t_big;
            A.status->steps = steps;
            A.status->npart = npart;
            A.status->reason = reason;
            A.status->ni_next = ni_next;
            A.status->ni_last = ni_last;
            for (int k = 0; k < 8; ++k) A.status->phase_ns[k] = ph[k];
            if (reason == HL_BIG) { *A.B.d_ni = ni_next; *A.B.d_tnext = t_big; }
            else if (ni_last > 0) { *A.B.d_ni = ni_last; *A.B.d_tnext = t_sys; }
        }
    }
}

}  // namespace g6
