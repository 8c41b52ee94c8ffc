// g6_hermite_dev.cuh -- device-resident 4th-order Hermite block-step integrator:
// the block selection, the prediction of the i-particles, the corrector and the step choice run on the
// GPU, so that per block step only two numbers (n_i and the block time) cross to the host, instead of the
// i-block, the forces and n_i calls of g6_set_j_particle.  The paper keeps these O(n_i) steps on the CPU
// (Fig. 1) because the GRAPE host codes did; it names the force as the only O(N n_i) part
// (PAPER.md:49).  Formulas: DESIGN.md reading 16 (Makino & Aarseth 1992 / Aarseth 1985, cited at
// PAPER.md:31, :156), the same as the host driver g6_hermite.cpp, in fp64.
//
//   k_hd_select   t_next = min_p (t_p + dt_p); the active block = all p with t_p + dt_p == t_next, in
//                 increasing address order; Eq. 1-2 prediction of those i-particles in
//                 fp64 ("similarly implemented on the CPU" -- here on the device)
//   force         the library's own path (run_force: block-step kernel or predictor + sweep kernel)
//   k_hd_correct  corrector, Aarseth step, power-of-two quantisation, new j-store record
#pragma once
#include "g6_device.cuh"

namespace g6 {

struct HdState {
    double *x, *v, *a, *ad;     // [n][3] at each particle's own time t
    double *m, *t, *dt;         // [n]
    int n;
};

// what the host waits for, written with ONE 16-byte store to mapped host memory (one PCIe write: never torn)
struct alignas(16) HdNote {
    double tnext;
    int ni;
    unsigned int seq;
};

__device__ __forceinline__ void hd_notify(HdNote *h, double tnext, int ni, unsigned int seq)
{
    const unsigned long long lo = (unsigned long long)__double_as_longlong(tnext);
    const unsigned long long hi = (unsigned long long)(unsigned)ni | ((unsigned long long)seq << 32);
    asm volatile("st.global.v2.u64 [%0], {%1, %2};" ::"l"(h), "l"(lo), "l"(hi) : "memory");
}

// per-step scratch written by k_hd_select
struct HdBlock {
    int *act;                   // [n] active addresses, increasing
    int *cand;                  // [nblocks * HD_PER_BLOCK] per-thread-block candidates (particles at the block minimum)
    double *xi, *vi;            // [n][3] predicted i-particles
    double *bmin;               // [nblocks] per-thread-block minimum of t + dt
    int *bcnt;                  // [nblocks] particles of the block attaining it
    int *boff;                  // [nblocks] where the block's candidates go in the active list, -1: not in this block step
    unsigned int *ticket;
    HdNote *h_note;             // mapped host memory: (t_next, n_i, sequence number) of the block, one 16-byte store
    unsigned int seq;           // sequence number of this launch (the host spins on it instead of waiting for an event)
    int *d_ni;                  // device copy of n_i (read by k_hd_correct)
    double *d_tnext;
};

constexpr int HD_THREADS = 256;
constexpr int HD_PER_BLOCK = 1024;      // particles per thread block of k_hd_select

__device__ __forceinline__ double hd_block_min(double v, double *sm)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
    __syncthreads();
    double r = sm[0];
#pragma unroll
    for (int w = 1; w < HD_THREADS / 32; ++w) r = fmin(r, sm[w]);
    __syncthreads();
    return r;
}

// Eq. 1-2 in fp64 for particle p at time tn
__device__ __forceinline__ void hd_predict(const HdState &S, int p, double tn, double *xp, double *vp)
{
    // read from L2 (ld.global.cg): the state may have been written by another thread block of the same launch (the corrector of the
    // last-block patterns, the owners of the step loop), and nothing on this path invalidates L1
    const double h = tn - __ldcg(S.t + p), h2 = h * h / 2, h3 = h * h * h / 6;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const double x = __ldcg(S.x + 3 * (size_t)p + k), v = __ldcg(S.v + 3 * (size_t)p + k), a = __ldcg(S.a + 3 * (size_t)p + k), ad = __ldcg(S.ad + 3 * (size_t)p + k);
        xp[k] = x + v * h + a * h2 + ad * h3;
        vp[k] = v + a * h + ad * h2;
    }
}

// smallest power-of-two step <= cap that does not exceed `want` (the host driver's pow2_floor)
__device__ __forceinline__ double hd_pow2_floor(double want, double cap)
{
    double d = cap;
    while (d > want && d > 1e-300) d *= 0.5;
    return d;
}

// is t a multiple of the power-of-two step d?  (t / d is exact; fmod in fp64 is a long loop on the device)
__device__ __forceinline__ bool hd_is_multiple(double t, double d)
{
    const double q = t / d;
    return q == rint(q);
}

__device__ __forceinline__ double hd_norm3(const double *a) { return sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]); }

// write particle p's Hermite state into the raw j-store (what g6_set_j_particle + k_stage do on the host path)
__device__ __forceinline__ void hd_store_j(char *raw, const HdState &S, int p)
{
    char *T = raw_tile(raw, p);
    const int l = p % JT;
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

// corrector + Aarseth step + power-of-two rule + new j-store record for entry k of the block (reading 16)
struct HdCorr {
    const double *a1, *ad1;     // forces of the block, [n_i][3]
    double eta, dt_max;
    char *raw;                  // the library's j-store
    unsigned long long *dt_min_bits;
};

// the arithmetic of one corrector step, by value: step h, old (a0, ad0), new (a1, ad1) forces, predicted (xi, vi) at the new
// time tn -> corrected x1, v1 and the new step (return value)
__device__ __forceinline__ double hd_correct_core(double h, const double *a0, const double *ad0, const double *a1, const double *ad1,
                                                  const double *xi, const double *vi, double tn, double eta, double dt_max,
                                                  double *x1, double *v1)
{
    // fp64 division costs ~60 dependent instructions on the device and the corrector sits on the critical path of every small
    // block step: ONE reciprocal of h (exact when h is a power of two, as the steps are for a power-of-two dt_max) and
    // reciprocal constants replace the ten divisions per component; results agree with the host driver's to rounding
    const double h2 = h * h, h3 = h2 * h, h4 = h3 * h, h5 = h4 * h;
    const double ih = 1.0 / h, ih2 = ih * ih, ih3 = ih2 * ih;
    constexpr double R6 = 1.0 / 6, R24 = 1.0 / 24, R120 = 1.0 / 120;
    double a2n[3], a3[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double da = a0[c] - a1[c];
        const double a2 = (-6 * da - h * (4 * ad0[c] + 2 * ad1[c])) * ih2;
        a3[c] = (12 * da + 6 * h * (ad0[c] + ad1[c])) * ih3;
        x1[c] = xi[c] + h4 * a2 * R24 + h5 * a3[c] * R120;
        v1[c] = vi[c] + h3 * a2 * R6 + h4 * a3[c] * R24;
        a2n[c] = a2 + h * a3[c];
    }
    const double na = hd_norm3(a1), nad = hd_norm3(ad1), n2 = hd_norm3(a2n), n3 = hd_norm3(a3);
    const double den = nad * n3 + n2 * n2;
    const double want = den > 0 ? sqrt(eta * (na * n2 + nad * nad) / den) : dt_max;
    double d = h;
    if (want < d) {
        while (d > want && d > 1e-300) d *= 0.5;     // floor: a zero or NaN wish must not loop forever (the host then sees no progress)
    } else if (want >= 2 * d && 2 * d <= dt_max && hd_is_multiple(tn, 2 * d)) {
        d *= 2;
    }
    return d;
}

// The same corrector step by the first four lanes of a warp (the step loop's owners: the corrector sits on the critical path of
// every small block step and a single thread's fp64 latency chain was 2-3 us of it).  Lanes 0-2 take one component each -- the
// expressions of hd_correct_core, so the same numbers -- the components meet through shuffles, lanes 0-3 take one of the four
// norms (a square root each), lane 0 the Aarseth formula and the power-of-two rule.  Call with the whole warp converged.
//   in : h, tn, eta, dt_max (uniform); lane c < 3: a0c, ad0c, a1c, ad1c, xic, vic of component c
//   out: lane c < 3: x1c, v1c; return value (all lanes): the new step
__device__ __forceinline__ double hd_correct_warp(int lane, double h, double a0c, double ad0c, double a1c, double ad1c, double xic, double vic,
                                                  double tn, double eta, double dt_max, double &x1c, double &v1c)
{
    const unsigned FULL = 0xffffffffu;
    const double h2 = h * h, h3 = h2 * h, h4 = h3 * h, h5 = h4 * h;
    const double ih = 1.0 / h, ih2 = ih * ih, ih3 = ih2 * ih;
    constexpr double R6 = 1.0 / 6, R24 = 1.0 / 24, R120 = 1.0 / 120;
    const double da = a0c - a1c;
    const double a2 = (-6 * da - h * (4 * ad0c + 2 * ad1c)) * ih2;
    const double a3c = (12 * da + 6 * h * (ad0c + ad1c)) * ih3;
    x1c = xic + h4 * a2 * R24 + h5 * a3c * R120;
    v1c = vic + h3 * a2 * R6 + h4 * a3c * R24;
    const double a2nc = a2 + h * a3c;
    // lane L < 4 gets vector L of (a1, ad1, a2n, a3)
    double vec[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double q0 = __shfl_sync(FULL, a1c, c), q1 = __shfl_sync(FULL, ad1c, c), q2 = __shfl_sync(FULL, a2nc, c), q3 = __shfl_sync(FULL, a3c, c);
        vec[c] = lane == 0 ? q0 : lane == 1 ? q1 : lane == 2 ? q2 : q3;
    }
    const double nrm = hd_norm3(vec);
    const double na = __shfl_sync(FULL, nrm, 0), nad = __shfl_sync(FULL, nrm, 1), n2 = __shfl_sync(FULL, nrm, 2), n3 = __shfl_sync(FULL, nrm, 3);
    double d = h;
    if (lane == 0) {
        const double den = nad * n3 + n2 * n2;
        const double want = den > 0 ? sqrt(eta * (na * n2 + nad * nad) / den) : dt_max;
        if (want < d) {
            while (d > want && d > 1e-300) d *= 0.5;
        } else if (want >= 2 * d && 2 * d <= dt_max && hd_is_multiple(tn, 2 * d)) {
            d *= 2;
        }
    }
    return __shfl_sync(FULL, d, 0);
}

__device__ __forceinline__ void hd_correct_one(const HdState &S, const HdBlock &B, const HdCorr &C, int k, double tn)
{
    const int p = B.act[k];
    double a0[3], ad0[3], a1[3], ad1[3], xi[3], vi[3], x1[3], v1[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        a0[c] = S.a[3 * (size_t)p + c]; ad0[c] = S.ad[3 * (size_t)p + c];
        a1[c] = C.a1[3 * (size_t)k + c]; ad1[c] = C.ad1[3 * (size_t)k + c];
        xi[c] = B.xi[3 * (size_t)k + c]; vi[c] = B.vi[3 * (size_t)k + c];
    }
    const double d = hd_correct_core(S.dt[p], a0, ad0, a1, ad1, xi, vi, tn, C.eta, C.dt_max, x1, v1);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        S.x[3 * (size_t)p + c] = x1[c]; S.v[3 * (size_t)p + c] = v1[c];
        S.a[3 * (size_t)p + c] = a1[c]; S.ad[3 * (size_t)p + c] = ad1[c];
    }
    S.t[p] = tn;
    S.dt[p] = d;
    atomicMin(C.dt_min_bits, (unsigned long long)__double_as_longlong(d));
    hd_store_j(C.raw, S, p);
}

// One launch finishes the previous block step (phase 0) and selects the next block.  Phase 1, every thread block: reduce its HD_PER_BLOCK particles to the
// minimum of t + dt and write the particles that attain it, in address order, to its segment of `cand`.
// Phase 2, the LAST thread block to finish (atomic ticket): global minimum over the per-block minima (held in
// shared memory), prefix sum of the counts of the thread blocks that attain it, then the active list = the
// concatenation of their candidate segments, with the fp64 prediction of each i-particle.
constexpr int HD_GATHER_INLINE = 32;
constexpr int HD_MAX_BLOCKS = 2048;     // x HD_PER_BLOCK = 2^21 particles, the library's largest capacity

__global__ void __launch_bounds__(HD_THREADS)
k_hd_select(HdState S, HdBlock B, HdCorr C, int correct_first)
{
    __shared__ double smin[HD_THREADS / 32];
    __shared__ int scnt[HD_THREADS / 32];
    __shared__ int s_last;
    __shared__ double s_bmin[HD_MAX_BLOCKS];
    __shared__ int s_cnt[HD_MAX_BLOCKS], s_off[HD_MAX_BLOCKS];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, b = blockIdx.x, nb = gridDim.x;
    const int p0 = b * HD_PER_BLOCK;
    const double INF = __longlong_as_double(0x7ff0000000000000LL);
    // Phase 0 (correct_first): the corrector of the PREVIOUS block step, owner computes -- this thread block's
    // own particles of that block are entries [boff[b], boff[b] + bcnt[b]) of its active list (written by the
    // previous launch), so no other thread block touches the t, dt this one is about to read.
    if (correct_first) {
        const int base = B.boff[b];
        if (base >= 0) {
            const int cntb = B.bcnt[b];
            const double tprev = *B.d_tnext;
            for (int u = tid; u < cntb; u += HD_THREADS) hd_correct_one(S, B, C, base + u, tprev);
        }
        __syncthreads();
    }
    double tn[HD_PER_BLOCK / HD_THREADS];
    double lmin = INF;
#pragma unroll
    for (int q = 0; q < HD_PER_BLOCK / HD_THREADS; ++q) {
        const int p = p0 + q * HD_THREADS + tid;
        tn[q] = p < S.n ? S.t[p] + S.dt[p] : INF;
        lmin = fmin(lmin, tn[q]);
    }
    const double bm = hd_block_min(lmin, smin);
    // ordered compaction of the particles at the block minimum (order = address = (q, tid))
    int off = 0;
#pragma unroll
    for (int q = 0; q < HD_PER_BLOCK / HD_THREADS; ++q) {
        const bool on = tn[q] == bm;
        const unsigned bal = __ballot_sync(0xffffffffu, on);
        if (lane == 0) scnt[wid] = __popc(bal);
        __syncthreads();
        int before = 0, total = 0;
#pragma unroll
        for (int w = 0; w < HD_THREADS / 32; ++w) {
            const int cw = scnt[w];
            before += w < wid ? cw : 0;
            total += cw;
        }
        if (on) B.cand[p0 + off + before + __popc(bal & ((1u << lane) - 1u))] = p0 + q * HD_THREADS + tid;
        off += total;
        __syncthreads();
    }
    if (tid == 0) {
        B.bmin[b] = bm;
        B.bcnt[b] = off;
    }
    __syncthreads();
    if (tid == 0) {
        fence_acq_rel_gpu();                              // release: this block's minimum, count and candidates (ordered before by the barrier)
        s_last = atomicAdd(B.ticket, 1u) == (unsigned)nb - 1u;
        if (s_last) fence_acq_rel_gpu();                  // acquire: the other blocks' (read with ld.global.cg below)
    }
    __syncthreads();
    if (!s_last) return;

    // ---- last thread block
    double g = INF;
    for (int k = tid; k < nb; k += HD_THREADS) {
        const double v = __ldcg(B.bmin + k);
        s_bmin[k] = v;
        s_cnt[k] = __ldcg(B.bcnt + k);
        g = fmin(g, v);
    }
    const double tnext = hd_block_min(g, smin);          // (its barriers also publish s_bmin / s_cnt)
    int ni = 0;
    if (wid == 0) {                                       // warp 0: offsets of the thread blocks at the minimum, in order
        for (int c0 = 0; c0 < nb; c0 += 32) {
            const int k = c0 + lane;
            const bool hit = k < nb && s_bmin[k] == tnext;
            const int c = hit ? s_cnt[k] : 0;
            int inc = c;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int u = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += u;
            }
            if (k < nb) { s_off[k] = hit ? ni + inc - c : -1; B.boff[k] = s_off[k]; }
            ni += __shfl_sync(0xffffffffu, inc, 31);
        }
        if (lane == 0) scnt[0] = ni;
    }
    __syncthreads();
    ni = scnt[0];
    // small blocks are gathered and predicted right here; for large ones the host, which is told n_i anyway,
    // launches k_hd_gather over all thread blocks (HD_GATHER_INLINE)
    for (int k = 0; k < (ni <= HD_GATHER_INLINE ? nb : 0); ++k) {
        const int base = s_off[k];
        if (base < 0) continue;                           // uniform over the thread block
        const int cntk = s_cnt[k];
        for (int u = tid; u < cntk; u += HD_THREADS) {
            const int p = __ldcg(B.cand + k * HD_PER_BLOCK + u);
            B.act[base + u] = p;
            hd_predict(S, p, tnext, B.xi + 3 * (size_t)(base + u), B.vi + 3 * (size_t)(base + u));
        }
    }
    if (tid == 0) {
        *B.d_ni = ni;
        *B.d_tnext = tnext;
        *B.ticket = 0u;
        hd_notify(B.h_note, tnext, ni, B.seq);
    }
}

// large blocks: thread block k moves its candidates to their place in the active list and predicts them
__global__ void __launch_bounds__(HD_THREADS)
k_hd_gather(HdState S, HdBlock B)
{
    const int k = blockIdx.x;
    const int base = B.boff[k];
    if (base < 0) return;
    const int cntk = B.bcnt[k];
    const double tnext = *B.d_tnext;
    for (int u = threadIdx.x; u < cntk; u += HD_THREADS) {
        const int p = B.cand[k * HD_PER_BLOCK + u];
        B.act[base + u] = p;
        hd_predict(S, p, tnext, B.xi + 3 * (size_t)(base + u), B.vi + 3 * (size_t)(base + u));
    }
}

// first call: forces at t = 0 are in (a1, ad1) for ALL particles -> state, first steps, j-store
__global__ void __launch_bounds__(HD_THREADS)
k_hd_init(HdState S, const double *__restrict__ a1, const double *__restrict__ ad1, double eta_start, double dt_max, char *raw,
          unsigned long long *dt_min_bits)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= S.n) return;
    double a[3], ad[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) { a[k] = a1[3 * (size_t)p + k]; ad[k] = ad1[3 * (size_t)p + k]; S.a[3 * (size_t)p + k] = a[k]; S.ad[3 * (size_t)p + k] = ad[k]; }
    const double na = hd_norm3(a), nad = hd_norm3(ad);
    const double d = hd_pow2_floor(nad > 0 ? eta_start * na / nad : dt_max, dt_max);
    S.dt[p] = d;
    S.t[p] = 0.0;
    atomicMin(dt_min_bits, (unsigned long long)__double_as_longlong(d));
    hd_store_j(raw, S, p);
}

// the corrector alone (the pending block at the end of g6hd_evolve); one thread per particle
__global__ void __launch_bounds__(HD_THREADS)
k_hd_correct(HdState S, HdBlock B, HdCorr C)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= *B.d_ni) return;
    hd_correct_one(S, B, C, k, *B.d_tnext);
}

// ---- shared-time-step variant ("shared or block time steps"; reading 21) --------------------
// every particle takes every step with one common step = the smallest of the per-particle wishes
__global__ void __launch_bounds__(HD_THREADS)
k_hd_min_dt(HdState S, unsigned long long *bits)
{
    __shared__ double smin[HD_THREADS / 32];
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    const double d = hd_block_min(p < S.n ? S.dt[p] : __longlong_as_double(0x7ff0000000000000LL), smin);
    if (threadIdx.x == 0) atomicMin(bits, (unsigned long long)__double_as_longlong(d));
}

// the common step to every particle; the block is everybody, predicted to t + h
__global__ void __launch_bounds__(HD_THREADS)
k_hd_shared_apply(HdState S, HdBlock B, const unsigned long long *bits)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= S.n) return;
    const double h = __longlong_as_double((long long)*bits);
    const double tn = S.t[p] + h;
    S.dt[p] = h;
    B.act[p] = p;
    hd_predict(S, p, tn, B.xi + 3 * (size_t)p, B.vi + 3 * (size_t)p);
    if (p == 0) {
        *B.d_ni = S.n;
        *B.d_tnext = tn;
        hd_notify(B.h_note, tn, S.n, B.seq);
    }
}

__global__ void k_hd_set_u64(unsigned long long *p, unsigned long long v) { *p = v; }

// shared steps need every particle at the system time: count those that are not (bits[0] += 1 each)
__global__ void __launch_bounds__(HD_THREADS)
k_hd_count_unsynchronised(HdState S, double t, unsigned long long *count)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    const bool off = p < S.n && S.t[p] != t;
    const unsigned bal = __ballot_sync(0xffffffffu, off);
    if ((threadIdx.x & 31) == 0 && bal) atomicAdd(count, (unsigned long long)__popc(bal));
}

__global__ void k_hd_iota(int *act, int n)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p < n) act[p] = p;
}

// Eq. 1-2 of every particle to the time tn (state read-out)
__global__ void __launch_bounds__(HD_THREADS)
k_hd_predict_all(HdState S, double tn, double *__restrict__ xo, double *__restrict__ vo)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= S.n) return;
    hd_predict(S, p, tn, xo + 3 * (size_t)p, vo + 3 * (size_t)p);
}

}  // namespace g6
