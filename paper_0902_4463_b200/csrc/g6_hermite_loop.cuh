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
//  * the CTAs meet through SELF-VALIDATING 8-byte words {32 bits of payload, 32-bit step number} written and polled with
//    single 64-bit accesses (single-copy atomic): the data is its own flag, so an exchange costs one store and one L2 round
//    trip, with no separate barrier and no fence (the protocol NCCL calls LL).  A block step has two such exchanges:
//      A  per owned tile: (min of t + dt, count at the min, slots of the first HL_INLINE particles at the min)  -> records
//         every CTA polls all records: t_next = global min, n_i, the active list in increasing address.  If no tile holds more
//         than HL_INLINE active particles EVERY CTA reads the Hermite state of all n_i particles and predicts them itself in
//         fp64 (Eq. 1-2): no second exchange.  Otherwise the owners predict into the global i-block and the CTAs
//         meet at a flag barrier.
//      B  i-block -> double-single in shared memory, Eq. 1-2 of the resident j-particles (same routine as k_predict), then all
//         pairs with the packed, checked pair code of the block-step kernel (pair2_checked; Eq. 3).  Lanes of a warp
//         = (i-particle, j-sub-range): "several threads share an i and split the j"; the lanes of one i are
//         summed by a fixed shuffle tree once per step, then the warps and the CTAs in fixed order in fp64 (reading 9):
//         bit-reproducible.  One partial per (i, CTA)                                                          -> chunks
//      C  the owner of each active particle polls its G partials (a warp per particle, summed in the order of k_combine_wide),
//         runs the corrector, the Aarseth step and the power-of-two rule (hd_correct_core), updates its resident tile.
//    Records are double-buffered by step parity (an owner without active particles may run one step ahead of a slow poller);
//    partials need no second buffer (a CTA writes those of step s + 1 only after every CTA has published its records of s + 1,
//    i.e. has finished step s).
//  * a block with n_i > max_i is selected and predicted by its owners and handed to the host, which runs the library's sweep
//    path on it (hd_force) and re-enters the loop.
// The nearest neighbour is not tracked (the Hermite driver does not use it).
#pragma once
#include "g6_block_step.cuh"
#include "g6_hermite_dev.cuh"

namespace g6 {

constexpr int HL_THREADS = 512;
constexpr int HL_NW = HL_THREADS / 32;
constexpr int HL_KMAX = 4;                    // resident raw tiles per CTA
constexpr int HL_MAX_I = 768;                 // largest block the loop can step itself
constexpr int HL_MAX_G = 148;                 // CTAs (one per SM)
constexpr int HL_MAX_TILES = HL_MAX_G * HL_KMAX;
constexpr int HL_INLINE = 8;                  // active particles per tile that travel inside the tile's record
constexpr int HL_REC_WORDS = 6;               // tmin lo, tmin hi, count, slots 0-3, slots 4-7, (pad): three 16-byte stores / loads
constexpr int HL_CHUNK_WORDS = 14;            // 7 fp64 sums = 14 halves
static_assert(true, "");
constexpr int HL_CQ = 3;                      // particles whose partials an owner gathers at a time (staged in the idle wsum)
constexpr int HL_CPOLL = 6;                   // 16-byte word pairs a thread polls per round: the HL_CQ x 7 x G pairs of one gather are all in flight together

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
    long long inline_steps;  // steps whose i-block every CTA predicted itself (no second exchange)
};

struct HlArgs {
    HdState S;
    HdBlock B;
    HdCorr C;
    double *a1, *ad1, *pot;        // forces of the current block (= C.a1, C.ad1), writable
    int ntiles, nj;
    double t_sys, t_end;
    long long max_steps;
    int max_i;
    float eps2;
    int ds;
    unsigned int gen0;             // step numbers of this launch are gen0 + 1, gen0 + 2, ... (never 0, never reused)
    unsigned long long *rec;       // [2][G][ntiles][HL_REC_WORDS]   tile records: double-buffered by step parity, one copy per consumer CTA
    unsigned long long *chunk;     // [max_i][G][HL_CHUNK_WORDS]  partial forces: the 14 words of one (particle, CTA) are contiguous (seven 16-byte stores)
    unsigned int *flag;            // [G] flag barrier of the non-inline path
    HlStatus *status;              // device-visible (mapped host memory)
    unsigned long long *prof;      // [32] PROF build only: summed clock64() intervals between the marks (see HL_MK), steps with n_i < 8
};

struct HlSmem {
    alignas(16) char raw[HL_KMAX][RAW_TILE_BYTES];      // the CTA's own raw j-tiles, resident
    alignas(16) float pred[HL_KMAX][TILE_FLOATS];       // their Eq. 1-2 predictions at the block time
    double tnext[HL_KMAX][JT];                          // t + dt of the own particles (+inf past the end)
    float ipart[HL_MAX_I][9];                           // i-block: hi[3], lo[3], v[3]
    int iidx[HL_MAX_I];                                 // ... and the particles' addresses (= indices)
    double wsum[HL_NW][32][7];                          // per-warp sums of one i-chunk
    double s_tm[HL_MAX_TILES];                          // the tile records of this step
    int s_tc[HL_MAX_TILES];
    int s_off[HL_MAX_TILES];
    unsigned int s_sl[HL_MAX_TILES][2];
    int own_k[HL_KMAX * JT], own_l[HL_KMAX * JT];       // my active particles: position in the active list, slot kk * JT + l
    double own_st[HL_KMAX * HL_INLINE][20];             // inline path: xi[3] vi[3] a0[3] ad0[3] h, of my active particles
    double red[HL_NW][2];
    unsigned int bal[HL_KMAX][JT / 32];
    unsigned int recw[HL_KMAX][HL_REC_WORDS];
    int nown_prev;
    long long mk[32];                                   // PROF build: clock64() marks of thread 0
    int mk_open;
    double tmin[HL_KMAX];
    double gmin;
    int ni, nown, inl;
};
static_assert(sizeof(HlSmem) <= 232448, "loop kernel shared memory");
static_assert(sizeof(double) * HL_NW * 32 * 7 >= sizeof(unsigned int) * HL_CQ * HL_CHUNK_WORDS * HL_MAX_G, "chunk staging fits in wsum");

// acquire-release fence at device scope.  (__threadfence() is the sequentially consistent fence and, on sm_100, also invalidates the
// whole L1: MEMBAR.SC.GPU + CCTL.IVALL, measured several microseconds per step with the exchange stores in flight.)
__device__ __forceinline__ void hl_fence() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }

__device__ __forceinline__ void hl_store_word(unsigned long long *p, unsigned int payload, unsigned int gen)
{
    const unsigned long long v = (unsigned long long)payload | ((unsigned long long)gen << 32);
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long hl_load_word(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
// two consecutive words (16-byte aligned) with one instruction; each 8-byte half is single-copy atomic, which is all the
// self-validating words need
__device__ __forceinline__ void hl_store_word2(unsigned long long *p, unsigned int pay0, unsigned int pay1, unsigned int gen)
{
    const unsigned long long g = (unsigned long long)gen << 32;
    asm volatile("st.relaxed.gpu.global.v2.u64 [%0], {%1, %2};" ::"l"(p), "l"(g | pay0), "l"(g | pay1) : "memory");
}
__device__ __forceinline__ void hl_load_word2(const unsigned long long *p, unsigned long long &a, unsigned long long &b)
{
    asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "l"(p) : "memory");
}
// spin until the N words p[0], p[stride], ... all carry step number `gen` (all N loads of a round are in flight together);
// a protocol error fails the launch instead of hanging the device
template <int N>
__device__ __forceinline__ void hl_wait_words(const unsigned long long *p, size_t stride, unsigned int gen, unsigned int (&out)[N])
{
    unsigned int spins = 0;
    for (;;) {
        unsigned long long v[N];
#pragma unroll
        for (int k = 0; k < N; ++k) v[k] = hl_load_word(p + k * stride);
        bool ok = true;
#pragma unroll
        for (int k = 0; k < N; ++k) { ok = ok && (unsigned int)(v[k] >> 32) == gen; out[k] = (unsigned int)v[k]; }
        if (ok) return;
        if (++spins > (1u << 26)) __trap();
    }
}

// flag barrier (non-inline path only): every CTA publishes the step number, everybody polls all flags
__device__ __forceinline__ void hl_flag_barrier(unsigned int *flag, unsigned int G, unsigned int gen)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        hl_fence();
        asm volatile("st.volatile.global.u32 [%0], %1;" ::"l"(flag + blockIdx.x), "r"(gen) : "memory");
    }
    for (unsigned int s = threadIdx.x; s < G; s += HL_THREADS) {
        unsigned int v, spins = 0;
        do {
            asm volatile("ld.volatile.global.u32 %0, [%1];" : "=r"(v) : "l"(flag + s) : "memory");
            if (++spins > (1u << 26)) __trap();
        } while (v != gen);
        hl_fence();
    }
    __syncthreads();
}

// particle p's new Hermite state -> slot l of a raw tile (shared memory or the j-store): what hd_store_j writes
__device__ __forceinline__ void hl_store_tile(char *T, int l, int p, const double *x, const double *v, const double *a, const double *ad, double t, float m)
{
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        raw_x(T, k, l) = x[k];
        raw_v(T, k, l) = (float)v[k];
        raw_a2(T, k, l) = (float)(a[k] / 2);
        raw_j6(T, k, l) = (float)(ad[k] / 6);
    }
    raw_t(T, l) = t;
    raw_m(T, l) = m;
    raw_idx(T, l) = p;
}

// the record of one tile from the eight ballots of "slot is at the tile's minimum": count and the first HL_INLINE slots (increasing)
__device__ __forceinline__ void hl_make_record(const unsigned int *bal, double tmin, unsigned int *recw)
{
    int c = 0;
    unsigned int sl[2] = {0u, 0u};
    for (int q = 0; q < JT / 32; ++q) {
        unsigned b = bal[q];
        while (b) {
            const int l = __ffs(b) - 1;
            b &= b - 1;
            if (c < HL_INLINE) sl[c >> 2] |= (unsigned)(32 * q + l) << (8 * (c & 3));
            ++c;
        }
    }
    const unsigned long long tb = (unsigned long long)__double_as_longlong(tmin);
    recw[0] = (unsigned int)tb;
    recw[1] = (unsigned int)(tb >> 32);
    recw[2] = (unsigned int)c;
    recw[3] = sl[0];
    recw[4] = sl[1];
    recw[5] = 0u;
}

// PROF: thread 0 of every CTA also takes clock64() marks along the step (HlStatus::ph, ::own); a build of its own (env
// G6_HD_LOOP_PROFILE) because the marks cost registers the production loop does not have to spare
template <bool NEWTON, bool PROF = false>
__global__ void __launch_bounds__(HL_THREADS, 1)
k_hd_loop(const HlArgs A)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    HlSmem &sm = *reinterpret_cast<HlSmem *>(smem_raw);
    const unsigned FULL = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int slot = tid & (JT - 1), half = tid / JT, ws = slot >> 5;       // a particle slot and which half of the CTA works on it
    const int G = gridDim.x, cta = blockIdx.x;
    const double INF = __longlong_as_double(0x7ff0000000000000LL);
    const int Kc = cta < A.ntiles ? (A.ntiles - cta + G - 1) / G : 0;       // my tiles: cta, cta + G, ...

    // ---- load my tiles and the t + dt of their particles
    for (int kk = 0; kk < Kc; ++kk) {
        const int4 *src = reinterpret_cast<const int4 *>(A.C.raw + (size_t)(cta + kk * G) * RAW_TILE_BYTES);
        int4 *dst = reinterpret_cast<int4 *>(sm.raw[kk]);
        for (int q = tid; q < RAW_TILE_BYTES / 16; q += HL_THREADS) dst[q] = __ldcg(src + q);
        if (half == 0) {
            const int p = (cta + kk * G) * JT + slot;
            sm.tnext[kk][slot] = p < A.S.n ? __ldcg(A.S.t + p) + __ldcg(A.S.dt + p) : INF;
        }
    }
    __syncthreads();

    if (tid == 0) sm.nown_prev = 0;
    bool rescan = true;                    // my tiles' records must be recomputed (start; after I corrected particles)
    double t_sys = A.t_sys;
    long long steps = 0, npart = 0, n_inline = 0;
    long long hist = 0, hist_ns = 0;       // thread b < 64 of CTA 0 counts bin b
    unsigned long long t_step = 0;
    if (cta == 0) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_step));
    int reason = HL_END, ni_next = 0, ni_last = 0;
    double t_big = 0.0;
    // PROF: thread 0 of every CTA marks the clock along the step: 0-10 the step as every CTA walks it (summed for CTA 0), 16-25 the
    // chain of a CTA that owns an active particle (gather .. publish of the next step), summed over all owners
#define HL_MK(q) do { if (PROF && tid == 0) sm.mk[q] = clock64(); } while (0)
    if (PROF && tid == 0) sm.mk_open = 0;
    const float2 eps2 = dup(A.eps2);
    // the unchecked pair code needs s2 > 0 for every pair: a normal positive binary32 eps2 (as for the sweep kernel)
    const bool fast_ok = A.eps2 >= 4.0f * 1.17549435e-38f && A.eps2 < __builtin_huge_valf();
    const float2 eps2s = dup(pair_scale<NEWTON>() * A.eps2);
    const double kP = NEWTON ? 0.5 * sqrt((double)FOUR_THIRDS) : sqrt((double)THIRD), kA = kP * kP * kP;

    // (min, count, first slots at the min) of t + dt of my one resident tile -> sm.recw[0], sm.bal[0]; one whole warp
    const auto rescan_tile0 = [&]() {
        // t + dt >= 0 (or +inf): the doubles order like their bit patterns, and the minimum of 64-bit patterns over the
        // warp is two 32-bit warp reductions (high words, then the low words of the lanes at the high minimum)
        unsigned long long v[JT / 32], m = ~0ull;     // lane holds the slots lane, lane + 32, ...
#pragma unroll
        for (int r = 0; r < JT / 32; ++r) { v[r] = (unsigned long long)__double_as_longlong(sm.tnext[0][32 * r + lane]); m = v[r] < m ? v[r] : m; }
        const unsigned int mh = __reduce_min_sync(FULL, (unsigned int)(m >> 32));
        const unsigned int ml = __reduce_min_sync(FULL, (unsigned int)(m >> 32) == mh ? (unsigned int)m : 0xffffffffu);
        m = ((unsigned long long)mh << 32) | ml;
        unsigned int bal[JT / 32];
#pragma unroll
        for (int r = 0; r < JT / 32; ++r) {
            bal[r] = __ballot_sync(FULL, v[r] == m);
            if (lane == 0) sm.bal[0][r] = bal[r];      // (the non-inline path of phase A reads them)
        }
        // every lane has the ballots: the record in registers, no round trip through shared memory
        if (lane == 0) hl_make_record(bal, __longlong_as_double((long long)m), sm.recw[0]);
        __syncwarp();
    };
    bool pre_scanned = false;              // an idle warp rescanned my tile at the end of phase C (Kc == 1, I corrected particles)
    for (;;) {
        if (!(t_sys < A.t_end)) { reason = HL_END; break; }
        if (A.max_steps > 0 && steps >= A.max_steps) { reason = HL_STEPS; break; }
        const unsigned int gen = A.gen0 + 1u + (unsigned int)steps;
        HL_MK(0);
        // this step's records: [consumer CTA][tile][word] -- every consumer polls its OWN copy (a word polled by all CTAs at once
        // is a hot spot in its L2 slice: the publisher's store then queues behind hundreds of loads, measured 3-5 us)
        unsigned long long *rec = A.rec + (size_t)(gen & 1u) * G * A.ntiles * HL_REC_WORDS;

        // ================= phase A: per own tile (min, count, first slots at the min) of t + dt -> its record
        // Only a CTA that corrected particles in the last step (or starts) has anything to recompute; the others republish what
        // they had under the new step number.  Several resident tiles: the whole CTA rescans (its two halves take the tiles of
        // their parity, a warp holds 32 consecutive slots); one tile: warp 0 does it alone, with no block-wide barrier.
        if (rescan && Kc > 1) {
            for (int kk = half; kk < Kc; kk += 2) {
                double m = sm.tnext[kk][slot];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) m = fmin(m, __shfl_xor_sync(FULL, m, o));
                if (lane == 0) sm.red[w][kk >> 1] = m;
            }
            __syncthreads();
            for (int kk = half; kk < Kc; kk += 2) {
                double m = sm.red[half * (JT / 32)][kk >> 1];
#pragma unroll
                for (int q = 1; q < JT / 32; ++q) m = fmin(m, sm.red[half * (JT / 32) + q][kk >> 1]);
                const unsigned b = __ballot_sync(FULL, sm.tnext[kk][slot] == m);
                if (lane == 0) sm.bal[kk][ws] = b;
                if (slot == 0) sm.tmin[kk] = m;
            }
            __syncthreads();
            if (tid < Kc) hl_make_record(sm.bal[tid], sm.tmin[tid], sm.recw[tid]);
            __syncthreads();
        }
        if (w == 0) {
            // everything from here to the barrier below is warp 0's: rescan (one tile), publish, poll, select
            if (rescan && Kc == 1 && !pre_scanned) rescan_tile0();
            // (release: the owners' warps fenced after their state stores in phase C of the last step, before its closing barrier)
            HL_MK(23);
            HL_MK(24);
            for (int kk = 0; kk < Kc; ++kk) {
                unsigned int rw[HL_REC_WORDS];
#pragma unroll
                for (int wd = 0; wd < HL_REC_WORDS; ++wd) rw[wd] = sm.recw[kk][wd];
                for (int c = lane; c < G; c += 32) {                 // consumer c's private copy
                    unsigned long long *r = rec + ((size_t)c * A.ntiles + (cta + kk * G)) * HL_REC_WORDS;
#pragma unroll
                    for (int wd = 0; wd < HL_REC_WORDS; wd += 2) hl_store_word2(r + wd, rw[wd], rw[wd + 1], gen);
                }
            }

            HL_MK(1);
            HL_MK(25);
            if (PROF && tid == 0 && sm.mk_open) {
                for (int q = 16; q < 25; ++q) atomicAdd(A.prof + q, (unsigned long long)(sm.mk[q + 1] - sm.mk[q]));
                atomicAdd(A.prof + 31, 1ull);
                sm.mk_open = 0;
            }
            // poll every tile's record (my private copy): lane takes the tiles lane, lane + 32, ..., four at a time
            double m = INF;
            for (int g0 = 0; g0 < A.ntiles; g0 += 128) {
                bool done[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) done[u] = g0 + lane + 32 * u >= A.ntiles;
                unsigned int spins = 0;
                for (;;) {
                    unsigned long long v[4][HL_REC_WORDS];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        if (!done[u]) {
                            const unsigned long long *r = rec + ((size_t)cta * A.ntiles + g0 + lane + 32 * u) * HL_REC_WORDS;
#pragma unroll
                            for (int k = 0; k < HL_REC_WORDS; k += 2) hl_load_word2(r + k, v[u][k], v[u][k + 1]);
                        }
                    }
                    bool all = true;
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        if (!done[u]) {
                            bool ok = true;
#pragma unroll
                            for (int k = 0; k < HL_REC_WORDS; ++k) ok = ok && (unsigned int)(v[u][k] >> 32) == gen;
                            if (ok) {
                                const int T = g0 + lane + 32 * u;
                                const double tm = __longlong_as_double((long long)((v[u][1] << 32) | (v[u][0] & 0xffffffffull)));
                                sm.s_tm[T] = tm;
                                sm.s_tc[T] = (int)(unsigned int)v[u][2];
                                sm.s_sl[T][0] = (unsigned int)v[u][3];
                                sm.s_sl[T][1] = (unsigned int)v[u][4];
                                m = fmin(m, tm);
                                done[u] = true;
                            } else {
                                all = false;
                            }
                        }
                    }
                    if (all) break;
                    if (++spins > (1u << 26)) __trap();
                }
            }
            HL_MK(2);
            // No acquire fence here.  Everything read after this point that another CTA wrote (the Hermite state of the active
            // particles, the i-block) is read with ld.global.cg / ld.volatile, i.e. from L2, by instructions ISSUED after the poll
            // loop has seen the records (the loop's exit depends on the loaded words); the writers made that data visible before
            // their records (fence.acq_rel.gpu in front of the record stores).  A fence here has to wait for this warp's own
            // G x 5 record stores to be acknowledged and cost 3-4 us per block step (measured with the phase marks below).
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) m = fmin(m, __shfl_xor_sync(FULL, m, o));
            HL_MK(3);
            // t_next = m; offsets of the tiles in the active list (tile order = increasing address); n_i.  Lane l takes the
            // tiles [l R, l R + R): its own running count, one scan over the lanes, and it writes the offsets and (inline path)
            // the addresses of its tiles' active particles
            __syncwarp();                                     // the polling lanes' s_tm / s_tc / s_sl
            const int R = (A.ntiles + 31) >> 5;
            const unsigned long long mb = (unsigned long long)__double_as_longlong(m);        // bit patterns compare like the times
            const unsigned long long *tmb = reinterpret_cast<const unsigned long long *>(sm.s_tm);
            int mine = 0, over = 0;
            for (int r0 = 0; r0 < R; r0 += 4) {               // four tiles' loads in flight together
                unsigned long long tb[4];
                int tc[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int T = min(lane * R + r0 + u, A.ntiles - 1);
                    tb[u] = tmb[T];
                    tc[u] = sm.s_tc[T];
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int c = (r0 + u < R && lane * R + r0 + u < A.ntiles && tb[u] == mb) ? tc[u] : 0;
                    over |= c > HL_INLINE;
                    mine += c;
                }
            }
            HL_MK(11);
            int inc = mine;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int u = __shfl_up_sync(FULL, inc, o);
                if (lane >= o) inc += u;
            }
            const int run = __shfl_sync(FULL, inc, 31);
            over = __any_sync(FULL, over);
            const bool inl_w = !over && run <= A.max_i;
            HL_MK(12);
            {
                int base = inc - mine;
                for (int r0 = 0; r0 < R; r0 += 4) {
                    unsigned long long tb[4];
                    int tc[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int T = min(lane * R + r0 + u, A.ntiles - 1);
                        tb[u] = tmb[T];
                        tc[u] = sm.s_tc[T];
                    }
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int T = lane * R + r0 + u;
                        if (r0 + u < R && T < A.ntiles) {
                            const bool hit = tb[u] == mb;
                            const int c = hit ? tc[u] : 0;
                            sm.s_off[T] = hit ? base : -1;
                            if (inl_w)
                                for (int q = 0; q < c; ++q) sm.iidx[base + q] = T * JT + (int)((sm.s_sl[T][q >> 2] >> (8 * (q & 3))) & 0xffu);
                            base += c;
                        }
                    }
                }
            }
            __syncwarp();
            HL_MK(13);
            if (lane == 0) {
                sm.ni = run; sm.gmin = m; sm.inl = inl_w;
                if (inl_w) {
                    // my active particles: (position in the list, slot), tile by tile
                    int nown = 0;
                    for (int kk = 0; kk < Kc; ++kk) {
                        const int T = cta + kk * G, base = sm.s_off[T];
                        if (base < 0) continue;
                        for (int r = 0; r < sm.s_tc[T]; ++r) {
                            sm.own_k[nown] = base + r;
                            sm.own_l[nown] = kk * JT + (int)((sm.s_sl[T][r >> 2] >> (8 * (r & 3))) & 0xffu);
                            ++nown;
                        }
                    }
                    sm.nown = nown;
                }
            }
        }
        HL_MK(4);
        __syncthreads();
        HL_MK(5);
        const double tn = sm.gmin;
        const int ni = sm.ni;
        const bool big = ni > A.max_i, inl = sm.inl != 0;

        if (inl) {
            // ---- every CTA predicts all n_i particles itself (fp64 Eq. 1-2), straight into its i-block: the lower half of the
            // CTA; the upper half predicts the resident j-particles meanwhile (below)
            for (int k = tid; k < ni && tid < HL_THREADS / 2; k += HL_THREADS / 2) {
                const int p = sm.iidx[k];
                const double tp = __ldcg(A.S.t + p);
                const double h = tn - tp, h2 = h * h / 2, h3 = h * h * h / 6;
                const int T = p / JT;
                const bool mine = (T % G) == cta;
                double xi[3], vi[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const double x = __ldcg(A.S.x + 3 * (size_t)p + c), v = __ldcg(A.S.v + 3 * (size_t)p + c);
                    const double a = __ldcg(A.S.a + 3 * (size_t)p + c), ad = __ldcg(A.S.ad + 3 * (size_t)p + c);
                    xi[c] = x + v * h + a * h2 + ad * h3;              // same expressions as hd_predict
                    vi[c] = v + a * h + ad * h2;
                    float hi, lo;
                    ds_split(xi[c], hi, lo);
                    sm.ipart[k][c] = hi;
                    sm.ipart[k][3 + c] = A.ds ? lo : 0.0f;
                    sm.ipart[k][6 + c] = (float)vi[c];
                    if (mine) {
                        double *st = sm.own_st[(T / G) * HL_INLINE + (k - sm.s_off[T])];
                        st[c] = xi[c]; st[3 + c] = vi[c]; st[6 + c] = a; st[9 + c] = ad;
                    }
                    if (cta == 0) { A.B.xi[3 * (size_t)k + c] = xi[c]; A.B.vi[3 * (size_t)k + c] = vi[c]; }     // read-back only
                }
                if (mine) sm.own_st[(T / G) * HL_INLINE + (k - sm.s_off[T])][12] = A.S.dt[p];      // the stored step (= h when dt_max is a power of two)
                if (cta == 0) A.B.act[k] = p;
            }
        } else {
            // ---- owners: active particles of my tiles, in address order, predicted in fp64 into the global i-block
            int nown = 0;
            for (int kk = 0; kk < Kc; ++kk) {
                const int T = cta + kk * G;
                const int base = sm.s_off[T];
                if (base < 0) continue;                                     // uniform over the CTA
                if (half == 0) {
                    const bool on = sm.tnext[kk][slot] == tn;
                    int before = 0;
                    for (int q = 0; q < ws; ++q) before += __popc(sm.bal[kk][q]);
                    if (on) {
                        const int r = before + __popc(sm.bal[kk][ws] & ((1u << lane) - 1u));
                        const int k = base + r, p = T * JT + slot;
                        A.B.act[k] = p;
                        hd_predict(A.S, p, tn, A.B.xi + 3 * (size_t)k, A.B.vi + 3 * (size_t)k);
                        if (!big) { sm.own_k[nown + r] = k; sm.own_l[nown + r] = kk * JT + slot; }
                    }
                }
                nown += sm.s_tc[T];
            }
            if (tid == 0) sm.nown = nown;
            if (big) { reason = HL_BIG; ni_next = ni; t_big = tn; break; }   // the kernel's end publishes the i-block
            hl_flag_barrier(A.flag, G, gen);
            for (int q = tid; q < ni * 3; q += HL_THREADS) {
                const int i = q / 3, c = q % 3;
                float hi, lo;
                ds_split(__ldcg(A.B.xi + q), hi, lo);
                sm.ipart[i][c] = hi;
                sm.ipart[i][3 + c] = A.ds ? lo : 0.0f;
                sm.ipart[i][6 + c] = (float)__ldcg(A.B.vi + q);
            }
            for (int i = tid; i < ni; i += HL_THREADS) sm.iidx[i] = __ldcg(A.B.act + i);
        }

        // ================= phase B: my j-particles -> Eq. 1-2 at tn, then all pairs
        for (int q = inl ? tid - HL_THREADS / 2 : tid; q >= 0 && q < Kc * JT; q += inl ? HL_THREADS / 2 : HL_THREADS) {
            const int kk = q / JT, l = q % JT;
            char *R = sm.raw[kk];
            float *Pj = sm.pred[kk];
            const float dt = (float)(tn - raw_t(R, l));
#pragma unroll
            for (int k = 0; k < 3; ++k)
                predict_coord(dt, raw_x(R, k, l), raw_v(R, k, l), raw_a2(R, k, l), raw_j6(R, k, l), A.ds,
                              Pj[(F_XH + k) * JT + l], Pj[(F_XL + k) * JT + l], Pj[(F_V + k) * JT + l]);
            Pj[F_M * JT + l] = raw_m(R, l);
        }
        __syncthreads();

        HL_MK(6);
        // The pairs.  i-particles in chunks of 32, C = 1, 2, .. 16 chunks at a time; a chunk is worked on by HL_NW / C warps, each
        // taking a j-slice of JT C / HL_NW particles of every tile (small blocks: one chunk, 16 slices of 16 j; 512 particles:
        // 16 chunks at once, every warp sweeps whole tiles and no two warps share an i-particle).  Inside a warp the lanes are
        // 2^lg i-particles x 2^(5 - lg) j-sub-ranges (lg >= 2: every lane has whole packed pairs).  FP32 sums run over one
        // tile slice (<= 256 j) and are folded into fp64 (reading 9); the lanes of one i-particle are then added by a
        // fixed shuffle tree, the slices in slice order, the CTAs in CTA order (phase C): bit-reproducible.
        {
            const int nch = (ni + 31) / 32;
            // C chunks at a time, each by HL_NW / C warps: a pass costs about C + 1/2 (in sixteenths of a tile per warp, plus its
            // barriers and partial sums), so take the C that minimises passes x (C + 1/2); ties go to the larger C (fewer barriers).
            // 24 chunks: three passes of 8 instead of 16 + 8; 6 chunks: three passes of 2 instead of one pass that idles a quarter
            int C = 1;
            {
                int best = 1 << 30;
                for (int c = 1; c <= HL_NW; c <<= 1) {
                    const int cost = ((nch + c - 1) / c) * (2 * c + 1);
                    if (cost <= best) { best = cost; C = c; }
                }
            }
            const int nsl = HL_NW / C, cw = w / nsl, sw = w % nsl, jper = JT / nsl;
            for (int r0 = 0; r0 < nch; r0 += C) {
                const int c0 = (r0 + cw) * 32;
                const int nic = max(0, min(32, ni - c0));
                int lg = 2;
                while ((1 << lg) < nic) ++lg;
                const int pw = 1 << lg, jn = (jper * pw) >> 5;          // j-particles per lane and tile
                const int ii = lane & (pw - 1), jsub = lane >> lg;
                const bool act = ii < nic;
                double acc7[7] = {0, 0, 0, 0, 0, 0, 0};
                IPart I;
                int my = -1;
                if (act) {
#pragma unroll
                    for (int k = 0; k < 3; ++k) {
                        I.nxh[k] = dup(-sm.ipart[c0 + ii][k]);
                        I.nxl[k] = dup(-sm.ipart[c0 + ii][3 + k]);
                        I.nv[k] = dup(-sm.ipart[c0 + ii][6 + k]);
                    }
                    my = sm.iidx[c0 + ii];
                }
                for (int kk = 0; kk < Kc; ++kk) {
                    // Self-exclusion hoisted to tile level, as in the sweep kernel: a warp takes the checked pair code only on
                    // the tile that holds one of its i-particles (addresses are indices here) or on the ragged last tile
                    const int T = cta + kk * G;
                    const bool checked = !fast_ok || T * JT + JT > A.nj || __any_sync(FULL, act && my / JT == T);
                    if (!act) continue;
#pragma unroll
                    for (int k = 0; k < 3; ++k) { I.a[k] = dup(0.0f); I.j[k] = dup(0.0f); }
                    I.p = dup(0.0f);
                    const float *Pj = sm.pred[kk];
                    const int *JX = reinterpret_cast<const int *>(sm.raw[kk] + RAW_IDX);
                    const int jl0 = jper * sw + jsub * jn;
                    const int ja0 = T * JT + jl0;
                    if (checked) {
#pragma unroll 2
                        for (int q = 0; q < jn; q += 2) {
                            const int jl = jl0 + q, ja = ja0 + q;
                            float2 f[NF];
#pragma unroll
                            for (int k = 0; k < NF; ++k) f[k] = *reinterpret_cast<const float2 *>(Pj + k * JT + jl);
                            const int2 jx = *reinterpret_cast<const int2 *>(JX + jl);
                            float2 r2;
                            pair2_checked<NEWTON>(I, f[0], f[1], f[2], f[3], f[4], f[5], f[6], f[7], f[8], f[9], eps2,
                                                  (ja < A.nj) && (jx.x != my), (ja + 1 < A.nj) && (jx.y != my), r2);
                        }
#pragma unroll
                        for (int k = 0; k < 3; ++k) {
                            acc7[k] += (double)I.a[k].x + (double)I.a[k].y;
                            acc7[3 + k] += (double)I.j[k].x + (double)I.j[k].y;
                        }
                        acc7[6] -= (double)I.p.x + (double)I.p.y;
                    } else {
                        // the sweep kernel's pair code (no per-pair test, Newton step in three instructions on the scaled sigma);
                        // its sums come out scaled by (y s) and (y s)^3, undone here in fp64 with the binary32 scale
#pragma unroll 2
                        for (int q = 0; q < jn; q += 2) {
                            const int jl = jl0 + q;
                            float2 f[NF];
#pragma unroll
                            for (int k = 0; k < NF; ++k) f[k] = *reinterpret_cast<const float2 *>(Pj + k * JT + jl);
                            float2 r2;
                            pair2<NEWTON>(I, f[0], f[1], f[2], f[3], f[4], f[5], f[6], f[7], f[8], f[9], eps2s, r2);
                        }
#pragma unroll
                        for (int k = 0; k < 3; ++k) {
                            acc7[k] += kA * ((double)I.a[k].x + (double)I.a[k].y);
                            acc7[3 + k] += kA * ((double)I.j[k].x + (double)I.j[k].y);
                        }
                        acc7[6] -= kP * ((double)I.p.x + (double)I.p.y);
                    }
                }
                for (int o = pw; o < 32; o <<= 1) {
#pragma unroll
                    for (int k = 0; k < 7; ++k) acc7[k] += __shfl_xor_sync(FULL, acc7[k], o);
                }
                HL_MK(7);
                if (lane < pw) {
#pragma unroll
                    for (int k = 0; k < 7; ++k) sm.wsum[w][lane][k] = acc7[k];
                }
                __syncthreads();
                HL_MK(8);
                // the slices of every chunk in slice order: one partial per (i, CTA), published as 14 self-validating words
                for (int q = tid; q < C * 32 * 7; q += HL_THREADS) {
                    const int cq = q / (32 * 7), i = (q / 7) % 32, k = q % 7;
                    const int gi = (r0 + cq) * 32 + i;
                    if (gi < ni) {
                        double sv = sm.wsum[cq * nsl][i][k];
                        for (int u = 1; u < nsl; ++u) sv += sm.wsum[cq * nsl + u][i][k];
                        const unsigned long long b = (unsigned long long)__double_as_longlong(sv);
                        hl_store_word2(A.chunk + ((size_t)gi * G + cta) * HL_CHUNK_WORDS + 2 * k, (unsigned int)b, (unsigned int)(b >> 32), gen);
                    }
                }
                __syncthreads();
            }
        }

        // ================= phase C: owners poll the G partials of their particles (fixed order), correct, update the resident tile
        // The partials of HL_CQ particles at a time: every thread polls its share of their nq x 14 x G words (all loads of a round in
        // flight together: one L2 round trip after the last writer), the payloads go to shared memory (the idle wsum), then one
        // warp per particle adds them in fixed order.
        HL_MK(9);
        const int nown = sm.nown;
        HL_MK(16);
        unsigned int *stage = reinterpret_cast<unsigned int *>(&sm.wsum[0][0][0]);       // [HL_CQ][14][G]
        for (int q0 = 0; q0 < nown; q0 += HL_CQ) {
            const int nq = min(HL_CQ, nown - q0);
            const int perq = (HL_CHUNK_WORDS / 2) * G, npairs = nq * perq;          // 16-byte pairs: (CTA, component) of each particle
            for (int e0 = 0; e0 < npairs; e0 += HL_THREADS * HL_CPOLL) {
                unsigned int spins = 0;
                bool done[HL_CPOLL];
#pragma unroll
                for (int r = 0; r < HL_CPOLL; ++r) done[r] = e0 + r * HL_THREADS + tid >= npairs;
                for (;;) {
                    unsigned long long v[HL_CPOLL][2];
#pragma unroll
                    for (int r = 0; r < HL_CPOLL; ++r) {
                        const int e = e0 + r * HL_THREADS + tid;
                        const int qq = (e >= perq) + (e >= 2 * perq);           // which of the <= HL_CQ particles (no division on this path)
                        if (!done[r]) hl_load_word2(A.chunk + ((size_t)sm.own_k[q0 + qq] * perq + (e - qq * perq)) * 2, v[r][0], v[r][1]);
                    }
                    bool all = true;
#pragma unroll
                    for (int r = 0; r < HL_CPOLL; ++r) {
                        if (!done[r]) {
                            if ((unsigned int)(v[r][0] >> 32) == gen && (unsigned int)(v[r][1] >> 32) == gen) {
                                *reinterpret_cast<uint2 *>(stage + 2 * (e0 + r * HL_THREADS + tid)) = make_uint2((unsigned int)v[r][0], (unsigned int)v[r][1]);
                                done[r] = true;
                            } else all = false;
                        }
                    }
                    if (all) break;
                    if (++spins > (1u << 26)) __trap();
                }
            }
            if (q0 == 0) HL_MK(17);
            __syncthreads();
            if (q0 == 0) HL_MK(18);
            // The owner's chain is the critical path of a small block step (the other CTAs wait for its records), so it is ordered
            // for overlap: corrector and new step first -> t + dt into shared memory -> (last round, one tile) barrier -> an idle warp
            // rescans the tile for the next records WHILE the particle's warp stores the new state and runs the release fence.
            const bool last_round = Kc == 1 && q0 + HL_CQ >= nown;
            bool have = false;
            int c_k = 0, c_kk = 0, c_l = 0, c_p = 0, c_c = 0;
            double x1c = 0, v1c = 0, a1c = 0, ad1c = 0, d_new = 0, pot_new = 0;
            if (w < nq) {
            const int q = q0 + w;
            const int k = sm.own_k[q], sl = sm.own_l[q];
            const uint2 *sg = reinterpret_cast<const uint2 *>(stage) + (size_t)w * (HL_CHUNK_WORDS / 2) * G;      // [CTA][component]
            double v[7] = {0, 0, 0, 0, 0, 0, 0};
            for (int s = lane; s < G; s += 32) {
#pragma unroll
                for (int c = 0; c < 7; ++c) {
                    const uint2 u = sg[s * 7 + c];
                    v[c] += __longlong_as_double((long long)(((unsigned long long)u.y << 32) | u.x));
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
                for (int c = 0; c < 7; ++c) v[c] += __shfl_xor_sync(FULL, v[c], o);
            }
            if (q0 == 0) HL_MK(19);
                // the corrector, the Aarseth step and the power-of-two rule: lanes 0-2 one component each (hd_correct_warp)
                const int kk = sl / JT, l = sl % JT;
                const int p = (cta + kk * G) * JT + l;
                const int c = lane < 3 ? lane : 0;
                double a0c, ad0c, xic, vic, h;
                if (inl) {
                    const double *st = sm.own_st[kk * HL_INLINE + (k - sm.s_off[cta + kk * G])];
                    xic = st[c]; vic = st[3 + c]; a0c = st[6 + c]; ad0c = st[9 + c];
                    h = st[12];
                } else {
                    xic = A.B.xi[3 * (size_t)k + c]; vic = A.B.vi[3 * (size_t)k + c];
                    a0c = A.S.a[3 * (size_t)p + c]; ad0c = A.S.ad[3 * (size_t)p + c];
                    h = A.S.dt[p];
                }
                a1c = c == 0 ? v[0] : c == 1 ? v[1] : v[2];
                ad1c = c == 0 ? v[3] : c == 1 ? v[4] : v[5];
                d_new = hd_correct_warp(lane, h, a0c, ad0c, a1c, ad1c, xic, vic, tn, A.C.eta, A.C.dt_max, x1c, v1c);
                if (lane == 4) sm.tnext[kk][l] = tn + d_new;
                pot_new = v[6];
                have = true; c_k = k; c_kk = kk; c_l = l; c_p = p; c_c = c;
                if (q0 == 0) HL_MK(20);
            }
            if (last_round) __syncthreads();                     // every corrected particle's t + dt is in place
            if (have) {
                // each of lanes 0-2 stores its own component of the new state, of the resident tile and of the j-store record
                const int k = c_k, kk = c_kk, l = c_l, p = c_p, c = c_c;
                char *Ts = sm.raw[kk], *Tg = A.C.raw + (size_t)(cta + kk * G) * RAW_TILE_BYTES;      // my resident copy, the j-store
                if (lane < 3) {
                    A.a1[3 * (size_t)k + c] = a1c; A.ad1[3 * (size_t)k + c] = ad1c;
                    A.S.x[3 * (size_t)p + c] = x1c; A.S.v[3 * (size_t)p + c] = v1c;
                    A.S.a[3 * (size_t)p + c] = a1c; A.S.ad[3 * (size_t)p + c] = ad1c;
                    raw_x(Ts, c, l) = x1c; raw_v(Ts, c, l) = (float)v1c; raw_a2(Ts, c, l) = (float)(a1c / 2); raw_j6(Ts, c, l) = (float)(ad1c / 6);
                    raw_x(Tg, c, l) = x1c; raw_v(Tg, c, l) = (float)v1c; raw_a2(Tg, c, l) = (float)(a1c / 2); raw_j6(Tg, c, l) = (float)(ad1c / 6);
                }
                if (lane == 3) {
                    A.pot[k] = pot_new;
                    A.S.t[p] = tn;
                    A.S.dt[p] = d_new;
                    atomicMin(A.C.dt_min_bits, (unsigned long long)__double_as_longlong(d_new));
                }
                if (lane == 4) {
                    const float m = raw_m(Ts, l);
                    raw_t(Ts, l) = tn; raw_idx(Ts, l) = p;              // (mass and index do not change)
                    raw_t(Tg, l) = tn; raw_m(Tg, l) = m; raw_idx(Tg, l) = p;
                }
                // release: the new Hermite state must be visible to whoever reads this CTA's next records; the warp's stores are
                // ordered before lane 0's fence by the warp barrier, the fence before the records by the closing CTA barrier
                __syncwarp();
                if (lane == 0) hl_fence();
                if (q0 == 0) HL_MK(21);
            } else if (last_round && w == HL_NW - 1) {
                rescan_tile0();
            }
            __syncthreads();
        }
        HL_MK(10);
        HL_MK(22);
        if (PROF && tid == 0) {
            sm.mk_open = nown > 0 && nown <= HL_CQ && ni < 8;
            if (cta == 0 && ni < 8) {
                for (int q = 0; q < 10; ++q) atomicAdd(A.prof + q, (unsigned long long)(sm.mk[q + 1] - sm.mk[q]));
                atomicAdd(A.prof + 11, (unsigned long long)(sm.mk[11] - sm.mk[3]));
                atomicAdd(A.prof + 12, (unsigned long long)(sm.mk[12] - sm.mk[11]));
                atomicAdd(A.prof + 13, (unsigned long long)(sm.mk[13] - sm.mk[12]));
                atomicAdd(A.prof + 14, (unsigned long long)(sm.mk[4] - sm.mk[13]));
                atomicAdd(A.prof + 15, 1ull);
            }
        }
        if (tid == 0) sm.nown_prev = nown;
        rescan = nown > 0;
        pre_scanned = nown > 0 && Kc == 1;      // (the last round of phase C rescanned the tile)
        t_sys = tn;
        ++steps;
        npart += ni;
        ni_last = ni;
        n_inline += inl ? 1 : 0;
        if (cta == 0) {
            unsigned long long now;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(now));
            if (tid < 30 && ni >= (1 << tid) && ni < (2 << tid)) { ++hist; hist_ns += (long long)(now - t_step); }
            t_step = now;
        }
        // no barrier here: after the force phase's last barrier only phase C (which ends with one) touches shared memory, and the
        // next step begins with warp 0 alone up to the barrier that follows its selection
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
            A.status->inline_steps = n_inline;
            if (reason == HL_BIG) { *A.B.d_ni = ni_next; *A.B.d_tnext = t_big; }
            else if (ni_last > 0) { *A.B.d_ni = ni_last; *A.B.d_tnext = t_sys; }
        }
    }
}

}  // namespace g6
