// g6_block_step.cuh -- ONE kernel for the small active blocks of block time steps (n_i <= 64):
// j-store update + j-predictor + force + combine (steps a-1 .. a-5 of the path) in a single launch.
//
// For a handful of i-particles the step is bound by the one pass over the N_j stored particles
// (76 B each) and by launch/copy latency, not by arithmetic.  The paper's idea for
// small blocks (fewer i than threads => several threads share an i and split the
// j) is taken to its limit and the whole block step is fused:
//
//  * one persistent CTA of 8 warps per SM; CTA c owns the raw j-tiles c, c+G, c+2G, ...  A raw tile
//    (256 particles x 76 B, g6_device.cuh) is staged global -> shared by ONE TMA bulk copy
//    (cp.async.bulk + mbarrier complete_tx) into a ring of 9-11 slots that fills the SM's shared
//    memory, so ~100-200 KB per SM are in flight without costing a register -- that is what keeps
//    HBM busy while the warps compute.
//  * THE WARPS ARE THE WORKERS: tile number `it` of the CTA is handled by warp it % 8 alone --
//    no __syncthreads in the loop, one mbarrier per slot, and the warp that has read a slot into
//    registers re-issues the copy of the tile NS ahead into it at once.  (With a block-wide
//    predict / barrier / compute sequence all warps load, then all compute, and HBM idles half
//    the time: measured 28 us per step at N_j = 2^20 whether or not the j-store sat in L2.)
//  * a-1: the particles corrected in the previous step arrive INSIDE THE KERNEL PARAMETERS (no
//    staging kernel, no PCIe read); the warp that owns a particle's tile patches the staged copy
//    and writes the record through to the j-store.  The i-block travels the same way.
//  * a-2: LANES OVER j: every lane predicts 8 j of the tile (Eq. 1-2, same routine as k_predict)
//    straight into registers; nothing predicted ever goes to shared memory or HBM.
//  * a-4: the warp loops over all i-particles of the block (broadcast from shared memory) and
//    evaluates its 8 pairs per lane with the same packed FP32 arithmetic as the sweep kernel
//    (double-single separations, Eq. 3); the 7 sums of a (i, tile) are reduced over the warp by a
//    transposing butterfly (9 shuffles instead of 35) and folded into the warp's fp64 accumulators
//    in shared memory; the nearest neighbour by two warp-wide integer min-reductions (r2 bits,
//    then address).  At the end the 8 warps' sums are added in warp order.
//  * a-5: each CTA writes one partial per i; the LAST CTA to finish (atomic ticket) sums the G
//    partials in CTA order -- deterministic -- and writes the results, possibly straight into
//    mapped host memory (a-6).
// Every pair is checked (address < nj, index_j != index_i, s2 > 0), so eps2 = 0 is served too.
#pragma once
#include "g6_force_fast.cuh"

namespace g6 {

constexpr int BS_THREADS = 384;
// raw-tile slots of the shared-memory ring (one CTA per SM owns all of its shared memory)
__host__ __device__ constexpr int bs_nslots(int maxi) { return maxi <= 16 ? 10 : 8; }
constexpr int BS_MAX_I = 64;
constexpr int BS_NB_SCRATCH = 1024;     // addresses per warp in the last CTA's neighbour-list merge: the largest nb_maxlen served

// i-block and changed j-particles carried by value in the kernel parameters
template <int MAXI>
struct BsInline {
    double xi[MAXI][3];
    double vi[MAXI][3];
    int index[MAXI];
    JRecord upd[MAXI];
};

struct BsArgs {
    char *raw;                  // j-store (inline updates are written through)
    double ti;
    int nj, ntiles;
    int ni, n_upd;
    float eps2;
    int ds;
    int inline_i;               // 1: i-block from BsInline, 0: from the device-visible pointers below
    const int *i_index;
    const double *xi, *vi;
    Partials P;                 // [i][cta]: stride_s = 1, stride_i = gridDim.x
    unsigned int *counter;      // arrival ticket, zero before the launch, reset by the last CTA
    double *acc, *jerk, *pot;   // results (device or mapped host memory)
    int *nn_index;
    double *nn_r2;
    unsigned int *done_flag;    // not NULL: mapped host word that receives done_seq after the results are written
    unsigned int done_seq;
    // neighbour lists (reading 20); h2 == nullptr: none.  Every warp of the grid keeps its own
    // list per i-particle (it meets its tiles in increasing address order); the last CTA merges them by address.
    const double *h2;           // [ni] neighbour-sphere radius squared
    int nb_maxlen;
    int *nb_wcnt;               // [ni][G * NW]          neighbours found by warp (cta * NW + w), may exceed nb_maxlen
    int *nb_wlist;              // [G * NW][ni][maxlen]  their j addresses, increasing
    int *nb_cnt;                // [ni]          out: all neighbours found
    int *nb_list;               // [ni][maxlen]  out: callers' indices, increasing j address, the smallest addresses on overflow
    float *dbg_dx;              // DBG instantiation only (parity pin P11): [ni][nj][3] Eq.-3 separations; nullptr in the library
};

__device__ __forceinline__ int ld_acquire_cta(const volatile int *p)
{
    int v;
    asm volatile("ld.acquire.cta.shared.s32 %0, [%1];" : "=r"(v) : "r"(smem_u32(const_cast<const int *>(p))) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_cta(volatile int *p, int v)
{
    asm volatile("st.release.cta.shared.s32 [%0], %1;" ::"r"(smem_u32(const_cast<int *>(p))), "r"(v) : "memory");
}

template <int MAXI>
struct BsSmem {
    alignas(128) char raw[bs_nslots(MAXI)][RAW_TILE_BYTES];   // ring of raw tiles: tile `it` of the CTA lives in slot it % NS
    double acc[BS_THREADS / 32][MAXI][8];                     // per-warp fp64 sums of every i
    float r2[BS_THREADS / 32][MAXI];                          // per-warp nearest neighbour of every i
    int addr[BS_THREADS / 32][MAXI];
    float ipart[MAXI][9];
    float h2[MAXI];                                           // neighbour radii (binary32, like r2)
    int nbcnt[BS_THREADS / 32][MAXI];                         // per-warp running neighbour counts
    int iidx[MAXI];
    int uaddr[MAXI];
    alignas(8) uint64_t full[bs_nslots(MAXI)];
    volatile int armed[bs_nslots(MAXI)];                      // CTA tile number whose copy was last issued into the slot
    int is_last;
};
static_assert(sizeof(BsSmem<16>) <= 232448 && sizeof(BsSmem<64>) <= 232448, "block-step shared memory");

// two consecutive j against one i, every pair checked.  `ok` in: address < nj && index differs.
template <bool NEWTON, bool DBG = false>
__device__ __forceinline__ void pair2_checked(IPart &I, const float2 xh, const float2 yh, const float2 zh, const float2 xl,
                                              const float2 yl, const float2 zl, const float2 vx, const float2 vy, const float2 vz,
                                              float2 m, const float2 eps2, bool ok0, bool ok1, float2 &r2_out, float2 *dbg = nullptr)
{
    constexpr float INF = __builtin_huge_valf();
    const float2 dx = add2(add2(xh, I.nxh[0]), add2(xl, I.nxl[0]));      // Eq. 3
    const float2 dy = add2(add2(yh, I.nxh[1]), add2(yl, I.nxl[1]));
    const float2 dz = add2(add2(zh, I.nxh[2]), add2(zl, I.nxl[2]));
    if (DBG) { dbg[0] = dx; dbg[1] = dy; dbg[2] = dz; }      // parity pin P11 (csrc/debug/g6_debug_dx.cu only)
    const float2 dvx = add2(vx, I.nv[0]);
    const float2 dvy = add2(vy, I.nv[1]);
    const float2 dvz = add2(vz, I.nv[2]);
    const float2 r2 = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));
    float2 s2 = add2(r2, eps2);
    ok0 = ok0 && (s2.x > 0.0f);                                          // DESIGN.md reading 5
    ok1 = ok1 && (s2.y > 0.0f);
    s2 = make_float2(ok0 ? s2.x : 1.0f, ok1 ? s2.y : 1.0f);
    m = make_float2(ok0 ? m.x : 0.0f, ok1 ? m.y : 0.0f);
    float2 rinv = make_float2(rsqrt_approx(s2.x), rsqrt_approx(s2.y));
    if (NEWTON) {
        const float2 e = fma2(s2, mul2(rinv, rinv), dup(-1.0f));
        rinv = fma2(mul2(dup(-0.5f), rinv), e, rinv);
    }
    const float2 rinv2 = mul2(rinv, rinv);
    const float2 mrinv = mul2(m, rinv);
    const float2 mrinv3 = mul2(mrinv, rinv2);
    const float2 rv = fma2(dz, dvz, fma2(dy, dvy, mul2(dx, dvx)));
    const float2 alpha = mul2(dup(-3.0f), mul2(rv, rinv2));
    I.p = add2(I.p, mrinv);
    I.a[0] = fma2(mrinv3, dx, I.a[0]);
    I.a[1] = fma2(mrinv3, dy, I.a[1]);
    I.a[2] = fma2(mrinv3, dz, I.a[2]);
    I.j[0] = fma2(mrinv3, fma2(alpha, dx, dvx), I.j[0]);
    I.j[1] = fma2(mrinv3, fma2(alpha, dy, dvy), I.j[1]);
    I.j[2] = fma2(mrinv3, fma2(alpha, dz, dvz), I.j[2]);
    r2_out = make_float2(ok0 ? r2.x : INF, ok1 ? r2.y : INF);
}

// Sum 8 per-lane values over the 32 lanes of a warp with 9 shuffles: after the three exchange
// steps lane L holds quantity q(L) = 4*bit4(L) + 2*bit3(L) + bit2(L), summed over the lanes that
// share bits 1..0 of L... then two plain butterfly steps finish it.  Fixed tree => reproducible.
__device__ __forceinline__ float transpose_reduce8(const float (&v)[8], int lane)
{
    const unsigned FULL = 0xffffffffu;
    float w[4], u[2];
    const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float send = b4 ? v[k] : v[k + 4];
        const float keep = b4 ? v[k + 4] : v[k];
        w[k] = __fadd_rn(keep, __shfl_xor_sync(FULL, send, 16));
    }
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        const float send = b3 ? w[k] : w[k + 2];
        const float keep = b3 ? w[k + 2] : w[k];
        u[k] = __fadd_rn(keep, __shfl_xor_sync(FULL, send, 8));
    }
    const float send = b2 ? u[0] : u[1];
    const float keep = b2 ? u[1] : u[0];
    float t = __fadd_rn(keep, __shfl_xor_sync(FULL, send, 4));
    t = __fadd_rn(t, __shfl_xor_sync(FULL, t, 2));
    t = __fadd_rn(t, __shfl_xor_sync(FULL, t, 1));
    return t;
}

// `Dp`: the inline i-block / j updates of the launch (nullptr when there are none: device-resident callers)
template <int MAXI, bool NEWTON, bool DBG = false>
__device__ __forceinline__ void block_step_body(const BsArgs &A0, const BsInline<MAXI> *Dp)
{
    const BsArgs &A = A0;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    BsSmem<MAXI> &sm = *reinterpret_cast<BsSmem<MAXI> *>(smem_raw);
    constexpr float INF = __builtin_huge_valf();
    constexpr int NW = BS_THREADS / 32;
    const unsigned FULL = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int G = gridDim.x, cta = blockIdx.x;
    // The CTA (one per SM) owns the raw tiles cta, cta + G, ...; tile number `it` of that sequence is staged
    // in ring slot it % NS and worked on by warp it % NW alone: the warps never wait for one another inside
    // the loop (no __syncthreads), and NS > NW slots keep copies in flight while every warp computes.
    constexpr int NS = bs_nslots(MAXI);
    const int nt = cta < A.ntiles ? (A.ntiles - cta + G - 1) / G : 0;

    if (tid == 0) {
#pragma unroll
        for (int k = 0; k < NS; ++k) { mbar_init(&sm.full[k], 1); sm.armed[k] = k; }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
#pragma unroll
        for (int k = 0; k < NS; ++k)
            if (k < nt) {
                mbar_expect_tx(&sm.full[k], RAW_TILE_BYTES);
                tma_load_1d(sm.raw[k], A.raw + (size_t)(cta + k * G) * RAW_TILE_BYTES, RAW_TILE_BYTES, &sm.full[k]);
            }
    }
    // i-block -> shared memory (double-single split here: the host hands fp64)
    for (int k = tid; k < A.ni * 3; k += BS_THREADS) {
        const int i = k / 3, c = k % 3;
        const double x = A.inline_i ? Dp->xi[i][c] : A.xi[k];
        const double v = A.inline_i ? Dp->vi[i][c] : A.vi[k];
        float hi, lo;
        ds_split(x, hi, lo);
        sm.ipart[i][c] = hi;
        sm.ipart[i][3 + c] = A.ds ? lo : 0.0f;
        sm.ipart[i][6 + c] = (float)v;
    }
    for (int i = tid; i < MAXI; i += BS_THREADS) {
        if (i < A.ni) sm.iidx[i] = A.inline_i ? Dp->index[i] : A.i_index[i];
        sm.uaddr[i] = i < A.n_upd ? Dp->upd[i].addr : -1;
        sm.h2[i] = (A.h2 && i < A.ni) ? (float)A.h2[i] : 0.0f;
#pragma unroll
        for (int q = 0; q < NW; ++q) {
            sm.nbcnt[q][i] = 0;
            sm.r2[q][i] = INF;
            sm.addr[q][i] = 0x7fffffff;
#pragma unroll
            for (int k = 0; k < 8; ++k) sm.acc[q][i][k] = 0.0;
        }
    }
    __syncthreads();

    const float2 eps2 = dup(A.eps2);
    for (int it = w; it < nt; it += NW) {
        const int tile = cta + it * G;
        const int slot = it % NS;
        char *R = sm.raw[slot];
        // the copy of THIS tile must have been issued before its phase is waited for (a parity wait
        // cannot tell phase p+1 from the completed phase p-1)
        if (it >= NS) {
            uint32_t spins = 0;
            while (ld_acquire_cta(&sm.armed[slot]) != it) { if (++spins > (1u << 26)) __trap(); }
        }
        mbar_wait(&sm.full[slot], (uint32_t)(it / NS) & 1u);

        // ---- a-1: particles corrected in the last step that live in this tile: patch the staged copy
        // and write the record through to the j-store
        if (A.n_upd > 0) {
            for (int u = lane; u < A.n_upd; u += 32)
                if (sm.uaddr[u] / JT == tile) {
                    const JRecord r = Dp->upd[u];
                    store_record(R, r.addr % JT, r);
                    store_record(A.raw + (size_t)tile * RAW_TILE_BYTES, r.addr % JT, r);
                }
            __syncwarp();
        }
        // ---- a-2: predict my 8 j straight into registers (Eq. 1-2, same routine as k_predict); nothing
        // predicted ever goes to memory.  Lane l owns the pairs {2l, 2l+1} + 64 g, g = 0..3: one conflict-free
        // vector load per field and pair (double2 / float2 / int2, consecutive lanes on consecutive addresses)
        float2 jf[NF][4];
        int2 jx[4];
        const int ja0 = tile * JT + 2 * lane;                 // my pairs: ja0 + 64 g + {0, 1}
        const bool ragged = tile * JT + JT > A.nj;            // only the last tile of the j-range
#pragma unroll
        for (int g = 0; g < 4; ++g) {
            const int l0 = 2 * lane + 64 * g;
            const double2 tj = *reinterpret_cast<const double2 *>(R + RAW_T + 8 * l0);
            const float2 dt = make_float2((float)(A.ti - tj.x), (float)(A.ti - tj.y));
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const double2 x0 = *reinterpret_cast<const double2 *>(R + RAW_X + 8 * (k * JT + l0));
                const float2 v0 = *reinterpret_cast<const float2 *>(R + RAW_V + 4 * (k * JT + l0));
                const float2 a2 = *reinterpret_cast<const float2 *>(R + RAW_A2 + 4 * (k * JT + l0));
                const float2 j6 = *reinterpret_cast<const float2 *>(R + RAW_J6 + 4 * (k * JT + l0));
                predict_coord(dt.x, x0.x, v0.x, a2.x, j6.x, A.ds, jf[F_XH + k][g].x, jf[F_XL + k][g].x, jf[F_V + k][g].x);
                predict_coord(dt.y, x0.y, v0.y, a2.y, j6.y, A.ds, jf[F_XH + k][g].y, jf[F_XL + k][g].y, jf[F_V + k][g].y);
            }
            jf[F_M][g] = *reinterpret_cast<const float2 *>(R + RAW_M + 4 * l0);
            jx[g] = *reinterpret_cast<const int2 *>(R + RAW_IDX + 4 * l0);
            if (ragged) {                                     // addresses >= nj: finite and massless
                const bool in0 = ja0 + 64 * g < A.nj, in1 = ja0 + 64 * g + 1 < A.nj;
#pragma unroll
                for (int k = 0; k < NF; ++k) jf[k][g] = make_float2(in0 ? jf[k][g].x : 0.0f, in1 ? jf[k][g].y : 0.0f);
            }
        }
        // the slot is consumed: refill it with the tile NS ahead while the forces are computed
        __syncwarp();
        if (lane == 0 && it + NS < nt) {
            if (A.n_upd > 0) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // a-1 wrote the slot through the generic proxy
            mbar_expect_tx(&sm.full[slot], RAW_TILE_BYTES);
            tma_load_1d(R, A.raw + (size_t)(tile + NS * G) * RAW_TILE_BYTES, RAW_TILE_BYTES, &sm.full[slot]);
            st_release_cta(&sm.armed[slot], it + NS);
        }

        // ---- a-4: every i-particle of the block against my 8 j
        for (int i = 0; i < A.ni; ++i) {
            IPart I;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                I.nxh[k] = dup(-sm.ipart[i][k]);
                I.nxl[k] = dup(-sm.ipart[i][3 + k]);
                I.nv[k] = dup(-sm.ipart[i][6 + k]);
                I.a[k] = dup(0.0f);
                I.j[k] = dup(0.0f);
            }
            I.p = dup(0.0f);
            const int my = sm.iidx[i];
            float2 r2m[4];
#pragma unroll
            for (int g = 0; g < 4; ++g) {
                const int ja = ja0 + 64 * g;
                float2 dd[3];
                pair2_checked<NEWTON, DBG>(I, jf[0][g], jf[1][g], jf[2][g], jf[3][g], jf[4][g], jf[5][g], jf[6][g], jf[7][g], jf[8][g], jf[9][g], eps2,
                                           (ja < A.nj) && (jx[g].x != my), (ja + 1 < A.nj) && (jx[g].y != my), r2m[g], dd);
                if (DBG) {
#pragma unroll
                    for (int k = 0; k < 3; ++k) {
                        if (ja < A.nj) A.dbg_dx[((size_t)i * A.nj + ja) * 3 + k] = dd[k].x;
                        if (ja + 1 < A.nj) A.dbg_dx[((size_t)i * A.nj + ja + 1) * 3 + k] = dd[k].y;
                    }
                }
            }
            // the 7 sums of this (i, tile): FP32 tree over the 256 j, then fp64 (reading 9)
            const float v8[8] = {__fadd_rn(I.a[0].x, I.a[0].y), __fadd_rn(I.a[1].x, I.a[1].y), __fadd_rn(I.a[2].x, I.a[2].y),
                                 __fadd_rn(I.j[0].x, I.j[0].y), __fadd_rn(I.j[1].x, I.j[1].y), __fadd_rn(I.j[2].x, I.j[2].y),
                                 __fadd_rn(I.p.x, I.p.y), 0.0f};
            const float tot = transpose_reduce8(v8, lane);
            if ((lane & 3) == 0) sm.acc[w][i][lane >> 2] += (double)tot;
            // nearest neighbour: min r2 over the warp (non-negative floats order like unsigned integers)
            float lmin = fminf(fminf(r2m[0].x, r2m[0].y), fminf(r2m[1].x, r2m[1].y));
            lmin = fminf(lmin, fminf(fminf(r2m[2].x, r2m[2].y), fminf(r2m[3].x, r2m[3].y)));
            const unsigned gbits = __reduce_min_sync(FULL, __float_as_uint(lmin));
            // neighbour list: pairs with r2 < h2_i (masked pairs carry r2 = +inf), appended in address order
            // = (g, lane, x before y); rare, so the whole warp leaves the common path only when some lane has a hit
            if (A.h2 && gbits < __float_as_uint(sm.h2[i])) {
                const float h2i = sm.h2[i];
                int cnt = sm.nbcnt[w][i];
                int *dst = A.nb_wlist + ((size_t)(cta * NW + w) * A.ni + i) * A.nb_maxlen;
                const unsigned lt = (1u << lane) - 1u;
#pragma unroll
                for (int g = 0; g < 4; ++g) {
                    const bool hx = r2m[g].x < h2i, hy = r2m[g].y < h2i;
                    const unsigned mx = __ballot_sync(FULL, hx), my_ = __ballot_sync(FULL, hy);
                    const int px = cnt + __popc(mx & lt) + __popc(my_ & lt);
                    if (hx && px < A.nb_maxlen) dst[px] = ja0 + 64 * g;
                    if (hy && px + (hx ? 1 : 0) < A.nb_maxlen) dst[px + (hx ? 1 : 0)] = ja0 + 64 * g + 1;
                    cnt += __popc(mx) + __popc(my_);
                }
                __syncwarp();
                if (lane == 0) sm.nbcnt[w][i] = cnt;
            }
            if (gbits < __float_as_uint(sm.r2[w][i])) {     // strict: my earlier tiles (lower addresses) keep ties
                int cand = 0x7fffffff;
#pragma unroll
                for (int g = 3; g >= 0; --g) {               // descending, so the smallest address is kept
                    if (__float_as_uint(r2m[g].y) == gbits) cand = ja0 + 64 * g + 1;
                    if (__float_as_uint(r2m[g].x) == gbits) cand = ja0 + 64 * g;
                }
                const int gaddr = __reduce_min_sync(FULL, cand);
                __syncwarp();
                if (lane == 0) { sm.r2[w][i] = __uint_as_float(gbits); sm.addr[w][i] = gaddr; }
            }
            __syncwarp();
        }
    }
    __syncthreads();

    // ---- a-5, first half: one partial per (i, CTA): the warps' sums in warp order
    for (int i = tid; i < A.ni; i += BS_THREADS) {
        const size_t o = (size_t)cta * A.P.stride_s + (size_t)i * A.P.stride_i;
        double v[7];
#pragma unroll
        for (int k = 0; k < 7; ++k) v[k] = sm.acc[0][i][k];
        float best = sm.r2[0][i];
        int baddr = sm.addr[0][i];
#pragma unroll
        for (int q = 1; q < NW; ++q) {
#pragma unroll
            for (int k = 0; k < 7; ++k) v[k] += sm.acc[q][i][k];
            const float r2 = sm.r2[q][i];
            const int ad = sm.addr[q][i];
            if (r2 < best || (r2 == best && ad < baddr)) { best = r2; baddr = ad; }
        }
#pragma unroll
        for (int k = 0; k < 3; ++k) { A.P.acc[k][o] = v[k]; A.P.jrk[k][o] = v[3 + k]; }
        A.P.pot[o] = -v[6];
        const bool has = baddr != 0x7fffffff;
        A.P.nn_r2[o] = has ? best : INF;
        A.P.nn_addr[o] = has ? baddr : -1;
    }
    if (A.h2)
        for (int k = tid; k < A.ni * NW; k += BS_THREADS) {
            const int i = k / NW, q = k % NW;
            A.nb_wcnt[(size_t)i * (G * NW) + cta * NW + q] = sm.nbcnt[q][i];
        }
    // the ticket: the barrier orders the CTA's partial stores before thread 0, whose release fence is cumulative; the last CTA's
    // acquire fence sits between the ticket and its reads of the partials (ld.global.cg)
    __syncthreads();
    if (tid == 0) {
        fence_acq_rel_gpu();
        const unsigned ticket = atomicAdd(A.counter, 1u);
        sm.is_last = (ticket == (unsigned)G - 1u);
        if (sm.is_last) fence_acq_rel_gpu();
    }
    __syncthreads();
    if (!sm.is_last) return;

    // ---- a-5, second half (last CTA only): sum the G partials of every i in CTA order
    for (int i = w; i < A.ni; i += BS_THREADS / 32) {
        double v[7] = {0, 0, 0, 0, 0, 0, 0};
        float best = INF;
        int baddr = 0x7fffffff;
        // all loads of a chunk of 5 x 32 partials are issued before the first is used (one L2 round trip instead
        // of five); the lane still adds its partials s = lane, lane + 32, ... in that order
        for (int s0 = 0; s0 < G; s0 += 160) {
            double t[5][7];
            float r2[5];
            int ad[5];
#pragma unroll
            for (int q = 0; q < 5; ++q) {
                const int sq = s0 + lane + 32 * q;
                const bool in = sq < G;
                const size_t o = (size_t)(in ? sq : 0) * A.P.stride_s + (size_t)i * A.P.stride_i;
#pragma unroll
                for (int k = 0; k < 3; ++k) { t[q][k] = in ? __ldcg(A.P.acc[k] + o) : 0.0; t[q][3 + k] = in ? __ldcg(A.P.jrk[k] + o) : 0.0; }
                t[q][6] = in ? __ldcg(A.P.pot + o) : 0.0;
                r2[q] = in ? __ldcg(A.P.nn_r2 + o) : INF;
                ad[q] = in ? __ldcg(A.P.nn_addr + o) : -1;
            }
#pragma unroll
            for (int q = 0; q < 5; ++q) {
                if (s0 + lane + 32 * q < G) {
#pragma unroll
                    for (int k = 0; k < 7; ++k) v[k] += t[q][k];
                    if (ad[q] >= 0 && (r2[q] < best || (r2[q] == best && ad[q] < baddr))) { best = r2[q]; baddr = ad[q]; }
                }
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
            for (int k = 0; k < 7; ++k) v[k] += __shfl_xor_sync(FULL, v[k], o);
            const float r2 = __shfl_xor_sync(FULL, best, o);
            const int ad = __shfl_xor_sync(FULL, baddr, o);
            if (r2 < best || (r2 == best && ad < baddr)) { best = r2; baddr = ad; }
        }
        if (lane == 0) {
#pragma unroll
            for (int k = 0; k < 3; ++k) { A.acc[3 * (size_t)i + k] = v[k]; A.jerk[3 * (size_t)i + k] = v[3 + k]; }
            A.pot[i] = v[6];
            const bool has = baddr != 0x7fffffff;
            if (A.nn_index) A.nn_index[i] = has ? j_index(A.raw, baddr) : -1;
            if (A.nn_r2) A.nn_r2[i] = has ? (double)best : (double)INF;
        }
    }
    // ---- neighbour lists (last CTA): merge the per-warp lists of every i by j address.  One warp per i; the shared-memory
    // ring is idle now and serves as scratch (BS_NB_SCRATCH addresses per warp >= nb_maxlen, enforced by the host).
    if (A.h2) {
        const int NSEG = G * NW;
        int *scratch = reinterpret_cast<int *>(&sm.raw[0][0]) + w * BS_NB_SCRATCH;
        for (int i = w; i < A.ni; i += NW) {
            const int *wc = A.nb_wcnt + (size_t)i * NSEG;
            int tot = 0;
            for (int sg = lane; sg < NSEG; sg += 32) tot += __ldcg(wc + sg);
            tot = __reduce_add_sync(FULL, tot);
            // T: entries with address < T are kept.  No overflow: everything.  Overflow: the nb_maxlen smallest addresses,
            // found by bisection on the address (every per-warp list is sorted and holds its own nb_maxlen smallest).
            int T = 0x7fffffff;
            if (tot > A.nb_maxlen) {
                int lo = 0, hi = A.ntiles * JT;
                while (hi - lo > 1) {
                    const int mid = lo + (hi - lo) / 2;
                    int below = 0;
                    for (int sg = lane; sg < NSEG; sg += 32) {
                        const int c = min(__ldcg(wc + sg), A.nb_maxlen);
                        if (c > 0) {
                            const int *L = A.nb_wlist + ((size_t)sg * A.ni + i) * A.nb_maxlen;
                            int a = 0, b = c;                       // first entry >= mid
                            while (a < b) { const int m = (a + b) >> 1; if (__ldcg(L + m) < mid) a = m + 1; else b = m; }
                            below += a;
                        }
                    }
                    below = __reduce_add_sync(FULL, below);
                    if (below >= A.nb_maxlen) hi = mid; else lo = mid;
                }
                T = hi;
            }
            // gather the kept entries of all segments into the scratch (order irrelevant), then rank-sort by address
            int base = 0;
            for (int s0 = 0; s0 < NSEG; s0 += 32) {
                const int sg = s0 + lane;
                const int c = sg < NSEG ? min(__ldcg(wc + sg), A.nb_maxlen) : 0;
                const int *L = A.nb_wlist + ((size_t)(sg < NSEG ? sg : 0) * A.ni + i) * A.nb_maxlen;
                int keep = 0;
                while (keep < c && __ldcg(L + keep) < T) ++keep;
                int inc = keep;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int u = __shfl_up_sync(FULL, inc, o);
                    if (lane >= o) inc += u;
                }
                const int at = base + inc - keep;
                for (int k = 0; k < keep; ++k) scratch[at + k] = __ldcg(L + k);
                base += __shfl_sync(FULL, inc, 31);
            }
            __syncwarp();
            const int nkeep = base;                               // = min(tot, nb_maxlen)
            for (int e = lane; e < nkeep; e += 32) {
                const int v = scratch[e];
                int rank = 0;
                for (int k = 0; k < nkeep; ++k) rank += scratch[k] < v;
                A.nb_list[(size_t)i * A.nb_maxlen + rank] = j_index(A.raw, v);
            }
            if (lane == 0) A.nb_cnt[i] = tot;
            __syncwarp();
        }
    }
    if (tid == 0) *A.counter = 0u;
    // results that went straight to mapped host memory: tell the host they are complete (it spins on this word instead of
    // waiting for an event, a few microseconds sooner); the barrier orders the other warps' result stores before the
    // system-scope fence of this thread
    if (A.done_flag) {
        __syncthreads();
        if (tid == 0) {
            __threadfence_system();
            *reinterpret_cast<volatile unsigned int *>(A.done_flag) = A.done_seq;
        }
    }
}

template <int MAXI, bool NEWTON>
__global__ void __launch_bounds__(BS_THREADS)
k_block_step(const BsArgs A, const __grid_constant__ BsInline<MAXI> D)
{
    block_step_body<MAXI, NEWTON>(A, &D);
}

// the same kernel without the inline payload (i-block in device memory, no j updates): 2-8 KB fewer launch parameters
template <int MAXI, bool NEWTON>
__global__ void __launch_bounds__(BS_THREADS)
k_block_step_dev(const BsArgs A)
{
    block_step_body<MAXI, NEWTON>(A, nullptr);
}

// the DBG instantiation (every pair's separation also goes to A.dbg_dx); launched only by csrc/debug/g6_debug_dx.cu
template <int MAXI, bool NEWTON>
__global__ void __launch_bounds__(BS_THREADS)
k_block_step_dbg(const BsArgs A)
{
    block_step_body<MAXI, NEWTON, true>(A, nullptr);
}

// ================================================================================================
// k_block_step2 -- the block-step kernel without neighbour lists (the common case), second design.
//
// Same launch, same a-1 .. a-5 in one kernel, same ring of raw j-tiles fed by one TMA bulk copy per tile, same last-CTA
// combine; what changes is the pair phase.  The first design kept lanes over j for the forces too and therefore had to
// reduce the seven sums of every (i-particle, tile) over the warp (9 shuffles + two warp-wide integer reductions for the
// nearest neighbour): a third of the instructions of a small block step.  Here a warp predicts its unit (a half or a quarter
// tile, see below; lanes over j, as before), writes the predicted particles to its OWN buffer in shared memory and hands its
// share of the raw slot back to the ring at once; the pairs are then evaluated with LANES = (i-particle, j-sub-range) -- "several threads share an i and
// split the j" -- so that every lane keeps the sums and the nearest neighbour of ITS i-particle in
// registers across all the tiles the warp works on (FP32 over one tile slice, folded into fp64 per tile: DESIGN.md reading
// 9), and the lanes of one i are reduced by a fixed shuffle tree ONCE, at the end of the kernel.  Blocks above 16 particles
// take their i-particles in at most two power-of-two chunks (the predicted unit is re-read from shared memory, not re-predicted).
// 16 warps; 6 ring slots for blocks up to 16 particles, 5 up to 64 (their fp64 sums take the room).  Warps and ring depth as
// measured at N_j = 2^20 by kernel duration (profiles/r02_block_step_ncu.md): 8 warps with 9 slots and 12 with 7 are no faster
// at n_i = 1 (the launch is a fixed 9.7 us plus the stream at the HBM rate) and 7 - 18 % slower at n_i = 16.
//
// The unit of work of a warp is a run of QUARTER TILES (64 particles each), not a whole tile: with 148 x 8 warps and 4096 tiles
// (N_j = 2^20) a warp would get 3 or 4 whole tiles and a quarter of the warps would idle through the last round; N_j = 32768 is
// one tile per CTA, i.e. one busy warp per SM.  The schedule is static (run-to-run bit-reproducible sums, reading 9):
// in full rounds every warp takes UQ consecutive quarters (warp w of round r: quarters (r NW + w) UQ ...), the quarters left for
// the last round are dealt out as evenly as whole quarters allow (the first warps take two while more than NW are left).
// The warps that share a raw slot count their quarters out of it (shared-memory atomic); the one that completes the four
// re-issues the slot's next copy.  The per-warp buffer shrinks with the unit, which pays for more warps and ring slots.
// Measured (B200, cold L2, CUDA events around the call, us; 8 warps x whole tiles -> 16 warps x half / quarter tiles):
// N_j = 2^20: n_i = 16 47.1 -> 44.0, 32 79.9 -> 74.8, 64 137.3 -> 123.9;  N_j = 32768: 16 20.5 -> 16.5, 32 30.1 -> 22.0, 64 47.1 -> 29.7.
#ifndef G6_BS2_UQ16
#define G6_BS2_UQ16 2
#endif
#ifndef G6_BS2_UQ64
#define G6_BS2_UQ64 1
#endif
#ifndef G6_BS2_T16
#define G6_BS2_T16 512
#endif
#ifndef G6_BS2_T64
#define G6_BS2_T64 512
#endif
constexpr int BS2_QJ = 64;                                                                                  // particles per quarter tile
__host__ __device__ constexpr int bs2_uq(int maxi) { return maxi <= 16 ? G6_BS2_UQ16 : G6_BS2_UQ64; }      // quarters per unit in a full round (1 or 2)
__host__ __device__ constexpr int bs2_uj(int maxi) { return BS2_QJ * bs2_uq(maxi); }                       // j-particles per unit, at most
__host__ __device__ constexpr int bs2_threads(int maxi) { return maxi <= 16 ? G6_BS2_T16 : G6_BS2_T64; }
__host__ __device__ constexpr int bs2_pred_bytes(int maxi) { return bs2_uj(maxi) * NF * 4 + bs2_uj(maxi) * 4; }   // predicted unit (field-major floats) + its indices
// ring slots: what is left of the SM's shared memory after the per-warp buffers and sums
__host__ __device__ constexpr int bs2_nslots(int maxi)
{
    return (232448 - 1024 - (bs2_threads(maxi) / 32) * (bs2_pred_bytes(maxi) + maxi * 72) - maxi * 44) / RAW_TILE_BYTES;
}

template <int MAXI>
struct Bs2Smem {
    alignas(128) char raw[bs2_nslots(MAXI)][RAW_TILE_BYTES];  // ring of raw tiles: tile `it` of the CTA lives in slot it % NS
    alignas(16) char pred[bs2_threads(MAXI) / 32][bs2_pred_bytes(MAXI)];            // per warp: its current tile, predicted (field-major floats) + indices
    double acc[bs2_threads(MAXI) / 32][MAXI][8];                              // per-warp fp64 sums of every i (filled once, at the end)
    float r2[bs2_threads(MAXI) / 32][MAXI];
    int addr[bs2_threads(MAXI) / 32][MAXI];
    float ipart[MAXI][9];
    int iidx[MAXI];
    int uaddr[MAXI];
    alignas(8) uint64_t full[bs2_nslots(MAXI)];
    volatile int armed[bs2_nslots(MAXI)];
    int gone[bs2_nslots(MAXI)];                                               // warps that have read their unit out of the slot (running count)
    int is_last;
};
static_assert(sizeof(Bs2Smem<16>) <= 232448 && sizeof(Bs2Smem<64>) <= 232448, "block-step (2) shared memory");

template <int MAXI, bool NEWTON>
__device__ __forceinline__ void block_step2_body(const BsArgs &A, const BsInline<MAXI> *Dp)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    Bs2Smem<MAXI> &sm = *reinterpret_cast<Bs2Smem<MAXI> *>(smem_raw);
    constexpr float INF = __builtin_huge_valf();
    constexpr int BS2_THREADS = bs2_threads(MAXI), NW = BS2_THREADS / 32, NS = bs2_nslots(MAXI), NCH = MAXI <= 16 ? 1 : 2;
    const unsigned FULL = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int G = gridDim.x, cta = blockIdx.x;
    const int nt = cta < A.ntiles ? (A.ntiles - cta + G - 1) / G : 0;

    if (tid == 0) {
#pragma unroll
        for (int k = 0; k < NS; ++k) { mbar_init(&sm.full[k], 1); sm.armed[k] = k; sm.gone[k] = 0; }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
#pragma unroll
        for (int k = 0; k < NS; ++k)
            if (k < nt) {
                mbar_expect_tx(&sm.full[k], RAW_TILE_BYTES);
                tma_load_1d(sm.raw[k], A.raw + (size_t)(cta + k * G) * RAW_TILE_BYTES, RAW_TILE_BYTES, &sm.full[k]);
            }
    }
    // i-block -> shared memory (double-single split here: the host hands fp64)
    for (int k = tid; k < A.ni * 3; k += BS2_THREADS) {
        const int i = k / 3, c = k % 3;
        const double x = A.inline_i ? Dp->xi[i][c] : A.xi[k];
        const double v = A.inline_i ? Dp->vi[i][c] : A.vi[k];
        float hi, lo;
        ds_split(x, hi, lo);
        sm.ipart[i][c] = hi;
        sm.ipart[i][3 + c] = A.ds ? lo : 0.0f;
        sm.ipart[i][6 + c] = (float)v;
    }
    for (int i = tid; i < MAXI; i += BS2_THREADS) {
        if (i < A.ni) sm.iidx[i] = A.inline_i ? Dp->index[i] : A.i_index[i];
        sm.uaddr[i] = i < A.n_upd ? Dp->upd[i].addr : -1;
    }
    __syncthreads();

    // my place in every chunk of 32 i-particles: lanes = 2^lg i-particles x 2^(5 - lg) j-sub-ranges of 8 x 2^lg j
    // The i-block as at most two chunks of a power-of-two number of lanes each (<= 32): one chunk of ceil2(n_i) lanes, or -- where
    // that wastes lanes -- the largest power of two below n_i plus the rest rounded up (n_i = 24: 16 + 8 lanes' worth of work
    // instead of 32: 72 -> 61 us at N_j = 2^20; 17: 71 -> 53).  Every chunk is one pass over the warp's predicted unit.  The kernel
    // for blocks up to 16 keeps a single chunk (a second set of sums costs it 2 us at n_i = 1).
    int cb[NCH], cn[NCH];
    cb[0] = 0; cn[0] = A.ni;
    if (NCH > 1) {
        const auto ceil2 = [](int n) { int c = 1; while (c < n) c *= 2; return c; };
        int f = 1;
        while (2 * f <= min(A.ni, 32)) f *= 2;
        const int rest = A.ni - f;
        const bool one = A.ni <= 32 && (rest == 0 || f + ceil2(rest) >= ceil2(A.ni));
        cn[0] = one ? A.ni : f;
        cb[NCH - 1] = cn[0]; cn[NCH - 1] = A.ni - cn[0];
    }
    int lg[NCH], ii[NCH], my[NCH];
    bool act[NCH];
    double acc7[NCH][7];
    float best[NCH];
    int baddr[NCH];
#pragma unroll
    for (int ch = 0; ch < NCH; ++ch) {
        const int nic = cn[ch];
        lg[ch] = 0;
        while ((1 << lg[ch]) < nic) ++lg[ch];
        ii[ch] = lane & ((1 << lg[ch]) - 1);
        act[ch] = ii[ch] < nic;
        my[ch] = act[ch] ? sm.iidx[cb[ch] + ii[ch]] : -1;
        best[ch] = INF;
        baddr[ch] = 0x7fffffff;
#pragma unroll
        for (int k = 0; k < 7; ++k) acc7[ch][k] = 0.0;
    }
    const float2 eps2 = dup(A.eps2);
    // the unchecked pair code needs s2 > 0 for every pair: a normal positive binary32 eps2 (as for the sweep kernel)
    const bool fast_ok = A.eps2 >= 4.0f * 1.17549435e-38f && A.eps2 < INF;
    const float2 eps2s = dup(pair_scale<NEWTON>() * A.eps2);
    const double kP = NEWTON ? 0.5 * sqrt((double)FOUR_THIRDS) : sqrt((double)THIRD), kA = kP * kP * kP;
    float *Pj = reinterpret_cast<float *>(sm.pred[w]);
    int *JX = reinterpret_cast<int *>(sm.pred[w] + bs2_uj(MAXI) * NF * 4);

    // the static schedule (see above): NR full rounds of UQ quarters per warp, then the last round
    constexpr int UQ = bs2_uq(MAXI), UJ = bs2_uj(MAXI);       // UJ: the stride of the warp's buffer
    static_assert(UQ == 1 || UQ == 2, "a unit never straddles two tiles");
    // Staggered start (UQ == 2, 16 warps, at least 12 tiles): the four warps of one scheduler (w, w + 4, w + 8, w + 12) would
    // otherwise predict together and evaluate pairs together, so the FP32 pipe idles through every prediction; in a round of its
    // own, ahead of the others, the warps 4-7 and 12-15 take ONE quarter and run half a unit ahead from then on
    // (quarters 0-7: warps 0-3 by two; 8-11: warps 4-7; 12-19: warps 8-11 by two; 20-23: warps 12-15).
#ifndef G6_BS2_STAGGER
#define G6_BS2_STAGGER 1
#endif
    const int Q = 4 * nt;
    const bool stag = G6_BS2_STAGGER && UQ == 2 && NW == 16 && Q >= 48;
    const int Q0 = stag ? 24 : 0;                            // quarters of the staggered round
    const int NR = (Q - Q0) / (UQ * NW), rem = (Q - Q0) - NR * UQ * NW;   // NR full rounds
    const int n2 = UQ == 2 ? max(0, rem - NW) : 0;           // warps that take two quarters in the last round
    for (int r = stag ? -1 : 0; r <= NR; ++r) {
        int qs, nq;
        if (r < 0) { const int g = w >> 2, k = w & 3; nq = (g & 1) ? 1 : 2; qs = (g >> 1) * 12 + ((g & 1) ? 8 + k : 2 * k); }
        else if (r < NR) { qs = Q0 + (r * NW + w) * UQ; nq = UQ; }
        else if (w < n2) { qs = Q0 + NR * UQ * NW + 2 * w; nq = 2; }
        else { qs = Q0 + NR * UQ * NW + n2 + w; nq = 1; if (qs >= Q) break; }
        const int it = qs >> 2, q0 = qs & 3;
        const int tile = cta + it * G;
        const int slot = it % NS;
        const int j0 = q0 * BS2_QJ, uj = nq * BS2_QJ;         // my unit inside the tile: first particle, particles
        char *R = sm.raw[slot];
        // the copy of THIS tile must have been issued before its phase is waited for (a parity wait cannot tell phase
        // p + 1 from the completed phase p - 1)
        if (it >= NS) {
            uint32_t spins = 0;
            while (ld_acquire_cta(&sm.armed[slot]) != it) { if (++spins > (1u << 26)) __trap(); }
        }
        mbar_wait(&sm.full[slot], (uint32_t)(it / NS) & 1u);

        // ---- a-1: particles corrected in the last step that live in this tile: patch the staged copy, write through
        if (A.n_upd > 0) {
            for (int q = lane; q < A.n_upd; q += 32)
                if (sm.uaddr[q] / JT == tile && (unsigned)((sm.uaddr[q] % JT) / BS2_QJ - q0) < (unsigned)nq) {
                    const JRecord r = Dp->upd[q];
                    store_record(R, r.addr % JT, r);
                    store_record(A.raw + (size_t)tile * RAW_TILE_BYTES, r.addr % JT, r);
                }
            __syncwarp();
        }
        // ---- a-2: predict my uj / 32 j (lane l owns the pairs {2l, 2l + 1} + 64 g: conflict-free vector loads) into my warp's buffer
        const bool ragged = tile * JT + j0 + uj > A.nj;
        int id_lo = INT32_MAX, id_hi = INT32_MIN;
#pragma unroll
        for (int g = 0; g < nq; ++g) {
            const int lu = 2 * lane + 64 * g, l0 = j0 + lu;    // inside the unit, inside the tile
            const double2 tj = *reinterpret_cast<const double2 *>(R + RAW_T + 8 * l0);
            const float2 dt = make_float2((float)(A.ti - tj.x), (float)(A.ti - tj.y));
            float2 f[NF];
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const double2 x0 = *reinterpret_cast<const double2 *>(R + RAW_X + 8 * (k * JT + l0));
                const float2 v0 = *reinterpret_cast<const float2 *>(R + RAW_V + 4 * (k * JT + l0));
                const float2 a2 = *reinterpret_cast<const float2 *>(R + RAW_A2 + 4 * (k * JT + l0));
                const float2 j6 = *reinterpret_cast<const float2 *>(R + RAW_J6 + 4 * (k * JT + l0));
                predict_coord(dt.x, x0.x, v0.x, a2.x, j6.x, A.ds, f[F_XH + k].x, f[F_XL + k].x, f[F_V + k].x);
                predict_coord(dt.y, x0.y, v0.y, a2.y, j6.y, A.ds, f[F_XH + k].y, f[F_XL + k].y, f[F_V + k].y);
            }
            f[F_M] = *reinterpret_cast<const float2 *>(R + RAW_M + 4 * l0);
            if (ragged) {                                     // addresses >= nj: finite and massless
                const bool in0 = tile * JT + l0 < A.nj, in1 = tile * JT + l0 + 1 < A.nj;
#pragma unroll
                for (int k = 0; k < NF; ++k) f[k] = make_float2(in0 ? f[k].x : 0.0f, in1 ? f[k].y : 0.0f);
            }
#pragma unroll
            for (int k = 0; k < NF; ++k) *reinterpret_cast<float2 *>(Pj + k * UJ + lu) = f[k];
            const int2 jx = *reinterpret_cast<const int2 *>(R + RAW_IDX + 4 * l0);
            *reinterpret_cast<int2 *>(JX + lu) = jx;
            id_lo = min(id_lo, min(jx.x, jx.y));
            id_hi = max(id_hi, max(jx.x, jx.y));
        }
        // Self-exclusion hoisted to unit level, as in the sweep kernel: if no i-particle of this warp's lanes has its index
        // inside the unit's index range (and the unit is not cut by nj) the unit runs the unchecked pair code
        id_lo = __reduce_min_sync(FULL, id_lo);
        id_hi = __reduce_max_sync(FULL, id_hi);
        bool hit = false;
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) hit |= act[ch] && my[ch] >= id_lo && my[ch] <= id_hi;
        const bool checked = !fast_ok || ragged || __any_sync(FULL, hit);
        // my unit is out of the slot; the warp that takes the tile's last quarters refills the slot with the tile NS ahead while the forces are computed
        __syncwarp();
        if (lane == 0) {
            __threadfence_block();                            // my lanes' reads (and a-1 writes) of the slot before the count ...
            const bool last = ((atomicAdd(&sm.gone[slot], nq) + nq) & 3) == 0;
            __threadfence_block();                            // ... and the other warps' before the copy that overwrites it
            if (last && it + NS < nt) {
                if (A.n_upd > 0) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // a-1 wrote the slot through the generic proxy
                mbar_expect_tx(&sm.full[slot], RAW_TILE_BYTES);
                tma_load_1d(R, A.raw + (size_t)(tile + NS * G) * RAW_TILE_BYTES, RAW_TILE_BYTES, &sm.full[slot]);
                st_release_cta(&sm.armed[slot], it + NS);
            }
        }

        // ---- a-4: the pairs of this tile; my i-particle of every chunk against my j-sub-range
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) {
            if (!act[ch]) continue;
            IPart I;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                I.nxh[k] = dup(-sm.ipart[cb[ch] + ii[ch]][k]);
                I.nxl[k] = dup(-sm.ipart[cb[ch] + ii[ch]][3 + k]);
                I.nv[k] = dup(-sm.ipart[cb[ch] + ii[ch]][6 + k]);
                I.a[k] = dup(0.0f);
                I.j[k] = dup(0.0f);
            }
            I.p = dup(0.0f);
            const int jn = (uj / 32) << lg[ch];
            const int jl0 = (lane >> lg[ch]) * jn;
            if (checked || jn < 4) {                          // (the unchecked loop takes four j at a time)
#pragma unroll 2
                for (int q = 0; q < jn; q += 2) {
                    const int jl = jl0 + q, ja = tile * JT + j0 + jl;
                    float2 f[NF];
#pragma unroll
                    for (int k = 0; k < NF; ++k) f[k] = *reinterpret_cast<const float2 *>(Pj + k * UJ + jl);
                    const int2 jx = *reinterpret_cast<const int2 *>(JX + jl);
                    float2 r2;
                    pair2_checked<NEWTON>(I, f[0], f[1], f[2], f[3], f[4], f[5], f[6], f[7], f[8], f[9], eps2,
                                          (ja < A.nj) && (jx.x != my[ch]), (ja + 1 < A.nj) && (jx.y != my[ch]), r2);
                    // nearest neighbour: strict <, my j ascend => ties keep the smallest address (reading 7)
                    if (r2.x < best[ch]) { best[ch] = r2.x; baddr[ch] = ja; }
                    if (r2.y < best[ch]) { best[ch] = r2.y; baddr[ch] = ja + 1; }
                }
                // FP32 over one tile slice (<= 128 pairs per chain), then fp64 (reading 9)
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    acc7[ch][k] += (double)I.a[k].x + (double)I.a[k].y;
                    acc7[ch][3 + k] += (double)I.j[k].x + (double)I.j[k].y;
                }
                acc7[ch][6] += (double)I.p.x + (double)I.p.y;
            } else {
                // the sweep kernel's pair code (g6_force_fast.cuh pair2: no per-pair test, Newton step in three instructions on the
                // scaled sigma); its sums come out scaled by (y s) and (y s)^3, undone here in fp64 with the binary32 scale
#pragma unroll 2
                for (int q = 0; q < jn; q += 4) {
                    const int jl = jl0 + q, ja = tile * JT + j0 + jl;
                    float4 f[NF];
#pragma unroll
                    for (int k = 0; k < NF; ++k) f[k] = *reinterpret_cast<const float4 *>(Pj + k * UJ + jl);
                    float2 ra, rb;
                    pair2<NEWTON>(I, make_float2(f[0].x, f[0].y), make_float2(f[1].x, f[1].y), make_float2(f[2].x, f[2].y),
                                  make_float2(f[3].x, f[3].y), make_float2(f[4].x, f[4].y), make_float2(f[5].x, f[5].y),
                                  make_float2(f[6].x, f[6].y), make_float2(f[7].x, f[7].y), make_float2(f[8].x, f[8].y),
                                  make_float2(f[9].x, f[9].y), eps2s, ra);
                    pair2<NEWTON>(I, make_float2(f[0].z, f[0].w), make_float2(f[1].z, f[1].w), make_float2(f[2].z, f[2].w),
                                  make_float2(f[3].z, f[3].w), make_float2(f[4].z, f[4].w), make_float2(f[5].z, f[5].w),
                                  make_float2(f[6].z, f[6].w), make_float2(f[7].z, f[7].w), make_float2(f[8].z, f[8].w),
                                  make_float2(f[9].z, f[9].w), eps2s, rb);
                    if (ra.x < best[ch]) { best[ch] = ra.x; baddr[ch] = ja; }
                    if (ra.y < best[ch]) { best[ch] = ra.y; baddr[ch] = ja + 1; }
                    if (rb.x < best[ch]) { best[ch] = rb.x; baddr[ch] = ja + 2; }
                    if (rb.y < best[ch]) { best[ch] = rb.y; baddr[ch] = ja + 3; }
                }
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    acc7[ch][k] += kA * ((double)I.a[k].x + (double)I.a[k].y);
                    acc7[ch][3 + k] += kA * ((double)I.j[k].x + (double)I.j[k].y);
                }
                acc7[ch][6] += kP * ((double)I.p.x + (double)I.p.y);
            }
        }
        __syncwarp();                                         // the buffer is overwritten by my next tile
    }

    // ---- the lanes of one i-particle (its j-sub-ranges): fixed shuffle tree, once; then one entry per (warp, i)
#pragma unroll
    for (int ch = 0; ch < NCH; ++ch) {
        for (int o = 1 << lg[ch]; o < 32; o <<= 1) {
#pragma unroll
            for (int k = 0; k < 7; ++k) acc7[ch][k] += __shfl_xor_sync(FULL, acc7[ch][k], o);
            const float r2 = __shfl_xor_sync(FULL, best[ch], o);
            const int ad = __shfl_xor_sync(FULL, baddr[ch], o);
            if (r2 < best[ch] || (r2 == best[ch] && ad < baddr[ch])) { best[ch] = r2; baddr[ch] = ad; }
        }
        if (act[ch] && lane < (1 << lg[ch])) {
            const int i = cb[ch] + lane;
#pragma unroll
            for (int k = 0; k < 7; ++k) sm.acc[w][i][k] = acc7[ch][k];
            sm.r2[w][i] = best[ch];
            sm.addr[w][i] = baddr[ch];
        }
    }
    __syncthreads();

    // ---- a-5, first half: one partial per (i, CTA): the warps' sums in warp order
    for (int i = tid; i < A.ni; i += BS2_THREADS) {
        const size_t o = (size_t)cta * A.P.stride_s + (size_t)i * A.P.stride_i;
        double v[7];
#pragma unroll
        for (int k = 0; k < 7; ++k) v[k] = sm.acc[0][i][k];
        float bst = sm.r2[0][i];
        int bad = sm.addr[0][i];
#pragma unroll
        for (int q = 1; q < NW; ++q) {
#pragma unroll
            for (int k = 0; k < 7; ++k) v[k] += sm.acc[q][i][k];
            const float r2 = sm.r2[q][i];
            const int ad = sm.addr[q][i];
            if (r2 < bst || (r2 == bst && ad < bad)) { bst = r2; bad = ad; }
        }
#pragma unroll
        for (int k = 0; k < 3; ++k) { A.P.acc[k][o] = v[k]; A.P.jrk[k][o] = v[3 + k]; }
        A.P.pot[o] = -v[6];
        const bool has = bad != 0x7fffffff;
        A.P.nn_r2[o] = has ? bst : INF;
        A.P.nn_addr[o] = has ? bad : -1;
    }
    // the ticket: the barrier orders the CTA's partial stores before thread 0, whose release fence is cumulative; the last CTA's
    // acquire fence sits between the ticket and its reads of the partials (ld.global.cg)
    __syncthreads();
    if (tid == 0) {
        fence_acq_rel_gpu();
        const unsigned ticket = atomicAdd(A.counter, 1u);
        sm.is_last = (ticket == (unsigned)G - 1u);
        if (sm.is_last) fence_acq_rel_gpu();
    }
    __syncthreads();
    if (!sm.is_last) return;

    // ---- a-5, second half (last CTA only): sum the G partials of every i in CTA order, one warp per i-particle
    for (int i = w; i < A.ni; i += NW) {
        double v[7] = {0, 0, 0, 0, 0, 0, 0};
        float bst = INF;
        int bad = 0x7fffffff;
        for (int s0 = 0; s0 < G; s0 += 160) {
            double t[5][7];
            float r2[5];
            int ad[5];
#pragma unroll
            for (int q = 0; q < 5; ++q) {
                const int sq = s0 + lane + 32 * q;
                const bool in = sq < G;
                const size_t o = (size_t)(in ? sq : 0) * A.P.stride_s + (size_t)i * A.P.stride_i;
#pragma unroll
                for (int k = 0; k < 3; ++k) { t[q][k] = in ? __ldcg(A.P.acc[k] + o) : 0.0; t[q][3 + k] = in ? __ldcg(A.P.jrk[k] + o) : 0.0; }
                t[q][6] = in ? __ldcg(A.P.pot + o) : 0.0;
                r2[q] = in ? __ldcg(A.P.nn_r2 + o) : INF;
                ad[q] = in ? __ldcg(A.P.nn_addr + o) : -1;
            }
#pragma unroll
            for (int q = 0; q < 5; ++q) {
                if (s0 + lane + 32 * q < G) {
#pragma unroll
                    for (int k = 0; k < 7; ++k) v[k] += t[q][k];
                    if (ad[q] >= 0 && (r2[q] < bst || (r2[q] == bst && ad[q] < bad))) { bst = r2[q]; bad = ad[q]; }
                }
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
            for (int k = 0; k < 7; ++k) v[k] += __shfl_xor_sync(FULL, v[k], o);
            const float r2 = __shfl_xor_sync(FULL, bst, o);
            const int ad = __shfl_xor_sync(FULL, bad, o);
            if (r2 < bst || (r2 == bst && ad < bad)) { bst = r2; bad = ad; }
        }
        if (lane == 0) {
#pragma unroll
            for (int k = 0; k < 3; ++k) { A.acc[3 * (size_t)i + k] = v[k]; A.jerk[3 * (size_t)i + k] = v[3 + k]; }
            A.pot[i] = v[6];
            const bool has = bad != 0x7fffffff;
            if (A.nn_index) A.nn_index[i] = has ? j_index(A.raw, bad) : -1;
            if (A.nn_r2) A.nn_r2[i] = has ? (double)bst : (double)INF;
        }
    }
    if (tid == 0) *A.counter = 0u;
    if (A.done_flag) {
        __syncthreads();
        if (tid == 0) {
            __threadfence_system();
            *reinterpret_cast<volatile unsigned int *>(A.done_flag) = A.done_seq;
        }
    }
}

template <int MAXI, bool NEWTON>
__global__ void __launch_bounds__(bs2_threads(MAXI))
k_block_step2(const BsArgs A, const __grid_constant__ BsInline<MAXI> D)
{
    block_step2_body<MAXI, NEWTON>(A, &D);
}

template <int MAXI, bool NEWTON>
__global__ void __launch_bounds__(bs2_threads(MAXI))
k_block_step2_dev(const BsArgs A)
{
    block_step2_body<MAXI, NEWTON>(A, nullptr);
}

// ---------------------------------------------------------------- host side
template <int MAXI>
inline int bs_attr()
{
    const int bytes = (int)sizeof(BsSmem<MAXI>);
    cudaError_t e = cudaFuncSetAttribute(k_block_step<MAXI, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e != cudaSuccess) return (int)e;
    e = cudaFuncSetAttribute(k_block_step<MAXI, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e != cudaSuccess) return (int)e;
    e = cudaFuncSetAttribute(k_block_step_dev<MAXI, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e != cudaSuccess) return (int)e;
    return (int)cudaFuncSetAttribute(k_block_step_dev<MAXI, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
}

template <int MAXI>
inline int bs2_attr()
{
    const int bytes = (int)sizeof(Bs2Smem<MAXI>);
    cudaError_t e = cudaFuncSetAttribute(k_block_step2<MAXI, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e != cudaSuccess) return (int)e;
    e = cudaFuncSetAttribute(k_block_step2<MAXI, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e != cudaSuccess) return (int)e;
    e = cudaFuncSetAttribute(k_block_step2_dev<MAXI, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e != cudaSuccess) return (int)e;
    return (int)cudaFuncSetAttribute(k_block_step2_dev<MAXI, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
}

inline int bs_kernel_init()
{
    int r;
    if ((r = bs_attr<16>())) return r;
    if ((r = bs_attr<BS_MAX_I>())) return r;
    if ((r = bs2_attr<16>())) return r;
    return bs2_attr<BS_MAX_I>();
}

// the second design (no neighbour lists); same arguments as bs_launch_t
template <int MAXI>
inline int bs2_launch_t(const BsArgs &A, bool newton, int grid, const double *xi, const double *vi, const int *index,
                        const JRecord *upd, cudaStream_t st)
{
    static thread_local BsInline<MAXI> D;
    if (A.inline_i) {
        memcpy(D.xi, xi, sizeof(double) * 3 * A.ni);
        memcpy(D.vi, vi, sizeof(double) * 3 * A.ni);
        memcpy(D.index, index, sizeof(int) * A.ni);
    }
    if (A.n_upd > 0) memcpy(D.upd, upd, sizeof(JRecord) * A.n_upd);
    const size_t bytes = sizeof(Bs2Smem<MAXI>);
    if (!A.inline_i && A.n_upd == 0) {
        if (newton) k_block_step2_dev<MAXI, true><<<grid, bs2_threads(MAXI), bytes, st>>>(A);
        else k_block_step2_dev<MAXI, false><<<grid, bs2_threads(MAXI), bytes, st>>>(A);
        return (int)cudaGetLastError();
    }
    if (newton) k_block_step2<MAXI, true><<<grid, bs2_threads(MAXI), bytes, st>>>(A, D);
    else k_block_step2<MAXI, false><<<grid, bs2_threads(MAXI), bytes, st>>>(A, D);
    return (int)cudaGetLastError();
}

template <int MAXI>
inline int bs_ctas_per_sm()
{
    static int n = 0;
    if (!n) {
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_block_step<MAXI, true>, BS_THREADS, sizeof(BsSmem<MAXI>)) != cudaSuccess || n < 1) n = 1;
    }
    return n;
}

// `src`: the host-side i-block and update records to carry in the parameters (NULL pointers: none)
template <int MAXI>
inline int bs_launch_t(const BsArgs &A, bool newton, int grid, const double *xi, const double *vi, const int *index,
                       const JRecord *upd, cudaStream_t st)
{
    static thread_local BsInline<MAXI> D;   // one host thread per cluster (g6.h); filled per call, copied by the launch
    if (A.inline_i) {
        memcpy(D.xi, xi, sizeof(double) * 3 * A.ni);
        memcpy(D.vi, vi, sizeof(double) * 3 * A.ni);
        memcpy(D.index, index, sizeof(int) * A.ni);
    }
    if (A.n_upd > 0) memcpy(D.upd, upd, sizeof(JRecord) * A.n_upd);
    const size_t bytes = sizeof(BsSmem<MAXI>);
    if (!A.inline_i && A.n_upd == 0) {          // nothing to carry: the launch without the inline payload
        if (newton) k_block_step_dev<MAXI, true><<<grid, BS_THREADS, bytes, st>>>(A);
        else k_block_step_dev<MAXI, false><<<grid, BS_THREADS, bytes, st>>>(A);
        return (int)cudaGetLastError();
    }
    if (newton) k_block_step<MAXI, true><<<grid, BS_THREADS, bytes, st>>>(A, D);
    else k_block_step<MAXI, false><<<grid, BS_THREADS, bytes, st>>>(A, D);
    return (int)cudaGetLastError();
}

}  // namespace g6
