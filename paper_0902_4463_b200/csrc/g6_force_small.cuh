// g6_force_small.cuh -- force kernel for the small active blocks of block time steps (n_i <= 64),
// with the j-predictor fused in (steps a-2 + a-4 in one pass over the j-store).
//
// For a handful of i-particles there is nothing to gain from holding i in registers: the step is
// bound by the one pass over the N_j stored particles and by launch latency (SURVEY.md 8(d):
// 176 B per j for predict + force as two kernels, 76 B fused).  So the roles are swapped, the
// paper's Fig. 4 idea (when there are fewer i than threads, several threads
// share an i and split the j) taken to its limit: every LANE owns 8 j-particles of one tile,
// predicts them once (Eq. 1-2, same arithmetic as k_predict) into registers, then loops over the
// i-particles (broadcast from shared memory), evaluates its 8 pairs in FP32 with double-single
// separations (Eq. 3), and the warp reduces the 32 lane sums in fp64 with shuffles ("keeps the
// neighbour min-reduction in warp shuffles").  One warp per tile => S = number of tiles partial
// results per i, combined by k_combine_wide / k_combine_block.  Every pair is checked
// (address < nj, index_j != index_i, s2 > 0), so this path also serves eps2 = 0.
#pragma once
#include "g6_force_ref.cuh"

namespace g6 {

constexpr int SMALL_MAX_I = 64;
constexpr int SMALL_JPL = JT / 32;   // j-particles per lane

struct SmallArgs {
    JStore js;                // raw j store (predict fused) ...
    double ti;
    const float *pred;        // ... or predicted tiles when they are already valid for ti (fused = 0)
    int fused;
    int nj, ntiles;
    const int *i_index;
    const double *xi, *vi;
    int ni;
    float eps2;
    int ds;
    Partials P;               // [i][s] layout: stride_s = 1, stride_i = ntiles
};

template <bool NEWTON>
__global__ void __launch_bounds__(128)
k_force_small(SmallArgs A)
{
    __shared__ float s_i[SMALL_MAX_I][9];
    __shared__ int s_idx[SMALL_MAX_I];
    const int tid = threadIdx.x, lane = tid & 31;
    const int tile = blockIdx.x * 4 + (tid >> 5);
    constexpr float INF = __builtin_huge_valf();

    for (int k = tid; k < A.ni * 3; k += 128) {
        const int i = k / 3, c = k % 3;
        float hi, lo;
        ds_split(A.xi[k], hi, lo);
        s_i[i][c] = hi;
        s_i[i][3 + c] = A.ds ? lo : 0.0f;
        s_i[i][6 + c] = (float)A.vi[k];
    }
    for (int k = tid; k < A.ni; k += 128) s_idx[k] = A.i_index[k];
    __syncthreads();
    if (tile >= A.ntiles) return;

    // ---- my 8 j-particles: predicted into registers
    float xh[SMALL_JPL][3], xl[SMALL_JPL][3], vj[SMALL_JPL][3], mj[SMALL_JPL];
    int jid[SMALL_JPL];
    bool jok[SMALL_JPL];
#pragma unroll
    for (int u = 0; u < SMALL_JPL; ++u) {
        const int l = 32 * u + lane;
        const int j = tile * JT + l;
        jok[u] = j < A.nj;
        jid[u] = 0;
        mj[u] = 0.0f;
#pragma unroll
        for (int k = 0; k < 3; ++k) { xh[u][k] = xl[u][k] = vj[u][k] = 0.0f; }
        if (jok[u]) {
            jid[u] = A.js.idx[j];
            if (A.fused) {
                const float dt = (float)(A.ti - A.js.t[j]);
                const float dt3 = 3.0f * dt;
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    const float v0 = A.js.v[k][j], a2 = A.js.a2[k][j], j6 = A.js.j6[k][j];
                    const float d = __fmul_rn(dt, __fmaf_rn(dt, __fmaf_rn(dt, j6, a2), v0));
                    const double xp = A.js.x[k][j] + (double)d;
                    ds_split(xp, xh[u][k], xl[u][k]);
                    if (!A.ds) xl[u][k] = 0.0f;
                    vj[u][k] = __fmaf_rn(dt, __fmaf_rn(dt3, j6, __fadd_rn(a2, a2)), v0);
                }
                mj[u] = A.js.m[j];
            } else {
                const float *g = A.pred + (size_t)tile * TILE_FLOATS + l;
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    xh[u][k] = g[(F_XH + k) * JT];
                    xl[u][k] = g[(F_XL + k) * JT];
                    vj[u][k] = g[(F_V + k) * JT];
                }
                mj[u] = g[F_M * JT];
            }
        }
    }

    for (int i = 0; i < A.ni; ++i) {
        const float xih = s_i[i][0], yih = s_i[i][1], zih = s_i[i][2];
        const float xil = s_i[i][3], yil = s_i[i][4], zil = s_i[i][5];
        const float vix = s_i[i][6], viy = s_i[i][7], viz = s_i[i][8];
        const int my = s_idx[i];
        float a32[3] = {0, 0, 0}, j32[3] = {0, 0, 0}, p32 = 0;
        float best = INF;
        int baddr = 0x7fffffff;
#pragma unroll
        for (int u = 0; u < SMALL_JPL; ++u) {
            const float dx = ds_dx(xh[u][0], xl[u][0], xih, xil);
            const float dy = ds_dx(xh[u][1], xl[u][1], yih, yil);
            const float dz = ds_dx(xh[u][2], xl[u][2], zih, zil);
            const float dvx = __fsub_rn(vj[u][0], vix);
            const float dvy = __fsub_rn(vj[u][1], viy);
            const float dvz = __fsub_rn(vj[u][2], viz);
            const float r2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
            const float s2 = __fadd_rn(r2, A.eps2);
            const bool ok = jok[u] && (jid[u] != my) && (s2 > 0.0f);
            const float s2c = ok ? s2 : 1.0f;
            float rinv = rsqrt_approx(s2c);
            if (NEWTON) {
                const float e = __fmaf_rn(s2c, __fmul_rn(rinv, rinv), -1.0f);
                rinv = __fmaf_rn(__fmul_rn(-0.5f, rinv), e, rinv);
            }
            const float m = ok ? mj[u] : 0.0f;
            const float rinv2 = __fmul_rn(rinv, rinv);
            const float mrinv = __fmul_rn(m, rinv);
            const float mrinv3 = __fmul_rn(mrinv, rinv2);
            const float rv = __fmaf_rn(dz, dvz, __fmaf_rn(dy, dvy, __fmul_rn(dx, dvx)));
            const float alpha = __fmul_rn(-3.0f, __fmul_rn(rv, rinv2));
            p32 = __fsub_rn(p32, mrinv);
            a32[0] = __fmaf_rn(mrinv3, dx, a32[0]);
            a32[1] = __fmaf_rn(mrinv3, dy, a32[1]);
            a32[2] = __fmaf_rn(mrinv3, dz, a32[2]);
            j32[0] = __fmaf_rn(mrinv3, __fmaf_rn(alpha, dx, dvx), j32[0]);
            j32[1] = __fmaf_rn(mrinv3, __fmaf_rn(alpha, dy, dvy), j32[1]);
            j32[2] = __fmaf_rn(mrinv3, __fmaf_rn(alpha, dz, dvz), j32[2]);
            // ascending address within the lane (u outer): strict < keeps the first
            if (ok && r2 < best) { best = r2; baddr = tile * JT + 32 * u + lane; }
        }
        // warp reduction: fp64 sums (fixed xor tree => bit-reproducible), (r2, address) lexicographic min
        double v[7] = {(double)a32[0], (double)a32[1], (double)a32[2], (double)j32[0], (double)j32[1], (double)j32[2], (double)p32};
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
            for (int k = 0; k < 7; ++k) v[k] += __shfl_xor_sync(0xffffffffu, v[k], o);
            const float r2 = __shfl_xor_sync(0xffffffffu, best, o);
            const int ad = __shfl_xor_sync(0xffffffffu, baddr, o);
            if (r2 < best || (r2 == best && ad < baddr)) { best = r2; baddr = ad; }
        }
        if (lane == 0) {
            const size_t o = (size_t)tile * A.P.stride_s + (size_t)i * A.P.stride_i;
#pragma unroll
            for (int k = 0; k < 3; ++k) { A.P.acc[k][o] = v[k]; A.P.jrk[k][o] = v[3 + k]; }
            A.P.pot[o] = v[6];
            const bool has = baddr != 0x7fffffff;
            A.P.nn_r2[o] = has ? best : INF;
            A.P.nn_addr[o] = has ? baddr : -1;
        }
    }
}

}  // namespace g6
