// g6_device.cuh -- device data layout and the small kernels of libg6b200 (sm_100a).
//
// Steps of the path:
//   a-1  k_store_from_f64 / k_stage           : keep the j-particle store on the device
//   a-2  k_predict                            : Eq. 1-2, DS positions
//   a-4  force kernels (g6_force_ref.cuh, g6_force_fast.cuh)
//   a-5  k_combine                            : sum the per-split partial forces on the GPU
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace g6 {

// acquire-release fence at device scope.  __threadfence() is the sequentially consistent fence and on sm_100 compiles to MEMBAR.SC.GPU
// plus a whole-L1 invalidate (CCTL.IVALL), microseconds when stores are in flight; the "last CTA" patterns of this library only need
// release (partials before the ticket) and acquire (ticket before the partials, which are then read with ld.global.cg).
__device__ __forceinline__ void fence_acq_rel_gpu() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }


// ---- j-particle store (raw Hermite state at t_j): tiles of JT particles, field-major in a tile --
// "Only the position is stored in DP, whereas the rest of the terms are stored in SP".
// Tile k = RAW_TILE_BYTES bytes at raw + k * RAW_TILE_BYTES:
//   x[3][JT] f64 | t[JT] f64 | v[3][JT] f32 | a/2[3][JT] f32 | j/6[3][JT] f32 | m[JT] f32 | index[JT] i32
// = 76 B per particle, 19 456 B per tile, 16-byte aligned: ONE 1-D TMA bulk copy stages the whole raw
// tile in shared memory (block-step kernel, g6_block_step.cuh); consecutive lanes touching
// consecutive j of one field are coalesced (predictor, scatter).
constexpr int JT = 256;
constexpr int RAW_X = 0;                       // byte offsets inside a raw tile
constexpr int RAW_T = RAW_X + 3 * JT * 8;
constexpr int RAW_V = RAW_T + JT * 8;
constexpr int RAW_A2 = RAW_V + 3 * JT * 4;
constexpr int RAW_J6 = RAW_A2 + 3 * JT * 4;
constexpr int RAW_M = RAW_J6 + 3 * JT * 4;
constexpr int RAW_IDX = RAW_M + JT * 4;
constexpr int RAW_TILE_BYTES = RAW_IDX + JT * 4;
static_assert(RAW_TILE_BYTES == 76 * JT && RAW_TILE_BYTES % 16 == 0, "raw tile layout");

struct JStore {
    char *raw;   // capacity / JT raw tiles
};

// pointers to the fields of particle `a` (k = coordinate)
__host__ __device__ __forceinline__ char *raw_tile(char *raw, int a) { return raw + (size_t)(a / JT) * RAW_TILE_BYTES; }
__device__ __forceinline__ double &raw_x(char *tile, int k, int l) { return reinterpret_cast<double *>(tile + RAW_X)[k * JT + l]; }
__device__ __forceinline__ double &raw_t(char *tile, int l) { return reinterpret_cast<double *>(tile + RAW_T)[l]; }
__device__ __forceinline__ float &raw_v(char *tile, int k, int l) { return reinterpret_cast<float *>(tile + RAW_V)[k * JT + l]; }
__device__ __forceinline__ float &raw_a2(char *tile, int k, int l) { return reinterpret_cast<float *>(tile + RAW_A2)[k * JT + l]; }
__device__ __forceinline__ float &raw_j6(char *tile, int k, int l) { return reinterpret_cast<float *>(tile + RAW_J6)[k * JT + l]; }
__device__ __forceinline__ float &raw_m(char *tile, int l) { return reinterpret_cast<float *>(tile + RAW_M)[l]; }
__device__ __forceinline__ int &raw_idx(char *tile, int l) { return reinterpret_cast<int *>(tile + RAW_IDX)[l]; }
// the caller's index of j address `a`
__device__ __forceinline__ int j_index(const char *raw, int a)
{
    return __ldg(reinterpret_cast<const int *>(raw + (size_t)(a / JT) * RAW_TILE_BYTES + RAW_IDX) + (a % JT));
}
// the 256 indices of tile t (16-byte aligned)
__device__ __forceinline__ const int *tile_indices(const char *raw, int t)
{
    return reinterpret_cast<const int *>(raw + (size_t)t * RAW_TILE_BYTES + RAW_IDX);
}

// one j-particle on its way host -> device (g6_set_j_particle staging); 80 bytes
struct JRecord {
    double x[3];
    double t;
    float v[3], a2[3], j6[3];
    float m;
    int idx;
    int addr;
};

// write one record into slot l of a raw tile (global or shared memory)
__device__ __forceinline__ void store_record(char *T, int l, const JRecord &r)
{
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        raw_x(T, k, l) = r.x[k];
        raw_v(T, k, l) = r.v[k];
        raw_a2(T, k, l) = r.a2[k];
        raw_j6(T, k, l) = r.j6[k];
    }
    raw_t(T, l) = r.t;
    raw_m(T, l) = r.m;
    raw_idx(T, l) = r.idx;
}

// ---- predicted j-particles: tiles of JT particles, field-major inside a tile --------------
// tile k = floats [k*JT*NF, (k+1)*JT*NF): x_hi[JT] y_hi z_hi x_lo y_lo z_lo vx vy vz m.
// One contiguous 10 KiB block per tile = one TMA bulk copy into shared memory; consecutive
// lanes reading consecutive j are coalesced; LDS.128 yields four consecutive j of one field.
constexpr int NF = 10;
constexpr int F_XH = 0, F_XL = 3, F_V = 6, F_M = 9;
constexpr int TILE_FLOATS = JT * NF;
constexpr int TILE_BYTES = TILE_FLOATS * 4;

// ---- partial results of one j-split, structure of arrays, element [s * stride_s + i * stride_i]
// few splits: (stride_s, stride_i) = (ni, 1), one thread per i combines; many splits (small
// blocks): (1, S), one warp per i combines with coalesced reads.
struct Partials {
    double *acc[3];
    double *jrk[3];
    double *pot;
    float *nn_r2;    // unsoftened, +inf when none
    int *nn_addr;    // j address, -1 when none
    int stride_s, stride_i;
};

// double -> double-single (reading 12): hi = RN32(x), lo = RN32(x - hi)
__device__ __forceinline__ void ds_split(double x, float &hi, float &lo)
{
    hi = __double2float_rn(x);
    lo = __double2float_rn(x - (double)hi);
}

// Eq. 3: dx = (xj_hi - xi_hi) + (xj_lo - xi_lo), three binary32 adds
__device__ __forceinline__ float ds_dx(float xj_hi, float xj_lo, float xi_hi, float xi_lo)
{
    return __fadd_rn(__fsub_rn(xj_hi, xi_hi), __fsub_rn(xj_lo, xi_lo));
}

__device__ __forceinline__ float rsqrt_approx(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ---- a-1: bulk load from fp64 device arrays (physical acc, jerk) --------------------------
__global__ void __launch_bounds__(256)
k_store_from_f64(JStore S, int addr0, int n, const int *__restrict__ index, const double *__restrict__ tj,
                 const double *__restrict__ mass, const double *__restrict__ jerk, const double *__restrict__ acc,
                 const double *__restrict__ v, const double *__restrict__ x)
{
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const int a = addr0 + p;
    char *T = raw_tile(S.raw, a);
    const int l = a % JT;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        raw_x(T, k, l) = x[3 * (size_t)p + k];
        raw_v(T, k, l) = (float)v[3 * (size_t)p + k];
        raw_a2(T, k, l) = (float)(acc[3 * (size_t)p + k] * 0.5);
        raw_j6(T, k, l) = (float)(jerk[3 * (size_t)p + k] / 6.0);
    }
    raw_t(T, l) = tj[p];
    raw_m(T, l) = (float)mass[p];
    raw_idx(T, l) = index[p];
}

// ---- a-1 + a-3: scatter of the particles changed since the last force call, and the i block -----
// `rec`, `xi_src`, ... may point into mapped pinned HOST memory (small batches: no DMA set-up
// latency) or into device memory (large batches, after one packed copy).
__global__ void __launch_bounds__(128)
k_stage(JStore S, const JRecord *__restrict__ rec, int n_rec, int n_i, const double *__restrict__ xi_src,
        const double *__restrict__ vi_src, const int *__restrict__ idx_src, double *__restrict__ xi_dst,
        double *__restrict__ vi_dst, int *__restrict__ idx_dst)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p < n_rec) {
        const JRecord r = rec[p];
        char *T = raw_tile(S.raw, r.addr);
        store_record(T, r.addr % JT, r);
    }
    if (p < n_i) {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            xi_dst[3 * p + k] = xi_src[3 * p + k];
            vi_dst[3 * p + k] = vi_src[3 * p + k];
        }
        idx_dst[p] = idx_src[p];
    }
}

// ---- j-particle read-back: records of addresses [addr0, addr0 + n) exactly as stored (x, t fp64; the rest binary32) ----
__global__ void __launch_bounds__(128)
k_fetch_records(JStore S, int addr0, int n, JRecord *__restrict__ out)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const int a = addr0 + p;
    char *T = raw_tile(S.raw, a);
    const int l = a % JT;
    JRecord r;
#pragma unroll
    for (int k = 0; k < 3; ++k) { r.x[k] = raw_x(T, k, l); r.v[k] = raw_v(T, k, l); r.a2[k] = raw_a2(T, k, l); r.j6[k] = raw_j6(T, k, l); }
    r.t = raw_t(T, l);
    r.m = raw_m(T, l);
    r.idx = raw_idx(T, l);
    r.addr = a;
    out[p] = r;
}

// Eq. 1-2 for one coordinate (reading 11): FP32 Horner increment, fp64 add to x0, DS re-split
__device__ __forceinline__ void predict_coord(float dt, double x0, float v0, float a2, float j6, int ds,
                                              float &xh, float &xl, float &vp)
{
    // dx = dt (v0 + dt (a0/2 + dt j0/6))
    const float d = __fmul_rn(dt, __fmaf_rn(dt, __fmaf_rn(dt, j6, a2), v0));
    const double xp = x0 + (double)d;
    ds_split(xp, xh, xl);
    if (!ds) xl = 0.0f;
    // v_p = v0 + dt (a0 + dt j0/2) = v0 + dt (2 (a0/2) + 3 dt (j0/6))
    vp = __fmaf_rn(dt, __fmaf_rn(__fmul_rn(3.0f, dt), j6, __fadd_rn(a2, a2)), v0);
}

// ---- a-2: predictor, one thread per j, one CTA per tile ------------------------------------
// Eq. 1-2 with dt = t_i - t_j (reading 3).  "the multiplications and
// divisions can be carried out in SP, but the summation should be carried out in DP"
// (PAPER.md:66): the Taylor increment is formed in FP32 (Horner), added to the fp64 x0 and the
// sum is re-split into a double-single pair (reading 11).  The kernel is HBM-bound
// (76 B read + 40 B written per particle); it also records the index range of every tile,
// which lets the force kernel skip per-pair self checks on tiles that cannot hold the i-particle.
__global__ void __launch_bounds__(JT)
k_predict(JStore S, int n_stored, double ti, int ds, float *__restrict__ pred,
          int *__restrict__ tile_imin, int *__restrict__ tile_imax)
{
    const int tile = blockIdx.x;
    const int l = threadIdx.x;
    const int j = tile * JT + l;
    float f[NF];
    int id_lo = INT32_MAX, id_hi = INT32_MIN;
    if (j < n_stored) {
        char *T = S.raw + (size_t)tile * RAW_TILE_BYTES;
        const float dt = (float)(ti - raw_t(T, l));
#pragma unroll
        for (int k = 0; k < 3; ++k)
            predict_coord(dt, raw_x(T, k, l), raw_v(T, k, l), raw_a2(T, k, l), raw_j6(T, k, l), ds, f[F_XH + k], f[F_XL + k], f[F_V + k]);
        f[F_M] = raw_m(T, l);
        id_lo = id_hi = raw_idx(T, l);
    } else {
#pragma unroll
        for (int k = 0; k < NF; ++k) f[k] = 0.0f;      // padding of the last tile: finite, massless
    }
    float *out = pred + (size_t)tile * TILE_FLOATS + l;
#pragma unroll
    for (int k = 0; k < NF; ++k) out[k * JT] = f[k];

    // index range of the tile
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        id_lo = min(id_lo, __shfl_xor_sync(0xffffffffu, id_lo, o));
        id_hi = max(id_hi, __shfl_xor_sync(0xffffffffu, id_hi, o));
    }
    __shared__ int s_lo[JT / 32], s_hi[JT / 32];
    if ((l & 31) == 0) { s_lo[l >> 5] = id_lo; s_hi[l >> 5] = id_hi; }
    __syncthreads();
    if (l == 0) {
#pragma unroll
        for (int w = 1; w < JT / 32; ++w) { id_lo = min(id_lo, s_lo[w]); id_hi = max(id_hi, s_hi[w]); }
        tile_imin[tile] = id_lo;
        tile_imax[tile] = id_hi;
    }
}

// ---- a-5: combine the S partial results of every i (fixed order => bit-reproducible) --------
// "reduce the partial forces directly in the GPU memory and only copy back the final result"
// (PAPER.md:106).  Sums in fp64 in split order; nearest neighbour: smallest r2, ties -> lowest
// split = lowest j address (reading 7); address -> caller's index.
__global__ void __launch_bounds__(256)
k_combine(Partials P, int S, int ni, const char *__restrict__ jraw,
          double *__restrict__ acc, double *__restrict__ jerk, double *__restrict__ pot,
          int *__restrict__ nn_index, double *__restrict__ nn_r2)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= ni) return;
    double a[3] = {0, 0, 0}, jk[3] = {0, 0, 0}, ph = 0;
    float best = __int_as_float(0x7f800000);
    int baddr = -1;
    for (int s = 0; s < S; ++s) {
        size_t o = (size_t)s * P.stride_s + (size_t)i * P.stride_i;
#pragma unroll
        for (int k = 0; k < 3; ++k) { a[k] += P.acc[k][o]; jk[k] += P.jrk[k][o]; }
        ph += P.pot[o];
        float r2 = P.nn_r2[o];
        int ad = P.nn_addr[o];
        if (ad >= 0 && r2 < best) { best = r2; baddr = ad; }
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) { acc[3 * (size_t)i + k] = a[k]; jerk[3 * (size_t)i + k] = jk[k]; }
    pot[i] = ph;
    if (nn_index) nn_index[i] = baddr >= 0 ? j_index(jraw, baddr) : -1;
    if (nn_r2) nn_r2[i] = baddr >= 0 ? (double)best : (double)__int_as_float(0x7f800000);
}

// many splits, few i (the small active blocks of block time steps): one warp per i.  Lane l sums
// the splits s = l, l+32, ... in order, then a fixed xor-tree adds the 32 lane sums: the order is
// fixed by (S) alone, so results are bit-reproducible.  Nearest neighbour: (r2, address)
// lexicographic minimum = smallest r2, ties -> smallest address.
__global__ void __launch_bounds__(128)
k_combine_wide(Partials P, int S, int ni, const char *__restrict__ jraw,
               double *__restrict__ acc, double *__restrict__ jerk, double *__restrict__ pot,
               int *__restrict__ nn_index, double *__restrict__ nn_r2)
{
    const int i = blockIdx.x * 4 + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (i >= ni) return;
    double v[7] = {0, 0, 0, 0, 0, 0, 0};
    float best = __int_as_float(0x7f800000);
    int baddr = 0x7fffffff;
    for (int s = lane; s < S; s += 32) {
        const size_t o = (size_t)s * P.stride_s + (size_t)i * P.stride_i;
#pragma unroll
        for (int k = 0; k < 3; ++k) { v[k] += P.acc[k][o]; v[3 + k] += P.jrk[k][o]; }
        v[6] += P.pot[o];
        const float r2 = P.nn_r2[o];
        const int ad = P.nn_addr[o];
        if (ad >= 0 && (r2 < best || (r2 == best && ad < baddr))) { best = r2; baddr = ad; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int k = 0; k < 7; ++k) v[k] += __shfl_xor_sync(0xffffffffu, v[k], o);
        const float r2 = __shfl_xor_sync(0xffffffffu, best, o);
        const int ad = __shfl_xor_sync(0xffffffffu, baddr, o);
        if (r2 < best || (r2 == best && ad < baddr)) { best = r2; baddr = ad; }
    }
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < 3; ++k) { acc[3 * (size_t)i + k] = v[k]; jerk[3 * (size_t)i + k] = v[3 + k]; }
        pot[i] = v[6];
        const bool has = baddr != 0x7fffffff;
        if (nn_index) nn_index[i] = has ? j_index(jraw, baddr) : -1;
        if (nn_r2) nn_r2[i] = has ? (double)best : (double)__int_as_float(0x7f800000);
    }
}

// very many splits (one per j-tile, small-block kernel at large N_j): one CTA of 128 threads per i.
// Thread t sums s = t, t+128, ... in order; fixed xor tree inside each warp; the four warp sums are
// added in warp order by thread 0.
__global__ void __launch_bounds__(128)
k_combine_block(Partials P, int S, int ni, const char *__restrict__ jraw,
                double *__restrict__ acc, double *__restrict__ jerk, double *__restrict__ pot,
                int *__restrict__ nn_index, double *__restrict__ nn_r2)
{
    const int i = blockIdx.x;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    __shared__ double sv[4][7];
    __shared__ float sr[4];
    __shared__ int sa[4];
    double v[7] = {0, 0, 0, 0, 0, 0, 0};
    float best = __int_as_float(0x7f800000);
    int baddr = 0x7fffffff;
    for (int s = tid; s < S; s += 128) {
        const size_t o = (size_t)s * P.stride_s + (size_t)i * P.stride_i;
#pragma unroll
        for (int k = 0; k < 3; ++k) { v[k] += P.acc[k][o]; v[3 + k] += P.jrk[k][o]; }
        v[6] += P.pot[o];
        const float r2 = P.nn_r2[o];
        const int ad = P.nn_addr[o];
        if (ad >= 0 && (r2 < best || (r2 == best && ad < baddr))) { best = r2; baddr = ad; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int k = 0; k < 7; ++k) v[k] += __shfl_xor_sync(0xffffffffu, v[k], o);
        const float r2 = __shfl_xor_sync(0xffffffffu, best, o);
        const int ad = __shfl_xor_sync(0xffffffffu, baddr, o);
        if (r2 < best || (r2 == best && ad < baddr)) { best = r2; baddr = ad; }
    }
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < 7; ++k) sv[w][k] = v[k];
        sr[w] = best;
        sa[w] = baddr;
    }
    __syncthreads();
    if (tid == 0) {
#pragma unroll
        for (int q = 1; q < 4; ++q) {
#pragma unroll
            for (int k = 0; k < 7; ++k) v[k] += sv[q][k];
            if (sr[q] < best || (sr[q] == best && sa[q] < baddr)) { best = sr[q]; baddr = sa[q]; }
        }
#pragma unroll
        for (int k = 0; k < 3; ++k) { acc[3 * (size_t)i + k] = v[k]; jerk[3 * (size_t)i + k] = v[3 + k]; }
        pot[i] = v[6];
        const bool has = baddr != 0x7fffffff;
        if (nn_index) nn_index[i] = has ? j_index(jraw, baddr) : -1;
        if (nn_r2) nn_r2[i] = has ? (double)best : (double)__int_as_float(0x7f800000);
    }
}

// ---- a-5 for neighbour lists: concatenate the per-split lists of every i ------
// Split s covers an increasing address range and appends in address order, so the concatenation in
// split order is the list in increasing j address; the first `maxlen` entries are kept, the count
// is the total (count > maxlen = overflow, reading 20).  Addresses -> caller's indices.
// One warp per i.
__global__ void __launch_bounds__(128)
k_combine_nb(const int *__restrict__ part_cnt, const int *__restrict__ part_list, int S, int ni, int maxlen,
             const char *__restrict__ jraw, int *__restrict__ cnt, int *__restrict__ list)
{
    const int i = blockIdx.x * 4 + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (i >= ni) return;
    int total = 0;
    for (int s = 0; s < S; ++s) {
        const int c = part_cnt[(size_t)s * ni + i];
        const int stored = min(c, maxlen);
        const int *src = part_list + ((size_t)s * ni + i) * maxlen;
        for (int k = lane; k < stored; k += 32) {
            const int pos = total + k;
            if (pos < maxlen) list[(size_t)i * maxlen + pos] = j_index(jraw, src[k]);
        }
        total += c;
    }
    if (lane == 0) cnt[i] = total;
}

// ---- multi-GPU j-split (section 2.4): the exchange step's device-side halves ----------
// Every GPU holds N_j / Q of the j-particles (increasing address ranges by rank) and computes partial
// forces on the SAME i-block; the partial (a, adot, phi) are summed and the nearest neighbour is the
// minimum over the GPUs.  The paper sums on the host; here the two reductions are collectives on
// device buffers (NCCL allreduce): MIN on a 64-bit key, then SUM on [8][ni] fp64.
//   key = (bits of the binary32 r2) << 32 | rank      (non-negative floats order like integers; ties ->
//         lowest rank = lowest address range, reading 7);  no neighbour -> INT64_MAX
__global__ void __launch_bounds__(256)
k_jsplit_pack(int ni, int rank, const double *__restrict__ nn_r2, const int *__restrict__ nn_index, long long *__restrict__ key)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= ni) return;
    const long long none = 0x7fffffffffffffffLL;
    const float r2 = (float)nn_r2[i];               // exact: the kernels produce r2 in binary32
    key[i] = nn_index[i] < 0 ? none : (((long long)__float_as_uint(r2) << 32) | (long long)(unsigned)rank);
}

// after the MIN: the winning rank contributes its neighbour's index (as fp64, exact) to the SUM buffer
__global__ void __launch_bounds__(256)
k_jsplit_select(int ni, int rank, const long long *__restrict__ key_min, const int *__restrict__ nn_index, double *__restrict__ index_f64)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= ni) return;
    const long long k = key_min[i];
    const bool mine = k != 0x7fffffffffffffffLL && (int)(k & 0xffffffffLL) == rank;
    index_f64[i] = mine ? (double)nn_index[i] : 0.0;
}

// after the SUM: final nearest neighbour of every i
__global__ void __launch_bounds__(256)
k_jsplit_unpack(int ni, const long long *__restrict__ key_min, const double *__restrict__ index_sum, int *__restrict__ nn_index,
                double *__restrict__ nn_r2)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= ni) return;
    const long long k = key_min[i];
    const bool has = k != 0x7fffffffffffffffLL;
    if (nn_index) nn_index[i] = has ? (int)index_sum[i] : -1;
    if (nn_r2) nn_r2[i] = has ? (double)__uint_as_float((unsigned)(k >> 32)) : (double)__int_as_float(0x7f800000);
}

// ---- debug: the kernel's Eq.-3 separation for chosen (i, j) pairs (DESIGN.md pin P11) -------
__global__ void k_debug_dx(int n, const int *__restrict__ ipipe, const int *__restrict__ jaddr,
                           const double *__restrict__ xi, int ds, const float *__restrict__ pred,
                           float *__restrict__ out)
{
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    int i = ipipe[p], j = jaddr[p];
    const float *t = pred + (size_t)(j / JT) * TILE_FLOATS + (j % JT);
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        float hi, lo;
        ds_split(xi[3 * (size_t)i + k], hi, lo);
        if (!ds) lo = 0.0f;
        out[3 * (size_t)p + k] = ds_dx(t[(F_XH + k) * JT], t[(F_XL + k) * JT], hi, lo);
    }
}

}  // namespace g6
