// g6_debug_dx.cu -- parity-test hook, built as its own small library (libg6b200_dbg.so); NOT part of libg6b200.
//
// Pin P11: the kernels' Eq.-3 separation dx = (xj_hi - xi_hi) + (xj_lo - xi_lo)
// must equal a binary32 CPU transcription bit for bit.  This file instantiates the PRODUCTION
// kernels -- k_predict, k_force_fast (g6_force_fast.cuh) and the block-step kernel (g6_block_step.cuh), same
// headers, same pair code -- with their DBG template flag, which makes pair2 / pair2_checked hand the packed-lane
// separations of every (i, j) pair to the caller, and runs them on the caller's particles.  Nothing here computes:
// it allocates, launches and copies.
#include <cuda_runtime.h>

#include <algorithm>
#include <vector>

#include "../g6_block_step.cuh"

using namespace g6;

namespace {
struct Dev {
    std::vector<void *> p;
    ~Dev() { for (void *q : p) cudaFree(q); }
    template <class T> T *alloc(size_t n)
    {
        void *q = nullptr;
        if (cudaMalloc(&q, std::max<size_t>(n, 1) * sizeof(T)) != cudaSuccess) return nullptr;
        p.push_back(q);
        return (T *)q;
    }
    template <class T> T *upload(const T *h, size_t n)
    {
        T *d = alloc<T>(n);
        if (d && cudaMemcpy(d, h, n * sizeof(T), cudaMemcpyHostToDevice) != cudaSuccess) return nullptr;
        return d;
    }
};
}  // namespace

extern "C" {

// kernel: 2 = sweep kernel k_force_fast<128, 2, Newton> (its unchecked tiles, and its checked tiles wherever a warp holds an
//             i-particle whose index lies in a tile's index range, and the ragged last tile),
//         3 = block-step kernel (ni <= 64; every pair takes pair2_checked).
// xj[nj][3], index_j[nj]: the j-particles at t = 0 (v = a = jerk = 0, so the predictor is the double-single split);
// xi[ni][3], index_i[ni]: the i-particles; ds: 1 double-single, 0 lo words dropped.
// dx[ni][nj][3] (host, binary32) receives every pair's separation.  Returns 0, or a cudaError_t value, or -1 (bad arguments).
int g6dbg_pair_dx(int kernel, int nj, int ni, const double *xj, const int *index_j, const double *xi, const int *index_i,
                  double eps2, int ds, float *dx)
{
    if ((kernel != 2 && kernel != 3) || nj < 1 || ni < 1 || (kernel == 3 && ni > BS_MAX_I) || !xj || !index_j || !xi || !index_i || !dx) return -1;
    Dev D;
    const int ntiles = (nj + JT - 1) / JT;
    std::vector<double> zero3(3 * (size_t)std::max(nj, ni), 0.0), ones(nj, 1.0 / nj);
    char *raw = D.alloc<char>((size_t)ntiles * RAW_TILE_BYTES);
    float *pred = D.alloc<float>((size_t)ntiles * TILE_FLOATS);
    int *imin = D.alloc<int>(ntiles), *imax = D.alloc<int>(ntiles);
    const double *d_xj = D.upload(xj, 3 * (size_t)nj), *d_z = D.upload(zero3.data(), zero3.size()), *d_m = D.upload(ones.data(), nj);
    const int *d_ij = D.upload(index_j, nj), *d_ii = D.upload(index_i, ni);
    const double *d_xi = D.upload(xi, 3 * (size_t)ni);
    float *d_dx = D.alloc<float>(3 * (size_t)ni * nj);
    const int G = std::max(1, std::min(ntiles, 148));
    const size_t pe = (size_t)std::max(G, 1) * ni + 64;
    double *part = D.alloc<double>(8 * pe);
    double *out = D.alloc<double>(9 * (size_t)ni);
    unsigned int *counter = D.alloc<unsigned int>(1);
    if (!raw || !pred || !imin || !imax || !d_xj || !d_z || !d_m || !d_ij || !d_ii || !d_xi || !d_dx || !part || !out || !counter) return (int)cudaErrorMemoryAllocation;
    cudaMemset(raw, 0, (size_t)ntiles * RAW_TILE_BYTES);
    cudaMemset(counter, 0, sizeof(unsigned int));
    cudaMemset(d_dx, 0xff, 3 * (size_t)ni * nj * sizeof(float));         // NaN pattern: a pair nobody stored shows up
    JStore S{raw};
    k_store_from_f64<<<(nj + 255) / 256, 256>>>(S, 0, nj, d_ij, d_z, d_m, d_z, d_z, d_z, d_xj);
    Partials P{};
    for (int k = 0; k < 3; ++k) { P.acc[k] = part + (size_t)k * pe; P.jrk[k] = part + (size_t)(3 + k) * pe; }
    P.pot = part + 6 * pe;
    P.nn_r2 = (float *)(part + 7 * pe);
    P.nn_addr = (int *)(P.nn_r2 + pe);
    if (kernel == 2) {
        k_predict<<<ntiles, JT>>>(S, nj, 0.0, ds, pred, imin, imax);
        ForceArgs A{};
        A.pred = pred; A.jraw = raw; A.tile_imin = imin; A.tile_imax = imax;
        A.nj = nj; A.ntiles = ntiles; A.i_index = d_ii; A.xi = d_xi; A.vi = d_z; A.ni = ni;
        A.eps2 = (float)eps2; A.ds = ds; A.S = 1; A.P = P; A.P.stride_s = ni; A.P.stride_i = 1;
        A.dbg_dx = d_dx;
        const size_t bytes = sizeof(FastSmem<128, 2>);
        cudaFuncSetAttribute(k_force_fast<128, 2, true, false, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        k_force_fast<128, 2, true, false, true, true><<<dim3((ni + 255) / 256, 1), 128, bytes>>>(A);
    } else {
        BsArgs B{};
        B.raw = raw; B.ti = 0.0; B.nj = nj; B.ntiles = ntiles; B.ni = ni; B.n_upd = 0; B.eps2 = (float)eps2; B.ds = ds;
        B.inline_i = 0; B.i_index = d_ii; B.xi = d_xi; B.vi = d_z;
        B.P = P; B.P.stride_s = 1; B.P.stride_i = G;
        B.counter = counter;
        B.acc = out; B.jerk = out + 3 * (size_t)ni; B.pot = out + 6 * (size_t)ni; B.nn_index = nullptr; B.nn_r2 = nullptr;
        B.dbg_dx = d_dx;
        const size_t bytes = sizeof(BsSmem<BS_MAX_I>);
        cudaFuncSetAttribute(k_block_step_dbg<BS_MAX_I, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        k_block_step_dbg<BS_MAX_I, true><<<G, BS_THREADS, bytes>>>(B);
    }
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpy(dx, d_dx, 3 * (size_t)ni * nj * sizeof(float), cudaMemcpyDeviceToHost);
    return (int)e;
}

}  // extern "C"
