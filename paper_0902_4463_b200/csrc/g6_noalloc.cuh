// g6_noalloc.cuh -- g6x_calc_dev_noalloc: the sweep path (a-2 predictor, a-4 force kernel, a-5 combine) for callers
// that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// The regular path keeps the force kernel's per-split partial sums (a-4 -> a-5, "partial forces ... are
// reduced") in a buffer that ensure_partials() grows with cudaMalloc when a block needs more rows than any before it.
// Here the same kernels write their partials into a FILE-SCOPE device array of fixed size: nothing is allocated or
// freed by the call, at the price of a stated maximum and of 4 MiB of device memory held by every GPU that loads the
// library until the process exits.
//
// Included at the end of g6_api.cu (one translation unit: the array, the cudaGetSymbolAddress that resolves it and
// the launches that use it must live in the same .cu file).
#pragma once

namespace {

// rows = (j-splits S) x (i-particles n_i) of one call; one row = 7 fp64 sums + nearest-neighbour r2 (f32) + address (i32)
constexpr int NA_MAX_ROWS = 65536;
constexpr int NA_ROW_BYTES = 7 * (int)sizeof(double) + (int)sizeof(float) + (int)sizeof(int);
constexpr int NA_MAX_DEVICES = 64;

// In host code this name is a host-side stand-in, NOT a device address: only cudaGetSymbolAddress gives the pointer
// a kernel may use (na_scratch_ptr below).  Shared by every call on the device; holds the last call's partials.
static __device__ __align__(256) unsigned char g_na_scratch[(size_t)NA_MAX_ROWS * NA_ROW_BYTES];

unsigned char *g_na_ptr[NA_MAX_DEVICES] = {};      // per device: the array's device address, resolved once

// set-up, once per device, with that device current (g6_open made the cluster's device current on this thread)
int na_scratch_ptr(Cluster &c, unsigned char **out)
{
    if (c.device < 0 || c.device >= NA_MAX_DEVICES) return fail(c, G6_ERR_ARG, "device %d: the no-alloc scratch serves devices 0..%d", c.device, NA_MAX_DEVICES - 1);
    if (!g_na_ptr[c.device]) {
        int cur = -1;
        CK(cudaGetDevice(&cur));
        if (cur != c.device) CK(cudaSetDevice(c.device));
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_na_scratch);
        if (cur != c.device) cudaSetDevice(cur);
        if (e != cudaSuccess || !p) return fail(c, G6_ERR_CUDA, "cudaGetSymbolAddress(no-alloc scratch): %s", cudaGetErrorString(e));
        g_na_ptr[c.device] = static_cast<unsigned char *>(p);
    }
    *out = g_na_ptr[c.device];
    return G6_OK;
}

}  // namespace

extern "C" {

int g6x_noalloc_max_rows(void) { return NA_MAX_ROWS; }

int g6x_noalloc_init(int clusterid)
{
    GET_CLUSTER(clusterid);
    unsigned char *p;
    return na_scratch_ptr(c, &p);
}

int g6x_calc_dev_noalloc(int clusterid, int nj, int ni, const int *d_index, const double *d_xi, const double *d_vi,
                         double eps2, double *d_acc, double *d_jerk, double *d_pot, int *d_nn_index, double *d_nn_r2)
{
    GET_CLUSTER(clusterid);
    if (c.pending) return fail(c, G6_ERR_SEQUENCE, "g6x_calc_dev_noalloc between firsthalf and lasthalf");
    if (c.n_rec > 0) return fail(c, G6_ERR_SEQUENCE, "g6x_calc_dev_noalloc: %d j-particle updates are pending (g6_flush_jp_buffer first; this call stages nothing)", c.n_rec);
    int rc = check_force_args(c, nj, ni);
    if (rc) return rc;
    if (ni > NA_MAX_ROWS) return fail(c, G6_ERR_NI, "g6x_calc_dev_noalloc: ni = %d above the fixed scratch (%d rows); use g6x_calc_dev", ni, NA_MAX_ROWS);
    if (!d_index || !d_xi || !d_vi || !d_acc || !d_jerk || !d_pot) return fail(c, G6_ERR_ARG, "NULL device array");
    if (!(eps2 >= 0.0)) return fail(c, G6_ERR_ARG, "eps2 = %g", eps2);
    unsigned char *scratch;
    rc = na_scratch_ptr(c, &scratch);
    if (rc) return rc;

    ForceArgs A{};
    A.pred = c.pred;
    A.jraw = c.js.raw;
    A.tile_imin = c.tile_imin;
    A.tile_imax = c.tile_imax;
    A.nj = nj;
    A.ntiles = (nj + JT - 1) / JT;
    A.i_index = d_index;
    A.xi = d_xi;
    A.vi = d_vi;
    A.ni = ni;
    A.eps2 = (float)eps2;
    A.ds = c.opt_ds;

    rc = run_predict(c);                                  // a-2 into the cluster's predicted tiles (allocated with the j-store)
    if (rc) return rc;

    // kernel shape and j-splits as run_force picks them, the splits capped by the rows the scratch holds
    const bool fast_ok = A.eps2 >= 4.0f * std::numeric_limits<float>::min() && std::isfinite(A.eps2);
    const bool use_fast = (c.opt_kernel == 2 || c.opt_kernel == 0) && fast_ok;
    const FastVariant fv = fast_pick(ni, c.n_sm, c.opt_variant);
    const int itile = use_fast ? fv.threads * fv.it : REF_THREADS;
    const int n_itiles = (ni + itile - 1) / itile;
    const int slots = c.n_sm * (use_fast ? fast_ctas_per_sm(fv) : 8);
    const long long s_cap = NA_MAX_ROWS / ni;             // >= 1
    int S = c.opt_jsplit > 0 ? (int)std::min<long long>(c.opt_jsplit, s_cap) : choose_jsplit(n_itiles, A.ntiles, slots, ni, s_cap);
    S = std::max(1, std::min(S, A.ntiles));
    if ((long long)S * ni > NA_MAX_ROWS) return fail(c, G6_ERR_NI, "g6x_calc_dev_noalloc: %d splits x %d i-particles above %d rows", S, ni, NA_MAX_ROWS);
    A.S = S;

    // the partials of this call, carved out of the fixed array (every row the combine reads is written by the force
    // kernel first: nothing has to start at zero)
    const size_t rows = ((size_t)S * ni + 63) & ~(size_t)63;
    double *d = reinterpret_cast<double *>(scratch);
    for (int k = 0; k < 3; ++k) A.P.acc[k] = d + (size_t)k * rows;
    for (int k = 0; k < 3; ++k) A.P.jrk[k] = d + (size_t)(3 + k) * rows;
    A.P.pot = d + 6 * rows;
    A.P.nn_r2 = reinterpret_cast<float *>(d + 7 * rows);
    A.P.nn_addr = reinterpret_cast<int *>(A.P.nn_r2 + rows);
    const bool wide = S > 8;
    A.P.stride_s = wide ? 1 : ni;
    A.P.stride_i = wide ? S : 1;

    if (use_fast) {
        rc = launch_force_fast(A, c.opt_newton != 0, fv, n_itiles, S, c.stream);
        if (rc) return fail(c, G6_ERR_CUDA, "fast force kernel launch failed: %s", cudaGetErrorString((cudaError_t)rc));
    } else {
        dim3 grid(n_itiles, S);
        if (c.opt_newton) k_force_ref<true><<<grid, REF_THREADS, 0, c.stream>>>(A);
        else k_force_ref<false><<<grid, REF_THREADS, 0, c.stream>>>(A);
        CK(cudaGetLastError());
    }
    if (wide) k_combine_wide<<<(ni + 3) / 4, 128, 0, c.stream>>>(A.P, S, ni, c.js.raw, d_acc, d_jerk, d_pot, d_nn_index, d_nn_r2);
    else k_combine<<<(ni + 255) / 256, 256, 0, c.stream>>>(A.P, S, ni, c.js.raw, d_acc, d_jerk, d_pot, d_nn_index, d_nn_r2);
    CK(cudaGetLastError());
    c.last_ctas = n_itiles * S;
    c.last_S = S;
    c.last_kernel = use_fast ? 2 : 1;
    c.ev_valid = false;
    return G6_OK;
}

}  // extern "C"
