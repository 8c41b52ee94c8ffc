// g6_api.cu -- the C ABI of libg6b200 (include/g6.h): host state, staging, launch scheduling.
// Every step of the path runs in the CUDA kernels; there is no CPU fallback: without a CUDA
// device g6_open fails with G6_ERR_CUDA.
#include "../../include/g6.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <new>
#include <thread>
#include <vector>

#include "g6_device.cuh"
#include "g6_force_ref.cuh"
#include "g6_force_fast.cuh"
#include "g6_block_step.cuh"

using namespace g6;

namespace {

constexpr int MAX_CLUSTERS = 4;
constexpr int MAX_NPIPES = 1 << 21;
constexpr int N_EVENTS = 6;

int g_npipes = 0;   // 0 = not initialised yet (env G6_NPIPES or G6_DEFAULT_NPIPES)

struct Cluster {
    bool open = false;
    int device = 0;
    int n_sm = 148;
    cudaStream_t stream = nullptr;
    cudaStream_t own_stream = nullptr;
    char err[512] = "no error";

    // j store
    int capacity = 0;        // largest number of addresses this cluster may hold (env G6_NJMAX)
    int alloc_cap = 0;       // addresses the device arrays hold now (grown on demand up to `capacity`)
    int n_stored = 0;        // highest address set + 1
    JStore js{};
    unsigned int *d_counter = nullptr;   // arrival ticket of the block-step kernel
    float *pred = nullptr;   // predicted tiles
    int *tile_imin = nullptr, *tile_imax = nullptr;
    bool pred_valid = false;
    double pred_ti = 0.0;
    int pred_ds = 1;
    int pred_n = 0;

    // host -> device staging of changed j particles: two pinned+mapped buffers used alternately,
    // so the host can fill one while the device may still read the other
    JRecord *h_rec[2] = {nullptr, nullptr};   // pinned, mapped
    JRecord *hd_rec[2] = {nullptr, nullptr};  // device view of the same memory (zero-copy path)
    JRecord *d_rec = nullptr;                 // device copy (DMA path)
    cudaEvent_t ev_rec[2] = {nullptr, nullptr};
    bool rec_used[2] = {false, false};
    int rec_cur = 0;
    int rec_cap = 0, n_rec = 0;
    std::vector<int> slot_of_addr;   // address -> slot in h_rec[rec_cur] (or -1)

    // i block and results: one pinned+mapped block each, compact layout by ni
    //   i block : xi[3 ni] f64 | vi[3 ni] f64 | index[ni] i32
    //   results : acc[3 ni] f64 | jerk[3 ni] f64 | pot[ni] f64 | nn_r2[ni] f64 | nn_index[ni] i32
    int i_cap = 0;
    char *h_iblk = nullptr, *hd_iblk = nullptr, *d_iblk = nullptr;
    char *h_res = nullptr, *hd_res = nullptr, *d_res = nullptr;
    unsigned int *h_done = nullptr, *hd_done = nullptr;   // mapped word: the block-step kernel's "results are on the host" flag
    unsigned int done_seq = 0, pend_done_seq = 0;          // pend_done_seq != 0: lasthalf spins on h_done instead of an event
    bool res_on_host = false;   // last call's results were written straight into h_res
    bool iblk_on_device = false;   // last host call left a copy of the i-block in d_iblk

    // partial results
    Partials part{};
    void *part_block = nullptr;
    size_t part_elems = 0;

    // neighbour lists: per-split lists, combined lists, host copies; all on demand
    int *d_nb_pcnt = nullptr, *d_nb_plist = nullptr;   // [S][ni], [S][ni][maxlen]
    size_t nb_part_rows = 0;                           // S * ni rows allocated
    int *d_nb_wcnt = nullptr, *d_nb_wlist = nullptr;   // block-step kernel: per-warp lists [ni][warps], [warps][ni][maxlen]
    size_t nb_w_rows = 0;                              // warps * ni rows allocated
    int *d_nb_cnt = nullptr, *d_nb_list = nullptr;     // [ni], [ni][maxlen]
    int *h_nb_cnt = nullptr, *h_nb_list = nullptr;     // pinned
    double *h_h2 = nullptr, *d_h2 = nullptr;           // neighbour radii of the i-block
    int nb_cap = 0;                                    // ni the combined / host / h2 buffers hold
    int nb_alloc_maxlen = 0;                           // maxlen the buffers were sized for
    bool last_nb = false;                              // the last host force call built lists
    bool nb_on_host = false;                           // ... and they have been copied to h_nb_*
    int last_nb_maxlen = 0;

    // bulk-load staging (host fp64 arrays -> device)
    void *h_bulk = nullptr, *d_bulk = nullptr;
    size_t bulk_bytes = 0;

    // call state
    double ti = 0.0;
    bool pending = false;      // firsthalf issued, lasthalf not yet
    bool have_result = false;  // a host force call completed (neighbour / debug queries)
    int pend_nj = 0, pend_ni = 0;
    bool pend_nb = false;
    int last_ni = 0;
    cudaEvent_t ev[N_EVENTS] = {};
    bool ev_valid = false;
    int last_ctas = 0, last_S = 0;
    int last_kernel = 0;       // force kernel of the last call: 1 checked reference, 2 fast sweep kernel, 3 block-step kernel

    // options
    int opt_ds = 1, opt_newton = 1, opt_jsplit = 0, opt_kernel = 0, opt_timers = 0, opt_variant = 0, opt_small = 32, opt_nb_maxlen = 256, opt_bs_design = 0;
    bool small_explicit = false;   // option "small" was set by the caller (else the N_j-dependent rule of small_limit)
};

Cluster g_cl[MAX_CLUSTERS];

int fail(Cluster &c, int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(c.err, sizeof(c.err), fmt, ap);
    va_end(ap);
    return code;
}

#define CK(call)                                                                                  \
    do {                                                                                          \
        cudaError_t e_ = (call);                                                                  \
        if (e_ != cudaSuccess)                                                                    \
            return fail(c, G6_ERR_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_),  \
                        __FILE__, __LINE__);                                                      \
    } while (0)

#define GET_CLUSTER(id)                                                     \
    if ((id) < 0 || (id) >= MAX_CLUSTERS) return G6_ERR_CLUSTER;            \
    Cluster &c = g_cl[(id)];                                                \
    if (!c.open) return fail(c, G6_ERR_NOT_OPEN, "cluster %d is not open", (id))

int env_int(const char *name, int dflt)
{
    const char *v = getenv(name);
    if (!v || !*v) return dflt;
    char *end = nullptr;
    long x = strtol(v, &end, 0);
    return (end && *end == 0) ? (int)x : dflt;
}

void init_npipes()
{
    if (g_npipes == 0) g_npipes = std::min(std::max(env_int("G6_NPIPES", G6_DEFAULT_NPIPES), 1), MAX_NPIPES);
}

template <class T>
cudaError_t dalloc(T *&p, size_t n) { return cudaMalloc((void **)&p, n * sizeof(T)); }
template <class T>
cudaError_t halloc(T *&p, size_t n) { return cudaMallocHost((void **)&p, n * sizeof(T)); }
template <class T>
void dfree(T *&p) { if (p) cudaFree(p); p = nullptr; }
template <class T>
void hfree(T *&p) { if (p) cudaFreeHost(p); p = nullptr; }

inline size_t iblk_bytes(size_t ni) { return ni * (6 * sizeof(double) + sizeof(int)); }
inline size_t res_bytes(size_t ni) { return ni * (8 * sizeof(double) + sizeof(int)); }

// views into an i block / result block laid out for `ni` particles
struct IView { const double *xi, *vi; const int *idx; };
struct RView { double *acc, *jerk, *pot, *nnr2; int *nnidx; };
inline IView iview(char *base, size_t ni)
{
    const double *d = (const double *)base;
    return IView{d, d + 3 * ni, (const int *)(d + 6 * ni)};
}
inline RView rview(char *base, size_t ni)
{
    double *d = (double *)base;
    return RView{d, d + 3 * ni, d + 6 * ni, d + 7 * ni, (int *)(d + 8 * ni)};
}

template <class T>
cudaError_t mapped_alloc(T *&h, T *&hd, size_t bytes)
{
    cudaError_t e = cudaHostAlloc((void **)&h, bytes, cudaHostAllocMapped);
    if (e != cudaSuccess) return e;
    return cudaHostGetDevicePointer((void **)&hd, (void *)h, 0);
}

void free_i(Cluster &c)
{
    hfree(c.h_iblk); hfree(c.h_res); hfree(c.h_done);
    c.hd_done = nullptr;
    dfree(c.d_iblk); dfree(c.d_res);
    c.hd_iblk = c.hd_res = nullptr;
    c.i_cap = 0;
}

// Host copies between the caller's arrays and the pinned staging buffers.  One thread moves ~10 GB/s; a full sweep's 250 MB of
// j-particles, i-particles and results then cost 25 ms of a 1.3 s step (the end-to-end figure of bench.py).  Large copies are
// split over a few threads (contiguous pieces: the result is the same bytes).
void big_memcpy(void *dst, const void *src, size_t bytes)
{
    constexpr size_t MIN_PER_THREAD = 4u << 20;
    const unsigned hw = std::thread::hardware_concurrency();
    const size_t nt = std::min<size_t>(std::min<size_t>(hw ? hw : 1, 12), bytes / MIN_PER_THREAD);
    if (nt < 2) { memcpy(dst, src, bytes); return; }
    std::vector<std::thread> th;
    const size_t per = ((bytes / nt) + 4095) & ~(size_t)4095;
    try {
        for (size_t t = 1; t < nt; ++t) {
            const size_t o = t * per, len = o >= bytes ? 0 : std::min(per, bytes - o);
            if (len) th.emplace_back([=] { memcpy((char *)dst + o, (const char *)src + o, len); });
        }
    } catch (...) {                                   // no thread to be had: copy what is left here
        for (auto &w : th) w.join();
        memcpy(dst, src, bytes);
        return;
    }
    memcpy(dst, src, std::min(per, bytes));
    for (auto &w : th) w.join();
}

int ensure_i(Cluster &c, int ni)
{
    if (ni <= c.i_cap) return G6_OK;
    CK(cudaStreamSynchronize(c.stream));
    free_i(c);
    // grown geometrically: the block sizes of a Hermite run creep upwards, and every reallocation is a stream synchronisation plus
    // cudaFree / cudaMalloc / cudaHostAlloc calls (measured: 1 ms to hundreds of ms each on the B200 box)
    size_t n = std::max<size_t>(std::max(ni, 4096), (size_t)c.i_cap + c.i_cap / 2);
    CK(mapped_alloc(c.h_iblk, c.hd_iblk, iblk_bytes(n)));
    CK(mapped_alloc(c.h_res, c.hd_res, res_bytes(n)));
    CK(mapped_alloc(c.h_done, c.hd_done, sizeof(unsigned int)));
    *c.h_done = 0;
    c.done_seq = c.pend_done_seq = 0;
    CK(cudaMalloc((void **)&c.d_iblk, iblk_bytes(n)));
    CK(cudaMalloc((void **)&c.d_res, res_bytes(n)));
    c.i_cap = (int)n;
    c.have_result = false;
    return G6_OK;
}

int ensure_partials(Cluster &c, size_t elems)
{
    if (elems <= c.part_elems) return G6_OK;
    const size_t prev = c.part_elems;
    CK(cudaStreamSynchronize(c.stream));
    if (c.part_block) cudaFree(c.part_block);
    c.part_block = nullptr;
    c.part_elems = 0;
    elems = std::max(elems, prev + prev / 2);          // geometric growth (see ensure_i)
    elems = (elems + 63) & ~(size_t)63;
    CK(cudaMalloc(&c.part_block, elems * (7 * sizeof(double) + sizeof(float) + sizeof(int))));
    double *d = (double *)c.part_block;
    for (int k = 0; k < 3; ++k) c.part.acc[k] = d + (size_t)k * elems;
    for (int k = 0; k < 3; ++k) c.part.jrk[k] = d + (size_t)(3 + k) * elems;
    c.part.pot = d + 6 * elems;
    c.part.nn_r2 = (float *)(d + 7 * elems);
    c.part.nn_addr = (int *)(c.part.nn_r2 + elems);
    c.part_elems = elems;
    return G6_OK;
}

void free_nb(Cluster &c)
{
    dfree(c.d_nb_pcnt); dfree(c.d_nb_plist); dfree(c.d_nb_cnt); dfree(c.d_nb_list); dfree(c.d_h2);
    dfree(c.d_nb_wcnt); dfree(c.d_nb_wlist);
    hfree(c.h_nb_cnt); hfree(c.h_nb_list); hfree(c.h_h2);
    c.nb_part_rows = 0;
    c.nb_w_rows = 0;
    c.nb_cap = 0;
    c.nb_alloc_maxlen = 0;
    c.last_nb = c.nb_on_host = false;
}

// maxlen changed since the buffers were sized: drop them all
int nb_check_maxlen(Cluster &c)
{
    if (c.opt_nb_maxlen != c.nb_alloc_maxlen) {
        CK(cudaStreamSynchronize(c.stream));
        free_nb(c);
        c.nb_alloc_maxlen = c.opt_nb_maxlen;
    }
    return G6_OK;
}

// per-split lists of a force call with neighbour lists (rows = S * ni)
int ensure_nb_part(Cluster &c, size_t rows)
{
    int rc = nb_check_maxlen(c);
    if (rc) return rc;
    if (rows <= c.nb_part_rows) return G6_OK;
    rows = std::max(rows, c.nb_part_rows + c.nb_part_rows / 2);
    CK(cudaStreamSynchronize(c.stream));
    dfree(c.d_nb_pcnt); dfree(c.d_nb_plist);
    c.nb_part_rows = 0;
    CK(dalloc(c.d_nb_pcnt, rows)); CK(dalloc(c.d_nb_plist, rows * c.opt_nb_maxlen));
    c.nb_part_rows = rows;
    return G6_OK;
}

// per-warp lists of the block-step kernel (rows = warps of the grid * ni)
int ensure_nb_warp(Cluster &c, size_t rows)
{
    int rc = nb_check_maxlen(c);
    if (rc) return rc;
    if (rows <= c.nb_w_rows) return G6_OK;
    rows = std::max(rows, c.nb_w_rows + c.nb_w_rows / 2);
    CK(cudaStreamSynchronize(c.stream));
    dfree(c.d_nb_wcnt); dfree(c.d_nb_wlist);
    c.nb_w_rows = 0;
    CK(dalloc(c.d_nb_wcnt, rows)); CK(dalloc(c.d_nb_wlist, rows * c.opt_nb_maxlen));
    c.nb_w_rows = rows;
    return G6_OK;
}

// combined lists, radii and their pinned host copies for a HOST force call on ni particles
int ensure_nb_host(Cluster &c, int ni)
{
    int rc = nb_check_maxlen(c);
    if (rc) return rc;
    if (ni <= c.nb_cap) return G6_OK;
    const int prev_cap = c.nb_cap;
    CK(cudaStreamSynchronize(c.stream));
    dfree(c.d_nb_cnt); dfree(c.d_nb_list); dfree(c.d_h2);
    hfree(c.h_nb_cnt); hfree(c.h_nb_list); hfree(c.h_h2);
    c.nb_cap = 0;
    c.last_nb = c.nb_on_host = false;
    const size_t n = std::max<size_t>(std::max(ni, 1024), (size_t)prev_cap + prev_cap / 2), ml = c.opt_nb_maxlen;
    CK(dalloc(c.d_nb_cnt, n)); CK(dalloc(c.d_nb_list, n * ml)); CK(dalloc(c.d_h2, n));
    CK(halloc(c.h_nb_cnt, n)); CK(halloc(c.h_nb_list, n * ml)); CK(halloc(c.h_h2, n));
    c.nb_cap = (int)n;
    return G6_OK;
}

int ensure_bulk(Cluster &c, size_t bytes)
{
    if (bytes <= c.bulk_bytes) return G6_OK;
    bytes = std::max(bytes, c.bulk_bytes + c.bulk_bytes / 2);
    CK(cudaStreamSynchronize(c.stream));
    if (c.h_bulk) cudaFreeHost(c.h_bulk);
    if (c.d_bulk) cudaFree(c.d_bulk);
    c.h_bulk = c.d_bulk = nullptr;
    c.bulk_bytes = 0;
    CK(cudaMallocHost(&c.h_bulk, bytes));
    CK(cudaMalloc(&c.d_bulk, bytes));
    c.bulk_bytes = bytes;
    return G6_OK;
}

int ensure_rec(Cluster &c, int n)
{
    if (n <= c.rec_cap) return G6_OK;
    const int cap = std::max(std::max(n, 2 * c.rec_cap), 4096);
    CK(cudaStreamSynchronize(c.stream));   // nothing may still read the old buffers
    JRecord *h[2] = {nullptr, nullptr}, *hd[2] = {nullptr, nullptr}, *d = nullptr;
    for (int b = 0; b < 2; ++b) CK(mapped_alloc(h[b], hd[b], sizeof(JRecord) * cap));
    CK(dalloc(d, cap));
    if (c.n_rec) memcpy(h[c.rec_cur], c.h_rec[c.rec_cur], sizeof(JRecord) * c.n_rec);
    for (int b = 0; b < 2; ++b) { hfree(c.h_rec[b]); c.h_rec[b] = h[b]; c.hd_rec[b] = hd[b]; c.rec_used[b] = false; }
    dfree(c.d_rec);
    c.d_rec = d;
    c.rec_cap = cap;
    return G6_OK;
}

// j-store, predicted tiles and per-tile index ranges for `need` addresses: grown on demand (doubling) up to c.capacity,
// so a small system does not pay for the largest one (SURVEY.md 8(b) "grown on demand").  Old contents are kept.
int ensure_capacity(Cluster &c, long long need)
{
    if (need <= c.alloc_cap) return G6_OK;
    if (need > c.capacity) return fail(c, G6_ERR_ADDRESS, "%lld addresses asked for, capacity is %d (env G6_NJMAX)", need, c.capacity);
    long long cap = std::max<long long>(need, std::min<long long>(2LL * c.alloc_cap, c.capacity));
    cap = std::min<long long>(((cap + JT - 1) / JT) * JT, c.capacity);
    const size_t tiles = (size_t)(cap / JT), old_tiles = (size_t)(c.alloc_cap / JT);
    char *raw = nullptr;
    float *pred = nullptr;
    int *imin = nullptr, *imax = nullptr;
    int rc = [&]() -> int {
        CK(dalloc(raw, tiles * RAW_TILE_BYTES));
        CK(dalloc(pred, tiles * (size_t)TILE_FLOATS));
        CK(dalloc(imin, tiles)); CK(dalloc(imax, tiles));
        if (old_tiles) CK(cudaMemcpyAsync(raw, c.js.raw, old_tiles * RAW_TILE_BYTES, cudaMemcpyDeviceToDevice, c.stream));
        CK(cudaMemsetAsync(raw + old_tiles * RAW_TILE_BYTES, 0, (tiles - old_tiles) * RAW_TILE_BYTES, c.stream));
        CK(cudaStreamSynchronize(c.stream));       // nothing may still read the old arrays
        return G6_OK;
    }();
    if (rc == G6_OK) {
        try { c.slot_of_addr.resize((size_t)cap, -1); } catch (const std::bad_alloc &) { rc = fail(c, G6_ERR_NOMEM, "host allocation failed"); }
    }
    if (rc != G6_OK) { dfree(raw); dfree(pred); dfree(imin); dfree(imax); return rc; }
    dfree(c.js.raw); dfree(c.pred); dfree(c.tile_imin); dfree(c.tile_imax);
    c.js.raw = raw; c.pred = pred; c.tile_imin = imin; c.tile_imax = imax;
    c.alloc_cap = (int)cap;
    c.pred_valid = false;
    return G6_OK;
}

void release(Cluster &c)
{
    if (c.stream) cudaStreamSynchronize(c.stream);
    dfree(c.js.raw); dfree(c.d_counter);
    dfree(c.pred); dfree(c.tile_imin); dfree(c.tile_imax);
    for (int b = 0; b < 2; ++b) { hfree(c.h_rec[b]); if (c.ev_rec[b]) cudaEventDestroy(c.ev_rec[b]); }
    dfree(c.d_rec);
    free_i(c);
    free_nb(c);
    if (c.part_block) cudaFree(c.part_block);
    if (c.h_bulk) cudaFreeHost(c.h_bulk);
    if (c.d_bulk) cudaFree(c.d_bulk);
    for (auto &e : c.ev) if (e) { cudaEventDestroy(e); e = nullptr; }
    if (c.own_stream) cudaStreamDestroy(c.own_stream);
    char keep[sizeof(c.err)];
    memcpy(keep, c.err, sizeof(keep));
    c = Cluster{};
    memcpy(c.err, keep, sizeof(keep));
}

// zero-copy thresholds: below these the kernels read the staging buffers / write the results
// through mapped pinned memory (no DMA set-up latency); above, one packed copy each way
constexpr int ZC_MAX_I = 2048;
constexpr int ZC_MAX_REC = 2048;

// Step a-1 (+ a-3): scatter of the j particles changed since the last force call and, when
// `with_i`, the i block host staging -> device.  Small batches are read by the kernel straight
// from mapped pinned memory; large ones are DMA-copied first.
int stage_inputs(Cluster &c, bool with_i, int ni)
{
    const int nrec = c.n_rec;
    const int b = c.rec_cur;
    const bool zc_rec = nrec <= ZC_MAX_REC;
    const bool zc_i = with_i && ni <= ZC_MAX_I;
    if (nrec == 0 && !with_i) return G6_OK;
    if (nrec > 0 && !zc_rec)
        CK(cudaMemcpyAsync(c.d_rec, c.h_rec[b], sizeof(JRecord) * nrec, cudaMemcpyHostToDevice, c.stream));
    if (with_i && !zc_i)
        CK(cudaMemcpyAsync(c.d_iblk, c.h_iblk, iblk_bytes(ni), cudaMemcpyHostToDevice, c.stream));
    const int n_i_copy = zc_i ? ni : 0;
    const int nthreads = std::max(nrec, n_i_copy);
    if (nthreads > 0) {
        const IView src = iview(c.hd_iblk, ni), dst = iview(c.d_iblk, ni);
        k_stage<<<(nthreads + 127) / 128, 128, 0, c.stream>>>(c.js, zc_rec ? c.hd_rec[b] : c.d_rec, nrec, n_i_copy,
                                                              src.xi, src.vi, src.idx, (double *)dst.xi, (double *)dst.vi, (int *)dst.idx);
        CK(cudaGetLastError());
    }
    if (nrec > 0) {
        CK(cudaEventRecord(c.ev_rec[b], c.stream));
        c.rec_used[b] = true;
        for (int k = 0; k < nrec; ++k) c.slot_of_addr[c.h_rec[b][k].addr] = -1;
        c.n_rec = 0;
        c.pred_valid = false;
        // switch to the other staging buffer; its previous upload (two flushes ago) must be done
        c.rec_cur = b ^ 1;
        if (c.rec_used[c.rec_cur]) { CK(cudaEventSynchronize(c.ev_rec[c.rec_cur])); c.rec_used[c.rec_cur] = false; }
    }
    return G6_OK;
}

int flush_j(Cluster &c) { return stage_inputs(c, false, 0); }

bool pred_is_current(const Cluster &c)
{
    return c.pred_valid && c.pred_ti == c.ti && c.pred_ds == c.opt_ds && c.pred_n == c.n_stored;
}

// predictor over all stored particles (step a-2); skipped when nothing changed
int run_predict(Cluster &c)
{
    if (pred_is_current(c)) return G6_OK;
    int ntiles = (c.n_stored + JT - 1) / JT;
    if (ntiles > 0) {
        k_predict<<<ntiles, JT, 0, c.stream>>>(c.js, c.n_stored, c.ti, c.opt_ds, c.pred, c.tile_imin, c.tile_imax);
        CK(cudaGetLastError());
    }
    c.pred_valid = true;
    c.pred_ti = c.ti;
    c.pred_ds = c.opt_ds;
    c.pred_n = c.n_stored;
    return G6_OK;
}

// i/j-split scheduler (PAPER.md:82 "j-particles distributed evenly among the P MPs", :104 generalised):
// pick the number of j-splits S that minimises  waves(S) x (tiles per CTA + per-CTA overhead) + tail,
// waves(S) = ceil(i-tiles x S / resident CTA slots), S up to ~4 waves or CTAs of >= 64 tiles, whichever allows more.  Small blocks get S ~ slots (every
// SM busy at n_i = 1); big sweeps get the S that makes the last wave full; in between, whole numbers of
// waves of shorter CTAs (measured at N_j = 2^20, 256 x 1 threads: n_i = 1024 at 1 / 2 / 4 / 8 waves ->
// 0.67 / 0.716 / 0.723 / 0.716 of the FP32 peak; 1.5 or 1.7 waves cost 5-10 %).  Partials are capped at 1 GiB.
int choose_jsplit(int n_itiles, int ntiles, int slots, int ni, long long s_cap = 1LL << 30)
{
    const double OVH = 0.25;       // CTA prologue + epilogue, in tile times
    const double TAIL = 0.06;      // CTAs of the last wave do not finish together: a fraction of one CTA's length is lost
    const double COMBINE = 0.004;  // per extra split: partial traffic + combine work, in tile times
    long long smax = std::min<long long>(ntiles, (1LL << 30) / (72LL * std::max(ni, 1)));
    smax = std::max<long long>(1, std::min<long long>(std::min(smax, s_cap), std::max<long long>(std::max(8, ntiles / 64), 4LL * slots / std::max(n_itiles, 1) + 2)));
    int best = 1;
    double best_cost = 1e300;
    for (int S = 1; S <= smax; ++S) {
        const long long ctas = (long long)n_itiles * S;
        const long long waves = (ctas + slots - 1) / slots;
        const int per = (ntiles + S - 1) / S;
        const double cost = waves * (per + OVH) + TAIL * per + COMBINE * S;
        if (cost < best_cost - 1e-9) { best_cost = cost; best = S; }
    }
    return best;
}

// force + combine (steps a-4, a-5) on device-resident i-blocks; all asynchronous
// small active blocks take the fused block-step kernel unless an experiment switch pins another path
// Largest block the block-step kernel serves: all it is built for (BS_MAX_I = 64).  Since its warps work on sub-tiles
// (g6_block_step.cuh) it beats the sweep path (predictor + sweep kernel + combine: three launches) at every block size it
// takes, measured by CUDA events around the device call, cold L2: n_i = 64 at N_j = 32768 33 us against 50, at N_j = 2^20
// 131 us against 161 (the earlier crossovers were 28 and ~56).  Option "small" set by the caller overrides the rule.
// With neighbour lists the first design runs (lanes over j, a reduction per (i, tile)): its crossovers stay as measured.
int small_limit(const Cluster &c, int nj, bool nb = false)
{
    if (c.small_explicit) return c.opt_small;
    if (!nb && c.opt_bs_design != 1) return BS_MAX_I;
    const int ntiles = (nj + JT - 1) / JT;
    return ntiles >= 1024 ? 64 : (ntiles >= 256 ? 40 : 28);
}

bool use_block_step(const Cluster &c, int ni, int nj, bool nb = false)
{
    // with neighbour lists the kernel's last-CTA merge holds one list per warp in shared memory
    return (!nb || c.opt_nb_maxlen <= BS_NB_SCRATCH) && ni <= small_limit(c, nj, nb) && c.opt_kernel != 1 && c.opt_kernel != 2 && c.opt_jsplit == 0;
}

struct HostBlock { const double *xi, *vi; const int *index; };   // host copy of the i-block (small blocks travel in kernel parameters)
// neighbour-list request of a force call: radii in, combined counts and lists out (all device memory)
struct NbReq { const double *d_h2; int *d_cnt; int *d_list; };

int run_force(Cluster &c, int nj, int ni, const int *d_index, const double *d_xi, const double *d_vi,
              double eps2, double *d_acc, double *d_jerk, double *d_pot, int *d_nn_index, double *d_nn_r2,
              cudaEvent_t ev_pred_done, cudaEvent_t ev_force_done, const HostBlock *hb, const NbReq *nb = nullptr)
{
    c.pend_done_seq = 0;
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

    // small active blocks: the whole block step in one kernel (g6_block_step.cuh)
    if (use_block_step(c, ni, nj, nb != nullptr)) {
        // a-1: changed j-particles ride in the kernel parameters when they fit and lie inside the j-range
        const int maxi_need = std::max(ni, hb ? c.n_rec : 0);
        bool inline_upd = hb && c.n_rec > 0 && c.n_rec <= BS_MAX_I;
        if (inline_upd)
            for (int k = 0; k < c.n_rec; ++k)
                if (c.h_rec[c.rec_cur][k].addr >= A.ntiles * JT) { inline_upd = false; break; }
        if (c.n_rec > 0 && !inline_upd) {
            int rc = flush_j(c);
            if (rc) return rc;
        }
        const bool big = (inline_upd ? maxi_need : ni) > 16;
        const int per_sm = big ? bs_ctas_per_sm<BS_MAX_I>() : bs_ctas_per_sm<16>();
        const int G = std::max(1, std::min(A.ntiles, c.n_sm * per_sm));
        int rc = ensure_partials(c, (size_t)G * ni);
        if (rc) return rc;
        BsArgs B{};
        B.raw = c.js.raw;
        B.ti = c.ti;
        B.nj = nj;
        B.ntiles = A.ntiles;
        B.ni = ni;
        B.n_upd = inline_upd ? c.n_rec : 0;
        B.eps2 = A.eps2;
        B.ds = c.opt_ds;
        B.inline_i = hb ? 1 : 0;
        B.i_index = d_index; B.xi = d_xi; B.vi = d_vi;
        B.P = c.part;
        B.P.stride_s = 1;
        B.P.stride_i = G;
        B.counter = c.d_counter;
        B.acc = d_acc; B.jerk = d_jerk; B.pot = d_pot; B.nn_index = d_nn_index; B.nn_r2 = d_nn_r2;
        if (hb && c.hd_done) {          // host call, results through mapped memory (n_i <= ZC_MAX_I always holds here)
            if (++c.done_seq == 0) ++c.done_seq;
            B.done_flag = c.hd_done;
            B.done_seq = c.done_seq;
            c.pend_done_seq = c.done_seq;
        }
        if (nb) {
            rc = ensure_nb_warp(c, (size_t)G * (BS_THREADS / 32) * ni);
            if (rc) return rc;
            B.h2 = nb->d_h2;
            B.nb_maxlen = c.opt_nb_maxlen;
            B.nb_wcnt = c.d_nb_wcnt;
            B.nb_wlist = c.d_nb_wlist;
            B.nb_cnt = nb->d_cnt;
            B.nb_list = nb->d_list;
        }
        if (ev_pred_done) CK(cudaEventRecord(ev_pred_done, c.stream));     // predictor fused: no separate phase
        const JRecord *upd = inline_upd ? c.h_rec[c.rec_cur] : nullptr;
        // without neighbour lists: the second design (lanes = i-particle x j-sub-range in the pair phase); option "bs_design" = 1 pins the first
        if (!nb && c.opt_bs_design != 1)
            rc = big ? bs2_launch_t<BS_MAX_I>(B, c.opt_newton != 0, G, hb ? hb->xi : nullptr, hb ? hb->vi : nullptr, hb ? hb->index : nullptr, upd, c.stream)
                     : bs2_launch_t<16>(B, c.opt_newton != 0, G, hb ? hb->xi : nullptr, hb ? hb->vi : nullptr, hb ? hb->index : nullptr, upd, c.stream);
        else
        rc = big ? bs_launch_t<BS_MAX_I>(B, c.opt_newton != 0, G, hb ? hb->xi : nullptr, hb ? hb->vi : nullptr, hb ? hb->index : nullptr, upd, c.stream)
                 : bs_launch_t<16>(B, c.opt_newton != 0, G, hb ? hb->xi : nullptr, hb ? hb->vi : nullptr, hb ? hb->index : nullptr, upd, c.stream);
        if (rc) return fail(c, G6_ERR_CUDA, "block-step kernel launch failed: %s", cudaGetErrorString((cudaError_t)rc));
        if (inline_upd) {      // the records were copied into the launch: the staging slots are free again
            for (int k = 0; k < c.n_rec; ++k) c.slot_of_addr[c.h_rec[c.rec_cur][k].addr] = -1;
            c.n_rec = 0;
            c.pred_valid = false;
        }
        if (ev_force_done) CK(cudaEventRecord(ev_force_done, c.stream));
        c.last_ctas = G;
        c.last_S = G;
        c.last_kernel = 3;
        return G6_OK;
    }
    if (c.n_rec > 0) {         // callers of the sweep path have normally flushed already
        int rcf = flush_j(c);
        if (rcf) return rcf;
    }
    int rcp = run_predict(c);
    if (rcp) return rcp;
    if (ev_pred_done) CK(cudaEventRecord(ev_pred_done, c.stream));

    // kernel choice: the fast kernel needs a normal FP32 eps2 > 0 (its unchecked tiles rely on s2 > 0)
    // (the kernel works on eps2 / 3, which must stay a normal float too)
    const bool fast_ok = A.eps2 >= 4.0f * std::numeric_limits<float>::min() && std::isfinite(A.eps2);
    const bool use_fast = (c.opt_kernel == 2 || c.opt_kernel == 0) && fast_ok;

    FastVariant fv = fast_pick(ni, c.n_sm, c.opt_variant);
    if (nb && !fast_has_nb(fv)) fv = fast_pick(ni, c.n_sm, 0);     // lists exist for the automatic shapes only
    const int itile = use_fast ? fv.threads * fv.it : REF_THREADS;
    const int n_itiles = (ni + itile - 1) / itile;
    const int slots = c.n_sm * (use_fast ? (nb ? fast_ctas_per_sm_nb(fv) : fast_ctas_per_sm(fv)) : 8);
    // per-split neighbour lists are capped at 2 GiB
    const long long s_cap = nb ? std::max(1LL, (1LL << 31) / (4LL * c.opt_nb_maxlen * ni)) : (1LL << 30);
    int S = c.opt_jsplit > 0 ? (int)std::min<long long>(c.opt_jsplit, s_cap) : choose_jsplit(n_itiles, A.ntiles, slots, ni, s_cap);
    S = std::max(1, std::min(S, A.ntiles));
    A.S = S;
    int rc = ensure_partials(c, (size_t)S * ni);
    if (rc) return rc;
    if (nb) {
        rc = ensure_nb_part(c, (size_t)S * ni);
        if (rc) return rc;
        A.h2 = nb->d_h2;
        A.nb_maxlen = c.opt_nb_maxlen;
        A.nb_cnt = c.d_nb_pcnt;
        A.nb_list = c.d_nb_plist;
    }
    A.P = c.part;
    const bool wide = S > 8;                 // many splits: [i][s] layout, one warp per i combines
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
    if (ev_force_done) CK(cudaEventRecord(ev_force_done, c.stream));
    if (wide) k_combine_wide<<<(ni + 3) / 4, 128, 0, c.stream>>>(A.P, S, ni, c.js.raw, d_acc, d_jerk, d_pot, d_nn_index, d_nn_r2);
    else k_combine<<<(ni + 255) / 256, 256, 0, c.stream>>>(A.P, S, ni, c.js.raw, d_acc, d_jerk, d_pot, d_nn_index, d_nn_r2);
    CK(cudaGetLastError());
    if (nb) {
        k_combine_nb<<<(ni + 3) / 4, 128, 0, c.stream>>>(c.d_nb_pcnt, c.d_nb_plist, S, ni, c.opt_nb_maxlen, c.js.raw, nb->d_cnt, nb->d_list);
        CK(cudaGetLastError());
    }
    c.last_ctas = n_itiles * S;
    c.last_S = S;
    c.last_kernel = use_fast ? 2 : 1;
    return G6_OK;
}

int check_force_args(Cluster &c, int nj, int ni)
{
    init_npipes();
    if (ni < 1 || ni > g_npipes) return fail(c, G6_ERR_NI, "ni = %d outside [1, g6_npipes() = %d]", ni, g_npipes);
    if (nj < 1 || nj > c.n_stored) return fail(c, G6_ERR_NJ, "nj = %d outside [1, stored = %d]", nj, c.n_stored);
    return G6_OK;
}

}  // namespace

// ================================================================================ C ABI =====
extern "C" {

int g6_npipes(void)
{
    init_npipes();
    return g_npipes;
}

int g6x_set_npipes(int npipes)
{
    if (npipes < 1 || npipes > MAX_NPIPES) return G6_ERR_ARG;
    g_npipes = npipes;
    return G6_OK;
}

const char *g6x_version(void)
{
    return "libg6b200 0.2 (sm_100a; FP32 + double-single separations; kernels: ref, fast[FFMA2+TMA, neighbour lists], block-step[TMA ring]; j-split exchange)";
}

const char *g6x_last_error(int clusterid)
{
    if (clusterid < 0 || clusterid >= MAX_CLUSTERS) return "clusterid out of range";
    return g_cl[clusterid].err;
}

int g6_open(int clusterid)
{
    if (clusterid < 0 || clusterid >= MAX_CLUSTERS) return G6_ERR_CLUSTER;
    Cluster &c = g_cl[clusterid];
    if (c.open) return fail(c, G6_ERR_ALREADY_OPEN, "cluster %d is already open", clusterid);
    init_npipes();
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev < 1)
        return fail(c, G6_ERR_CUDA, "no CUDA device (%s); this library has no CPU path",
                    e == cudaSuccess ? "device count 0" : cudaGetErrorString(e));
    c.device = env_int("G6_DEVICE", 0);
    if (c.device < 0 || c.device >= ndev) return fail(c, G6_ERR_CUDA, "G6_DEVICE = %d but %d devices", c.device, ndev);
    CK(cudaSetDevice(c.device));
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, c.device));
    if (prop.major < 10)
        return fail(c, G6_ERR_CUDA, "device %s is sm_%d%d; this library is built for sm_100a only", prop.name,
                    prop.major, prop.minor);
    c.n_sm = prop.multiProcessorCount;
    c.capacity = std::max(JT, env_int("G6_NJMAX", 1 << 21));
    c.capacity = ((c.capacity + JT - 1) / JT) * JT;
    int rc = [&]() -> int {
        CK(cudaStreamCreateWithFlags(&c.own_stream, cudaStreamNonBlocking));
        c.stream = c.own_stream;
        CK(dalloc(c.d_counter, 1));     // arrival ticket of the block-step kernel
        CK(cudaMemsetAsync(c.d_counter, 0, sizeof(unsigned int), c.stream));
        for (auto &ev : c.ev) CK(cudaEventCreate(&ev));
        for (auto &ev : c.ev_rec) CK(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
        int r = fast_kernel_init();
        if (!r) r = bs_kernel_init();
        if (r) return fail(c, G6_ERR_CUDA, "kernel attribute setup failed: %s", cudaGetErrorString((cudaError_t)r));
        return G6_OK;
    }();
    // the j-store starts at env G6_NJINIT addresses (default 16384 = 1.9 MB of device memory) and doubles on demand
    if (rc == G6_OK) rc = ensure_capacity(c, std::min(c.capacity, std::max(JT, env_int("G6_NJINIT", 16384))));
    if (rc != G6_OK) { release(c); return rc; }
    c.open = true;
    c.opt_newton = env_int("G6_NEWTON", 1) ? 1 : 0;
    c.opt_kernel = env_int("G6_KERNEL", 0);
    c.opt_timers = env_int("G6_TIMERS", 0) ? 1 : 0;
    snprintf(c.err, sizeof(c.err), "no error");
    return G6_OK;
}

int g6_close(int clusterid)
{
    GET_CLUSTER(clusterid);
    release(c);
    return G6_OK;
}

int g6_set_j_particle(int clusterid, int address, int index, double tj, double dtj, double mass,
                      const double snap_by18[3], const double jerk_by6[3], const double acc_by2[3],
                      const double v[3], const double x[3])
{
    GET_CLUSTER(clusterid);
    (void)dtj; (void)snap_by18;
    if (address < 0 || address >= c.capacity)
        return fail(c, G6_ERR_ADDRESS, "address %d outside [0, capacity = %d)", address, c.capacity);
    if (!jerk_by6 || !acc_by2 || !v || !x) return fail(c, G6_ERR_ARG, "NULL array in g6_set_j_particle");
    if (address >= c.alloc_cap) {
        int rc = ensure_capacity(c, (long long)address + 1);
        if (rc) return rc;
    }
    int slot = c.slot_of_addr[address];
    if (slot < 0) {
        int rc = ensure_rec(c, c.n_rec + 1);
        if (rc) return rc;
        slot = c.n_rec++;
        c.slot_of_addr[address] = slot;
    }
    JRecord &r = c.h_rec[c.rec_cur][slot];
    for (int k = 0; k < 3; ++k) {
        r.x[k] = x[k];
        r.v[k] = (float)v[k];
        r.a2[k] = (float)acc_by2[k];
        r.j6[k] = (float)jerk_by6[k];
    }
    r.t = tj;
    r.m = (float)mass;
    r.idx = index;
    r.addr = address;
    c.n_stored = std::max(c.n_stored, address + 1);
    return G6_OK;
}

int g6x_set_j_particles_dev(int clusterid, int addr0, int n, const int *d_index, const double *d_tj,
                            const double *d_mass, const double *d_jerk, const double *d_acc,
                            const double *d_v, const double *d_x)
{
    GET_CLUSTER(clusterid);
    if (n < 1) return fail(c, G6_ERR_ARG, "n = %d", n);
    if (addr0 < 0 || (long long)addr0 + n > c.capacity)
        return fail(c, G6_ERR_ADDRESS, "addresses [%d, %lld) outside capacity %d", addr0, (long long)addr0 + n, c.capacity);
    if (!d_index || !d_tj || !d_mass || !d_jerk || !d_acc || !d_v || !d_x) return fail(c, G6_ERR_ARG, "NULL device array");
    int rc = ensure_capacity(c, (long long)addr0 + n);
    if (rc) return rc;
    rc = flush_j(c);   // keep program order with earlier g6_set_j_particle calls
    if (rc) return rc;
    k_store_from_f64<<<(n + 255) / 256, 256, 0, c.stream>>>(c.js, addr0, n, d_index, d_tj, d_mass, d_jerk, d_acc, d_v, d_x);
    CK(cudaGetLastError());
    c.n_stored = std::max(c.n_stored, addr0 + n);
    c.pred_valid = false;
    return G6_OK;
}

int g6x_set_j_particles(int clusterid, int addr0, int n, const int index[], const double tj[],
                        const double mass[], const double jerk[][3], const double acc[][3],
                        const double v[][3], const double x[][3])
{
    GET_CLUSTER(clusterid);
    if (n < 1) return fail(c, G6_ERR_ARG, "n = %d", n);
    if (addr0 < 0 || (long long)addr0 + n > c.capacity)
        return fail(c, G6_ERR_ADDRESS, "addresses [%d, %lld) outside capacity %d", addr0, (long long)addr0 + n, c.capacity);
    if (!index || !tj || !mass || !jerk || !acc || !v || !x) return fail(c, G6_ERR_ARG, "NULL array");
    // staging layout: x v acc jerk [n][3] f64, tj mass [n] f64, index [n] i32
    const size_t n3 = 3 * (size_t)n * sizeof(double), n1 = (size_t)n * sizeof(double);
    const size_t bytes = 4 * n3 + 2 * n1 + (size_t)n * sizeof(int);
    int rc = ensure_bulk(c, bytes);
    if (rc) return rc;
    CK(cudaStreamSynchronize(c.stream));   // previous bulk upload must have left the pinned buffer
    char *h = (char *)c.h_bulk, *d = (char *)c.d_bulk;
    big_memcpy(h, x, n3); big_memcpy(h + n3, v, n3); big_memcpy(h + 2 * n3, acc, n3); big_memcpy(h + 3 * n3, jerk, n3);
    big_memcpy(h + 4 * n3, tj, n1); big_memcpy(h + 4 * n3 + n1, mass, n1); big_memcpy(h + 4 * n3 + 2 * n1, index, (size_t)n * sizeof(int));
    CK(cudaMemcpyAsync(d, h, bytes, cudaMemcpyHostToDevice, c.stream));
    return g6x_set_j_particles_dev(clusterid, addr0, n, (const int *)(d + 4 * n3 + 2 * n1), (const double *)(d + 4 * n3),
                                   (const double *)(d + 4 * n3 + n1), (const double *)(d + 3 * n3),
                                   (const double *)(d + 2 * n3), (const double *)(d + n3), (const double *)d);
}

// ---- the rest of the GRAPE-6 calling sequence (names and meanings recalled, unverified) ----
int g_tunit = 0, g_xunit = 0;     // GRAPE-6 fixed-point scales: kept for the caller, no effect on fp64 / double-single data

int g6_set_tunit(int newtunit) { g_tunit = newtunit; return G6_OK; }
int g6_set_xunit(int newxunit) { g_xunit = newxunit; return G6_OK; }
int g6x_get_units(int *tunit, int *xunit)
{
    if (!tunit || !xunit) return G6_ERR_ARG;
    *tunit = g_tunit;
    *xunit = g_xunit;
    return G6_OK;
}

int g6_reset(int clusterid)
{
    GET_CLUSTER(clusterid);
    CK(cudaStreamSynchronize(c.stream));
    if (c.alloc_cap) CK(cudaMemsetAsync(c.js.raw, 0, (size_t)(c.alloc_cap / JT) * RAW_TILE_BYTES, c.stream));
    std::fill(c.slot_of_addr.begin(), c.slot_of_addr.end(), -1);
    c.n_rec = 0;
    c.n_stored = 0;
    c.pred_valid = false;
    c.pending = false;
    c.have_result = false;
    c.pend_done_seq = 0;
    c.last_nb = c.nb_on_host = false;
    c.ti = 0.0;
    return G6_OK;
}

int g6_reset_fofpga(int clusterid)
{
    GET_CLUSTER(clusterid);      // there is no force-output FPGA to reset; the call only checks the cluster
    return G6_OK;
}

int g6_initialize_jp_buffer(int clusterid, int buf_size)
{
    GET_CLUSTER(clusterid);
    if (buf_size < 1) return fail(c, G6_ERR_ARG, "buf_size = %d", buf_size);
    return ensure_rec(c, std::min(buf_size, c.capacity));
}

int g6_flush_jp_buffer(int clusterid)
{
    GET_CLUSTER(clusterid);
    if (c.pending) return fail(c, G6_ERR_SEQUENCE, "g6_flush_jp_buffer between firsthalf and lasthalf");
    return flush_j(c);
}

int g6_getnjmax(int clusterid)
{
    GET_CLUSTER(clusterid);
    return c.capacity;
}

int g6x_get_j_particles(int clusterid, int addr0, int n, int index[], double tj[], double mass[], double jerk[][3],
                        double acc[][3], double v[][3], double x[][3])
{
    GET_CLUSTER(clusterid);
    if (c.pending) return fail(c, G6_ERR_SEQUENCE, "j-particle read-back between firsthalf and lasthalf");
    if (n < 1 || addr0 < 0 || (long long)addr0 + n > c.n_stored)
        return fail(c, G6_ERR_ADDRESS, "addresses [%d, %lld) outside stored [0, %d)", addr0, (long long)addr0 + n, c.n_stored);
    int rc = flush_j(c);
    if (rc) return rc;
    JRecord *d = nullptr;
    std::vector<JRecord> h;
    try { h.resize(n); } catch (const std::bad_alloc &) { return fail(c, G6_ERR_NOMEM, "host allocation failed"); }
    rc = [&]() -> int {
        CK(dalloc(d, n));
        k_fetch_records<<<(n + 127) / 128, 128, 0, c.stream>>>(c.js, addr0, n, d);
        CK(cudaGetLastError());
        CK(cudaMemcpyAsync(h.data(), d, sizeof(JRecord) * n, cudaMemcpyDeviceToHost, c.stream));
        CK(cudaStreamSynchronize(c.stream));
        return G6_OK;
    }();
    dfree(d);
    if (rc) return rc;
    for (int p = 0; p < n; ++p) {
        const JRecord &r = h[p];
        if (index) index[p] = r.idx;
        if (tj) tj[p] = r.t;
        if (mass) mass[p] = (double)r.m;
        for (int k = 0; k < 3; ++k) {
            if (x) x[p][k] = r.x[k];
            if (v) v[p][k] = (double)r.v[k];
            if (acc) acc[p][k] = 2.0 * (double)r.a2[k];
            if (jerk) jerk[p][k] = 6.0 * (double)r.j6[k];
        }
    }
    return G6_OK;
}

int g6_get_j_particle(int clusterid, int address, int *index, double *tj, double *mass, double jerk_by6[3],
                      double acc_by2[3], double v[3], double x[3])
{
    double j[1][3], a[1][3], vv[1][3], xx[1][3], t = 0, m = 0;
    int idx = 0;
    int rc = g6x_get_j_particles(clusterid, address, 1, &idx, &t, &m, j, a, vv, xx);
    if (rc) return rc;
    if (index) *index = idx;
    if (tj) *tj = t;
    if (mass) *mass = m;
    for (int k = 0; k < 3; ++k) {
        if (jerk_by6) jerk_by6[k] = j[0][k] / 6.0;      // exact: the stored binary32 value
        if (acc_by2) acc_by2[k] = a[0][k] / 2.0;
        if (v) v[k] = vv[0][k];
        if (x) x[k] = xx[0][k];
    }
    return G6_OK;
}

int g6_set_ti(int clusterid, double ti)
{
    GET_CLUSTER(clusterid);
    c.ti = ti;
    return G6_OK;
}

int g6x_calc_dev(int clusterid, int nj, int ni, const int *d_index, const double *d_xi, const double *d_vi,
                 double eps2, double *d_acc, double *d_jerk, double *d_pot, int *d_nn_index, double *d_nn_r2)
{
    return g6x_calc_dev_nb(clusterid, nj, ni, d_index, d_xi, d_vi, eps2, d_acc, d_jerk, d_pot, d_nn_index, d_nn_r2,
                           nullptr, nullptr, nullptr);
}

int g6x_calc_dev_nb(int clusterid, int nj, int ni, const int *d_index, const double *d_xi, const double *d_vi,
                    double eps2, double *d_acc, double *d_jerk, double *d_pot, int *d_nn_index, double *d_nn_r2,
                    const double *d_h2, int *d_nb_count, int *d_nb_list)
{
    GET_CLUSTER(clusterid);
    if ((d_h2 != nullptr) != (d_nb_count != nullptr) || (d_h2 != nullptr) != (d_nb_list != nullptr))
        return fail(c, G6_ERR_ARG, "d_h2, d_nb_count and d_nb_list must be given together");
    const NbReq nbr{d_h2, d_nb_count, d_nb_list};
    if (c.pending) return fail(c, G6_ERR_SEQUENCE, "g6x_calc_dev between firsthalf and lasthalf");
    int rc = flush_j(c);
    if (rc) return rc;
    rc = check_force_args(c, nj, ni);
    if (rc) return rc;
    if (!d_index || !d_xi || !d_vi || !d_acc || !d_jerk || !d_pot) return fail(c, G6_ERR_ARG, "NULL device array");
    if (!(eps2 >= 0.0)) return fail(c, G6_ERR_ARG, "eps2 = %g", eps2);
    const bool tm = c.opt_timers != 0;
    if (tm) { CK(cudaEventRecord(c.ev[0], c.stream)); CK(cudaEventRecord(c.ev[1], c.stream)); }
    rc = run_force(c, nj, ni, d_index, d_xi, d_vi, eps2, d_acc, d_jerk, d_pot, d_nn_index, d_nn_r2, tm ? c.ev[2] : nullptr,
                   tm ? c.ev[3] : nullptr, nullptr, d_h2 ? &nbr : nullptr);
    if (rc) return rc;
    if (tm) { CK(cudaEventRecord(c.ev[4], c.stream)); CK(cudaEventRecord(c.ev[5], c.stream)); }
    c.ev_valid = tm;
    return G6_OK;
}

int g6calc_firsthalf(int clusterid, int nj, int ni, const int index[], const double xi[][3], const double vi[][3],
                     const double acc_old[][3], const double jerk6_old[][3], const double phi_old[],
                     double eps2, const double h2[])
{
    GET_CLUSTER(clusterid);
    (void)acc_old; (void)jerk6_old; (void)phi_old;
    if (c.pending) return fail(c, G6_ERR_SEQUENCE, "g6calc_firsthalf called twice without g6calc_lasthalf");
    int rc = check_force_args(c, nj, ni);
    if (rc) return rc;
    if (!index || !xi || !vi) return fail(c, G6_ERR_ARG, "NULL i-particle array");
    if (!(eps2 >= 0.0)) return fail(c, G6_ERR_ARG, "eps2 = %g", eps2);
    rc = ensure_i(c, ni);
    if (rc) return rc;
    const bool tm = c.opt_timers != 0;
    if (tm) CK(cudaEventRecord(c.ev[0], c.stream));
    // neighbour lists when the caller passes radii
    const bool want_nb = h2 != nullptr;
    NbReq nbr{nullptr, nullptr, nullptr};
    if (want_nb) {
        rc = ensure_nb_host(c, ni);
        if (rc) return rc;
        memcpy(c.h_h2, h2, sizeof(double) * ni);
        CK(cudaMemcpyAsync(c.d_h2, c.h_h2, sizeof(double) * ni, cudaMemcpyHostToDevice, c.stream));
        nbr = NbReq{c.d_h2, c.d_nb_cnt, c.d_nb_list};
    }
    const bool bs = use_block_step(c, ni, nj, want_nb);
    const bool zc_out = ni <= ZC_MAX_I;
    const RView out = rview(zc_out ? c.hd_res : c.d_res, ni);
    if (bs) {
        // small block: the i-block and the changed j-particles travel inside the kernel launch
        // (copied from the caller's arrays by the launch itself); results come back through mapped memory
        if (tm) CK(cudaEventRecord(c.ev[1], c.stream));
        const HostBlock hb{&xi[0][0], &vi[0][0], index};
        {   // keep a host copy for the debug read-backs
            const IView hv = iview(c.h_iblk, ni);
            big_memcpy((void *)hv.xi, xi, sizeof(double) * 3 * ni);
            big_memcpy((void *)hv.vi, vi, sizeof(double) * 3 * ni);
            big_memcpy((void *)hv.idx, index, sizeof(int) * ni);
        }
        c.iblk_on_device = false;
        rc = run_force(c, nj, ni, nullptr, nullptr, nullptr, eps2, out.acc, out.jerk, out.pot, out.nnidx, out.nnr2, tm ? c.ev[2] : nullptr,
                       tm ? c.ev[3] : nullptr, &hb, want_nb ? &nbr : nullptr);
        if (rc) return rc;
    } else {
        // a-3: i block to pinned staging (the only per-step H2D payload) ...
        {
            const IView hv = iview(c.h_iblk, ni);
            big_memcpy((void *)hv.xi, xi, sizeof(double) * 3 * ni);
            big_memcpy((void *)hv.vi, vi, sizeof(double) * 3 * ni);
            big_memcpy((void *)hv.idx, index, sizeof(int) * ni);
        }
        // ... and, together with a-1 (changed j particles), on to the device
        rc = stage_inputs(c, true, ni);
        if (rc) return rc;
        c.iblk_on_device = true;
        if (tm) CK(cudaEventRecord(c.ev[1], c.stream));
        // a-2 (separate predictor kernel), a-4, a-5; blocks up to ZC_MAX_I: the combine kernel writes the
        // results straight into mapped host memory (a-6)
        const IView dv = iview(c.d_iblk, ni);
        rc = run_force(c, nj, ni, dv.idx, dv.xi, dv.vi, eps2, out.acc, out.jerk, out.pot, out.nnidx, out.nnr2, tm ? c.ev[2] : nullptr,
                       tm ? c.ev[3] : nullptr, nullptr, want_nb ? &nbr : nullptr);
        if (rc) return rc;
    }
    if (tm) CK(cudaEventRecord(c.ev[4], c.stream));
    // a-6
    if (!zc_out) CK(cudaMemcpyAsync(c.h_res, c.d_res, res_bytes(ni), cudaMemcpyDeviceToHost, c.stream));
    CK(cudaEventRecord(c.ev[5], c.stream));
    c.res_on_host = zc_out;
    c.ev_valid = tm;
    c.pending = true;
    c.pend_nj = nj;
    c.pend_ni = ni;
    c.pend_nb = want_nb;
    return G6_OK;
}

int g6calc_lasthalf2(int clusterid, int nj, int ni, const int index[], const double xi[][3], const double vi[][3],
                     double eps2, const double h2[], double acc[][3], double jerk[][3], double pot[], int nnb_index[])
{
    GET_CLUSTER(clusterid);
    (void)index; (void)xi; (void)vi; (void)eps2; (void)h2;
    if (!c.pending) return fail(c, G6_ERR_SEQUENCE, "g6calc_lasthalf without g6calc_firsthalf");
    if (nj != c.pend_nj || ni != c.pend_ni)
        return fail(c, G6_ERR_ARG, "lasthalf (nj=%d, ni=%d) does not match firsthalf (nj=%d, ni=%d)", nj, ni, c.pend_nj, c.pend_ni);
    if (!acc || !jerk || !pot) return fail(c, G6_ERR_ARG, "NULL result array");
    c.pending = false;
    if (c.pend_done_seq) {
        // the block-step kernel flags its results in mapped memory: spin on the word (sooner than an event wait), with a
        // look at the stream now and then so that a failed launch cannot hang the caller
        volatile unsigned int *flag = c.h_done;
        for (unsigned long long spins = 1; *flag != c.pend_done_seq; ++spins) {
            if ((spins & 0x3fff) == 0) {
                const cudaError_t q = cudaStreamQuery(c.stream);
                if (q == cudaSuccess) {
                    if (*flag == c.pend_done_seq) break;
                    return fail(c, G6_ERR_CUDA, "force call finished without flagging its results");
                }
                if (q != cudaErrorNotReady) return fail(c, G6_ERR_CUDA, "force call failed: %s", cudaGetErrorString(q));
            }
        }
        std::atomic_thread_fence(std::memory_order_acquire);
    } else {
        CK(cudaEventSynchronize(c.ev[5]));
    }
    const RView r = rview(c.h_res, ni);
    big_memcpy(acc, r.acc, sizeof(double) * 3 * ni);
    big_memcpy(jerk, r.jerk, sizeof(double) * 3 * ni);
    big_memcpy(pot, r.pot, sizeof(double) * ni);
    if (nnb_index) memcpy(nnb_index, r.nnidx, sizeof(int) * ni);
    c.have_result = true;
    c.last_ni = ni;
    c.last_nb = c.pend_nb;
    c.nb_on_host = false;
    c.last_nb_maxlen = c.opt_nb_maxlen;
    return G6_OK;
}

int g6calc_lasthalf(int clusterid, int nj, int ni, const int index[], const double xi[][3], const double vi[][3],
                    double eps2, const double h2[], double acc[][3], double jerk[][3], double pot[])
{
    return g6calc_lasthalf2(clusterid, nj, ni, index, xi, vi, eps2, h2, acc, jerk, pot, nullptr);
}

// copy the combined lists of the last host force call to the host (once)
static int nb_fetch(Cluster &c)
{
    if (c.nb_on_host) return G6_OK;
    if (c.last_nb_maxlen != c.nb_alloc_maxlen || c.last_ni > c.nb_cap)
        return fail(c, G6_ERR_SEQUENCE, "neighbour lists of the last force call are gone (nb_maxlen changed)");
    const size_t ni = c.last_ni, ml = c.last_nb_maxlen;
    CK(cudaMemcpyAsync(c.h_nb_cnt, c.d_nb_cnt, sizeof(int) * ni, cudaMemcpyDeviceToHost, c.stream));
    CK(cudaMemcpyAsync(c.h_nb_list, c.d_nb_list, sizeof(int) * ni * ml, cudaMemcpyDeviceToHost, c.stream));
    CK(cudaStreamSynchronize(c.stream));
    c.nb_on_host = true;
    return G6_OK;
}

int g6_read_neighbour_list(int clusterid)
{
    GET_CLUSTER(clusterid);
    if (c.pending || !c.have_result) return fail(c, G6_ERR_SEQUENCE, "no completed force call to read neighbours of");
    if (!c.last_nb) return 0;
    int rc = nb_fetch(c);
    if (rc) return rc;
    int over = 0;
    for (int i = 0; i < c.last_ni; ++i) over += c.h_nb_cnt[i] > c.last_nb_maxlen;
    return over;
}

int g6_get_neighbour_list(int clusterid, int ipipe, int maxlen, int *n, int list[])
{
    GET_CLUSTER(clusterid);
    if (c.pending || !c.have_result) return fail(c, G6_ERR_SEQUENCE, "no completed force call");
    if (ipipe < 0 || ipipe >= c.last_ni) return fail(c, G6_ERR_ARG, "ipipe = %d outside [0, %d)", ipipe, c.last_ni);
    if (!n || !list || maxlen < 1) return fail(c, G6_ERR_ARG, "bad neighbour list buffer");
    if (c.last_nb) {
        int rc = nb_fetch(c);
        if (rc) return rc;
        const int cnt = c.h_nb_cnt[ipipe];
        const int stored = std::min(cnt, c.last_nb_maxlen);
        const int ncopy = std::min(stored, maxlen);
        memcpy(list, c.h_nb_list + (size_t)ipipe * c.last_nb_maxlen, sizeof(int) * ncopy);
        *n = ncopy;
        return ncopy < cnt ? 1 : 0;
    }
    const int nb = rview(c.h_res, c.last_ni).nnidx[ipipe];
    if (nb >= 0) { *n = 1; list[0] = nb; }
    else *n = 0;
    return G6_OK;
}

int g6x_get_neighbour_lists(int clusterid, int ni, int maxlen, int count[], int list[])
{
    GET_CLUSTER(clusterid);
    if (c.pending || !c.have_result) return fail(c, G6_ERR_SEQUENCE, "no completed force call");
    if (!c.last_nb) return fail(c, G6_ERR_SEQUENCE, "the last force call built no neighbour lists (h2 was NULL)");
    if (ni != c.last_ni) return fail(c, G6_ERR_ARG, "ni = %d but the last call had %d", ni, c.last_ni);
    if (!count || !list || maxlen < 1) return fail(c, G6_ERR_ARG, "bad neighbour list buffer");
    int rc = nb_fetch(c);
    if (rc) return rc;
    int over = 0;
    for (int i = 0; i < ni; ++i) {
        const int cnt = c.h_nb_cnt[i];
        const int ncopy = std::min(std::min(cnt, c.last_nb_maxlen), maxlen);
        count[i] = cnt;
        memcpy(list + (size_t)i * maxlen, c.h_nb_list + (size_t)i * c.last_nb_maxlen, sizeof(int) * ncopy);
        for (int k = ncopy; k < maxlen; ++k) list[(size_t)i * maxlen + k] = -1;
        over += ncopy < cnt;
    }
    return over;
}

int g6x_get_nearest(int clusterid, int ni, int nn_index[], double nn_r2[])
{
    GET_CLUSTER(clusterid);
    if (c.pending || !c.have_result) return fail(c, G6_ERR_SEQUENCE, "no completed force call");
    if (ni != c.last_ni) return fail(c, G6_ERR_ARG, "ni = %d but the last call had %d", ni, c.last_ni);
    const RView r = rview(c.h_res, ni);
    if (nn_index) memcpy(nn_index, r.nnidx, sizeof(int) * ni);
    if (nn_r2) memcpy(nn_r2, r.nnr2, sizeof(double) * ni);
    return G6_OK;
}

int g6x_set_stream(int clusterid, void *cuda_stream)
{
    GET_CLUSTER(clusterid);
    if (c.pending) return fail(c, G6_ERR_SEQUENCE, "stream change between firsthalf and lasthalf");
    CK(cudaStreamSynchronize(c.stream));
    c.stream = cuda_stream ? (cudaStream_t)cuda_stream : c.own_stream;
    return G6_OK;
}

int g6x_synchronize(int clusterid)
{
    GET_CLUSTER(clusterid);
    CK(cudaStreamSynchronize(c.stream));
    return G6_OK;
}

int g6x_get_timers(int clusterid, double us[8])
{
    GET_CLUSTER(clusterid);
    if (!us) return fail(c, G6_ERR_ARG, "NULL");
    if (c.pending) return fail(c, G6_ERR_SEQUENCE, "force call still pending");
    if (!c.ev_valid) return fail(c, G6_ERR_SEQUENCE, "no timed force call (option timers = 0?)");
    CK(cudaEventSynchronize(c.ev[5]));
    for (int k = 0; k < 5; ++k) {
        float ms = 0;
        CK(cudaEventElapsedTime(&ms, c.ev[k], c.ev[k + 1]));
        us[k] = 1e3 * ms;
    }
    float ms = 0;
    CK(cudaEventElapsedTime(&ms, c.ev[0], c.ev[5]));
    us[5] = 1e3 * ms;
    us[6] = c.last_ctas;
    us[7] = c.last_S;
    return G6_OK;
}

static int *option_slot(Cluster &c, const char *key)
{
    if (!key) return nullptr;
    if (!strcmp(key, "ds")) return &c.opt_ds;
    if (!strcmp(key, "newton")) return &c.opt_newton;
    if (!strcmp(key, "jsplit")) return &c.opt_jsplit;
    if (!strcmp(key, "kernel")) return &c.opt_kernel;
    if (!strcmp(key, "timers")) return &c.opt_timers;
    if (!strcmp(key, "variant")) return &c.opt_variant;
    if (!strcmp(key, "small")) return &c.opt_small;
    if (!strcmp(key, "nb_maxlen")) return &c.opt_nb_maxlen;
    if (!strcmp(key, "bs_design")) return &c.opt_bs_design;
    return nullptr;
}

int g6x_set_option(int clusterid, const char *key, int value)
{
    GET_CLUSTER(clusterid);
    int *slot = option_slot(c, key);
    if (!slot) return fail(c, G6_ERR_ARG, "unknown option '%s'", key ? key : "(null)");
    const bool is_flag = slot == &c.opt_ds || slot == &c.opt_newton || slot == &c.opt_timers;
    if (value < 0 || (is_flag && value > 1) || (slot == &c.opt_kernel && value > 2) || (slot == &c.opt_jsplit && value > 65535) || (slot == &c.opt_small && value > BS_MAX_I) || (slot == &c.opt_bs_design && value > 2) ||
        (slot == &c.opt_nb_maxlen && (value < 1 || value > 4096)) ||
        (slot == &c.opt_variant && value != 0 && !fast_is_built(FastVariant{value / 8, value % 8}, true)))
        return fail(c, G6_ERR_ARG, "bad value %d for option '%s'", value, key);
    *slot = value;
    if (slot == &c.opt_small) c.small_explicit = true;
    return G6_OK;
}

int g6x_get_option(int clusterid, const char *key, int *value)
{
    GET_CLUSTER(clusterid);
    if (key && value && !strcmp(key, "last_kernel")) { *value = c.last_kernel; return G6_OK; }
    int *slot = option_slot(c, key);
    if (!slot || !value) return fail(c, G6_ERR_ARG, "unknown option '%s'", key ? key : "(null)");
    *value = *slot;
    return G6_OK;
}

int g6x_get_predicted(int clusterid, int addr0, int n, double xp[][3], double vp[][3])
{
    GET_CLUSTER(clusterid);
    if (c.pending) return fail(c, G6_ERR_SEQUENCE, "force call pending");
    int rc = flush_j(c);
    if (rc) return rc;
    if (n < 1 || addr0 < 0 || (long long)addr0 + n > c.n_stored)
        return fail(c, G6_ERR_ADDRESS, "addresses [%d, %lld) outside stored [0, %d)", addr0, (long long)addr0 + n, c.n_stored);
    if (!xp || !vp) return fail(c, G6_ERR_ARG, "NULL");
    rc = run_predict(c);
    if (rc) return rc;
    const int t0 = addr0 / JT, t1 = (addr0 + n - 1) / JT + 1;
    std::vector<float> h;
    try { h.resize((size_t)(t1 - t0) * TILE_FLOATS); } catch (const std::bad_alloc &) { return fail(c, G6_ERR_NOMEM, "host allocation failed"); }
    CK(cudaMemcpyAsync(h.data(), c.pred + (size_t)t0 * TILE_FLOATS, h.size() * sizeof(float), cudaMemcpyDeviceToHost, c.stream));
    CK(cudaStreamSynchronize(c.stream));
    for (int p = 0; p < n; ++p) {
        const int a = addr0 + p;
        const float *t = h.data() + (size_t)(a / JT - t0) * TILE_FLOATS + (a % JT);
        for (int k = 0; k < 3; ++k) {
            xp[p][k] = (double)t[(F_XH + k) * JT] + (double)t[(F_XL + k) * JT];
            vp[p][k] = (double)t[(F_V + k) * JT];
        }
    }
    return G6_OK;
}

int g6x_jsplit_pack_dev(int clusterid, int ni, int rank, const double *d_nn_r2, const int *d_nn_index, long long *d_key)
{
    GET_CLUSTER(clusterid);
    if (ni < 1 || rank < 0 || !d_nn_r2 || !d_nn_index || !d_key) return fail(c, G6_ERR_ARG, "bad j-split pack arguments");
    k_jsplit_pack<<<(ni + 255) / 256, 256, 0, c.stream>>>(ni, rank, d_nn_r2, d_nn_index, d_key);
    CK(cudaGetLastError());
    return G6_OK;
}

int g6x_jsplit_select_dev(int clusterid, int ni, int rank, const long long *d_key_min, const int *d_nn_index, double *d_index_f64)
{
    GET_CLUSTER(clusterid);
    if (ni < 1 || rank < 0 || !d_key_min || !d_nn_index || !d_index_f64) return fail(c, G6_ERR_ARG, "bad j-split select arguments");
    k_jsplit_select<<<(ni + 255) / 256, 256, 0, c.stream>>>(ni, rank, d_key_min, d_nn_index, d_index_f64);
    CK(cudaGetLastError());
    return G6_OK;
}

int g6x_jsplit_unpack_dev(int clusterid, int ni, const long long *d_key_min, const double *d_index_sum, int *d_nn_index, double *d_nn_r2)
{
    GET_CLUSTER(clusterid);
    if (ni < 1 || !d_key_min || !d_index_sum) return fail(c, G6_ERR_ARG, "bad j-split unpack arguments");
    k_jsplit_unpack<<<(ni + 255) / 256, 256, 0, c.stream>>>(ni, d_key_min, d_index_sum, d_nn_index, d_nn_r2);
    CK(cudaGetLastError());
    return G6_OK;
}

}  // extern "C"

// device-resident Hermite integrator (g6hd_*, include/g6_hermite.h): needs the internals above
#include "g6_hermite_dev_api.cuh"

// force call that allocates nothing (g6x_calc_dev_noalloc): partials in a fixed file-scope device array
#include "g6_noalloc.cuh"
