// g6_hermite_dev_api.cuh -- host side of the device-resident Hermite integrator (include/g6_hermite.h, g6hd_*).
// Included at the end of g6_api.cu: it drives the library's own force path (run_force) on device-resident
// i-blocks and keeps the whole particle state in HBM.  Per block step the host waits once, for (n_i, t_next).
#pragma once
#include "../../include/g6_hermite.h"
#include "g6_hermite_dev.cuh"
#include "g6_hermite_loop.cuh"

#include <atomic>
#include <chrono>

struct g6hd_system {
    int cl = 0, n = 0;
    double eps2 = 0, eta = 0, dt_max = 0, t = 0;
    HdState S{};
    HdBlock B{};
    double *a1 = nullptr, *ad1 = nullptr, *pot = nullptr;      // forces of the current block [n][3], [n]
    unsigned long long *dt_min_bits = nullptr;                // smallest step used so far (bits of a positive double)
    HdNote *h_note = nullptr;                                  // mapped host memory
    unsigned int seq = 0;
    int last_ni = 0;
    bool shared = false;                                       // one common step for all particles (reading 21)
    unsigned long long *shared_bits = nullptr;                 // the common step of the next shared step (bits of a double)
    bool pending = false;                                      // the last block's forces are computed, its corrector has not run yet
    long long nblock = 0, npart = 0, hist[64] = {};
    double inter = 0, wall = 0;
    // env G6_HD_PROFILE=1: device time of the three phases of every block step (CUDA events; slows the loop down)
    bool profile = false;
    cudaEvent_t pe[4] = {};
    double phase_us[3][64] = {};
    // the block-step loop on the device (g6_hermite_loop.cuh): env G6_HD_LOOP = 0 switches it off (one host wait per block step
    // instead), env G6_HD_LOOP_MAXI = largest block stepped inside the loop (default HD_LOOP_MAXI_DEFAULT, at most HL_MAX_I)
    bool loop = false;
    int loop_max_i = 0, loop_G = 0, loop_K = 0;
    unsigned long long *rec = nullptr, *chunk = nullptr;       // the loop kernel's exchange words (tile records, partial forces)
    unsigned int *flag = nullptr;
    unsigned int loop_gen = 0;                                 // step numbers handed out so far
    HlStatus *h_status = nullptr, *hd_status = nullptr;        // mapped host memory and its device view
    long long loop_launches = 0, loop_steps = 0;
    double loop_us[64] = {}, big_us[64] = {}, relaunch_us = 0;    // env G6_HD_LOOP_PROFILE: where the time of a run goes, by block size
    long long big_n[64] = {};
    long long inline_steps = 0;


    bool loop_profile = false, loop_marks = false;
    unsigned long long *prof = nullptr;     // [32] the marked build's summed intervals (device)
};

constexpr int HD_LOOP_MAXI_DEFAULT = HL_MAX_I;

namespace {

void hd_free(g6hd_system *s)
{
    if (!s) return;
    cudaFree(s->S.x); cudaFree(s->S.v); cudaFree(s->S.a); cudaFree(s->S.ad); cudaFree(s->S.m); cudaFree(s->S.t); cudaFree(s->S.dt);
    cudaFree(s->B.act); cudaFree(s->B.cand); cudaFree(s->B.xi); cudaFree(s->B.vi); cudaFree(s->B.bmin); cudaFree(s->B.bcnt); cudaFree(s->B.boff); cudaFree(s->B.ticket);
    cudaFree(s->B.d_ni); cudaFree(s->B.d_tnext);
    cudaFree(s->a1); cudaFree(s->ad1); cudaFree(s->pot); cudaFree(s->dt_min_bits); cudaFree(s->shared_bits);
    cudaFree(s->rec); cudaFree(s->chunk); cudaFree(s->flag); cudaFree(s->prof);
    if (s->h_status) cudaFreeHost(s->h_status);
    if (s->h_note) cudaFreeHost(s->h_note);
    for (auto &e : s->pe) if (e) cudaEventDestroy(e);
    delete s;
}

// force on the device-resident i-block (act, xi, vi)[0, ni) at time tn -> a1, ad1, pot; chunks of g6_npipes()
int hd_force(Cluster &c, g6hd_system &s, int ni, double tn)
{
    c.ti = tn;
    init_npipes();
    for (int i0 = 0; i0 < ni; i0 += g_npipes) {
        const int cnt = std::min(g_npipes, ni - i0);
        int rc = run_force(c, s.n, cnt, s.B.act + i0, s.B.xi + 3 * (size_t)i0, s.B.vi + 3 * (size_t)i0, s.eps2, s.a1 + 3 * (size_t)i0,
                           s.ad1 + 3 * (size_t)i0, s.pot + i0, nullptr, nullptr, nullptr, nullptr, nullptr);
        if (rc) return rc;
    }
    return G6_OK;
}

// Wait for the notification of launch `seq` (hd_notify): spin on the mapped record -- a few microseconds sooner than an
// event wait -- and look at the stream now and then so that a failed launch cannot hang the host.
int hd_wait_note(Cluster &c, g6hd_system &s, unsigned int seq, int &ni, double &tn)
{
    volatile HdNote *h = s.h_note;
    for (unsigned long long spins = 1;; ++spins) {
        if (h->seq == seq) break;
        if ((spins & 0x3fff) == 0) {
            const cudaError_t q = cudaStreamQuery(c.stream);
            if (q == cudaSuccess) {
                if (h->seq == seq) break;
                return fail(c, G6_ERR_CUDA, "block selection finished without its notification (seq %u)", seq);
            }
            if (q != cudaErrorNotReady) return fail(c, G6_ERR_CUDA, "block selection failed: %s", cudaGetErrorString(q));
        }
    }
    std::atomic_thread_fence(std::memory_order_acquire);
    ni = h->ni;
    tn = h->tnext;
    return G6_OK;
}

HdCorr hd_corr(const Cluster &c, const g6hd_system &s) { return HdCorr{s.a1, s.ad1, s.eta, s.dt_max, c.js.raw, s.dt_min_bits}; }

// run the corrector of the last block step now (it normally rides in the next k_hd_select)
int hd_finish(Cluster &c, g6hd_system &s)
{
    if (!s.pending) return G6_OK;
    k_hd_correct<<<(s.last_ni + HD_THREADS - 1) / HD_THREADS, HD_THREADS, 0, c.stream>>>(s.S, s.B, hd_corr(c, s));
    CK(cudaGetLastError());
    c.pred_valid = false;
    s.pending = false;
    return G6_OK;
}

// One launch of the device-side step loop: block steps until t_end, `max_steps` (> 0) or a block larger than loop_max_i.
// Returns with the stream drained and *st filled in.
int hd_loop_run(Cluster &c, g6hd_system &s, double t_end, long long max_steps, HlStatus *st)
{
    int rc = hd_finish(c, s);                       // the corrector of a block the host stepped
    if (rc) return rc;
    const int ntiles = (s.n + JT - 1) / JT;
    HlArgs A{};
    A.S = s.S; A.B = s.B; A.C = hd_corr(c, s);
    A.a1 = s.a1; A.ad1 = s.ad1; A.pot = s.pot;
    A.ntiles = ntiles; A.nj = s.n;
    A.t_sys = s.t; A.t_end = t_end; A.max_steps = max_steps; A.max_i = s.loop_max_i;
    A.eps2 = (float)s.eps2; A.ds = c.opt_ds;
    A.gen0 = s.loop_gen;
    A.rec = s.rec; A.chunk = s.chunk; A.flag = s.flag; A.status = s.hd_status; A.prof = s.prof;


    void *args[] = {(void *)&A};
    const void *fn = s.loop_marks ? (c.opt_newton ? (const void *)k_hd_loop<true, true> : (const void *)k_hd_loop<false, true>)
                                    : (c.opt_newton ? (const void *)k_hd_loop<true> : (const void *)k_hd_loop<false>);
    CK(cudaLaunchCooperativeKernel(fn, dim3(s.loop_G), dim3(HL_THREADS), args, sizeof(HlSmem), c.stream));
    CK(cudaStreamSynchronize(c.stream));
    *st = *s.h_status;
    s.loop_gen += (unsigned int)st->steps + 2u;     // step numbers are never reused (a handed-over block consumed one too)
    c.pred_valid = false;                           // the loop rewrote j-store records
    ++s.loop_launches;
    s.loop_steps += st->steps;
    return G6_OK;
}

}  // namespace

extern "C" {

g6hd_system *g6hd_create(int clusterid, int n, const double x[][3], const double v[][3], const double m[],
                         double eps2, double eta, double eta_start, double dt_max)
{
    if (clusterid < 0 || clusterid >= MAX_CLUSTERS) return nullptr;
    Cluster &c = g_cl[clusterid];
    if (!c.open) { fail(c, G6_ERR_NOT_OPEN, "cluster %d is not open", clusterid); return nullptr; }
    // k_hd_select keeps one entry per 1024-particle thread block in shared memory: HD_MAX_BLOCKS of them
    if (n < 1 || n > c.capacity || n > HD_MAX_BLOCKS * HD_PER_BLOCK || !x || !v || !m || !(eta > 0) || !(dt_max > 0) || !(eps2 >= 0) || c.pending) {
        fail(c, G6_ERR_ARG, "bad g6hd_create arguments (n = %d; capacity %d, device-resident driver limit %d)", n, c.capacity, HD_MAX_BLOCKS * HD_PER_BLOCK);
        return nullptr;
    }
    if (ensure_capacity(c, n) != G6_OK) return nullptr;
    g6hd_system *s = new (std::nothrow) g6hd_system;
    if (!s) return nullptr;
    s->cl = clusterid; s->n = n; s->eps2 = eps2; s->eta = eta; s->dt_max = dt_max;
    s->S.n = n;
    const size_t n3 = 3 * (size_t)n;
    const int nb = (n + HD_PER_BLOCK - 1) / HD_PER_BLOCK;
    int rc = [&]() -> int {
        CK(dalloc(s->S.x, n3)); CK(dalloc(s->S.v, n3)); CK(dalloc(s->S.a, n3)); CK(dalloc(s->S.ad, n3));
        CK(dalloc(s->S.m, n)); CK(dalloc(s->S.t, n)); CK(dalloc(s->S.dt, n));
        CK(dalloc(s->B.act, n)); CK(dalloc(s->B.cand, (size_t)nb * HD_PER_BLOCK)); CK(dalloc(s->B.xi, n3)); CK(dalloc(s->B.vi, n3));
        CK(dalloc(s->B.bmin, nb)); CK(dalloc(s->B.bcnt, nb)); CK(dalloc(s->B.boff, nb)); CK(dalloc(s->B.ticket, 1)); CK(dalloc(s->B.d_ni, 1)); CK(dalloc(s->B.d_tnext, 1));
        CK(dalloc(s->a1, n3)); CK(dalloc(s->ad1, n3)); CK(dalloc(s->pot, n)); CK(dalloc(s->dt_min_bits, 1)); CK(dalloc(s->shared_bits, 1));
        CK(cudaHostAlloc((void **)&s->h_note, sizeof(HdNote), cudaHostAllocMapped));
        memset(s->h_note, 0, sizeof(HdNote));
        CK(cudaHostGetDevicePointer((void **)&s->B.h_note, s->h_note, 0));
        // the device-side step loop: CTA c owns the j-tiles c, c + G, ... (at most HL_KMAX of them, resident in shared memory)
        {
            const int ntiles = (n + JT - 1) / JT;
            const int K = (ntiles + std::min(c.n_sm, HL_MAX_G) - 1) / std::min(c.n_sm, HL_MAX_G);
            s->loop_K = K;
            s->loop_G = (ntiles + K - 1) / K;
            s->loop_max_i = std::max(1, std::min(env_int("G6_HD_LOOP_MAXI", HD_LOOP_MAXI_DEFAULT), HL_MAX_I));
            s->loop = env_int("G6_HD_LOOP", 1) != 0 && K <= HL_KMAX;
            if (s->loop) {
                CK(cudaFuncSetAttribute(k_hd_loop<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(HlSmem)));
                CK(cudaFuncSetAttribute(k_hd_loop<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(HlSmem)));
                CK(cudaFuncSetAttribute(k_hd_loop<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(HlSmem)));
                CK(cudaFuncSetAttribute(k_hd_loop<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(HlSmem)));
                const size_t nrec = 2 * (size_t)s->loop_G * ntiles * HL_REC_WORDS, nchunk = (size_t)s->loop_max_i * HL_CHUNK_WORDS * s->loop_G;
                CK(dalloc(s->rec, nrec)); CK(dalloc(s->chunk, nchunk)); CK(dalloc(s->flag, s->loop_G)); CK(dalloc(s->prof, 32));
                CK(cudaMemset(s->prof, 0, 32 * sizeof(unsigned long long)));
                CK(cudaMemsetAsync(s->rec, 0, nrec * sizeof(unsigned long long), c.stream));           // step number 0 = never written
                CK(cudaMemsetAsync(s->chunk, 0, nchunk * sizeof(unsigned long long), c.stream));
                CK(cudaMemsetAsync(s->flag, 0, s->loop_G * sizeof(unsigned int), c.stream));
                CK(cudaHostAlloc((void **)&s->h_status, sizeof(HlStatus), cudaHostAllocMapped));
                memset(s->h_status, 0, sizeof(HlStatus));
                CK(cudaHostGetDevicePointer((void **)&s->hd_status, s->h_status, 0));
            }
        }
        s->loop_profile = env_int("G6_HD_LOOP_PROFILE", 0) != 0;      // 1: the build with phase marks; 2: the production loop, per-bin times only
        s->loop_marks = env_int("G6_HD_LOOP_PROFILE", 0) == 1;
        s->profile = env_int("G6_HD_PROFILE", 0) != 0;
        if (s->profile) for (auto &e : s->pe) CK(cudaEventCreate(&e));
        CK(cudaMemsetAsync(s->B.ticket, 0, sizeof(unsigned int), c.stream));
        const unsigned long long big = 0x7ff0000000000000ULL;
        CK(cudaMemcpyAsync(s->dt_min_bits, &big, sizeof(big), cudaMemcpyHostToDevice, c.stream));
        CK(cudaMemcpyAsync(s->S.x, x, n3 * sizeof(double), cudaMemcpyHostToDevice, c.stream));
        CK(cudaMemcpyAsync(s->S.v, v, n3 * sizeof(double), cudaMemcpyHostToDevice, c.stream));
        CK(cudaMemcpyAsync(s->S.m, m, n * sizeof(double), cudaMemcpyHostToDevice, c.stream));
        CK(cudaMemsetAsync(s->S.a, 0, n3 * sizeof(double), c.stream));
        CK(cudaMemsetAsync(s->S.ad, 0, n3 * sizeof(double), c.stream));
        CK(cudaMemsetAsync(s->S.t, 0, n * sizeof(double), c.stream));
        CK(cudaMemsetAsync(s->S.dt, 0, n * sizeof(double), c.stream));
        CK(cudaStreamSynchronize(c.stream));           // the caller's arrays may be pageable
        // t = 0: every particle is its own i-particle; a = adot = 0 makes the prediction the identity
        int r = flush_j(c);
        if (r) return r;
        k_hd_init<<<(n + HD_THREADS - 1) / HD_THREADS, HD_THREADS, 0, c.stream>>>(s->S, s->S.a, s->S.ad, eta_start, dt_max, c.js.raw, s->dt_min_bits);
        CK(cudaGetLastError());                        // loads the j-store (the steps it sets are overwritten below)
        c.n_stored = std::max(c.n_stored, n);
        c.pred_valid = false;
        k_hd_predict_all<<<(n + HD_THREADS - 1) / HD_THREADS, HD_THREADS, 0, c.stream>>>(s->S, 0.0, s->B.xi, s->B.vi);
        CK(cudaGetLastError());
        k_hd_iota<<<(n + HD_THREADS - 1) / HD_THREADS, HD_THREADS, 0, c.stream>>>(s->B.act, n);      // the first block is everybody
        CK(cudaGetLastError());
        r = hd_force(c, *s, n, 0.0);
        if (r) return r;
        CK(cudaMemcpyAsync(s->dt_min_bits, &big, sizeof(big), cudaMemcpyHostToDevice, c.stream));
        k_hd_init<<<(n + HD_THREADS - 1) / HD_THREADS, HD_THREADS, 0, c.stream>>>(s->S, s->a1, s->ad1, eta_start, dt_max, c.js.raw, s->dt_min_bits);
        CK(cudaGetLastError());
        c.pred_valid = false;
        CK(cudaStreamSynchronize(c.stream));
        return G6_OK;
    }();
    if (rc != G6_OK) { hd_free(s); return nullptr; }
    return s;
}

void g6hd_destroy(g6hd_system *s)
{
    if (s && s->cl >= 0 && s->cl < MAX_CLUSTERS && g_cl[s->cl].open) cudaStreamSynchronize(g_cl[s->cl].stream);
    hd_free(s);
}

int g6hd_evolve(g6hd_system *sp, double t_end, long long max_block_steps)
{
    if (!sp) return G6_ERR_ARG;
    g6hd_system &s = *sp;
    GET_CLUSTER(s.cl);
    if (c.pending) return fail(c, G6_ERR_SEQUENCE, "force call pending");
    const auto w0 = std::chrono::steady_clock::now();
    const int nb = (s.n + HD_PER_BLOCK - 1) / HD_PER_BLOCK;
    long long done = 0;
    while (s.shared && s.t < t_end && (max_block_steps <= 0 || done < max_block_steps)) {
        // shared steps: corrector of the previous step for everybody, common step = smallest wish, everybody predicted
        int rcf = hd_finish(c, s);
        if (rcf) return rcf;
        const int g = (s.n + HD_THREADS - 1) / HD_THREADS;
        k_hd_set_u64<<<1, 1, 0, c.stream>>>(s.shared_bits, 0x7ff0000000000000ULL);
        k_hd_min_dt<<<g, HD_THREADS, 0, c.stream>>>(s.S, s.shared_bits);
        s.B.seq = ++s.seq;
        k_hd_shared_apply<<<g, HD_THREADS, 0, c.stream>>>(s.S, s.B, s.shared_bits);
        CK(cudaGetLastError());
        int nall = 0;
        double tn = 0;
        int rcw = hd_wait_note(c, s, s.B.seq, nall, tn);
        if (rcw) return rcw;
        if (!(tn > s.t) || nall != s.n) return fail(c, G6_ERR_CUDA, "shared step returned n = %d, t = %g", nall, tn);
        int rc = hd_force(c, s, s.n, tn);
        if (rc) return rc;
        s.pending = true;
        s.t = tn;
        s.last_ni = s.n;
        ++s.nblock; ++done;
        s.npart += s.n;
        s.inter += (double)s.n * (double)s.n;
        int b = 0;
        while ((1LL << (b + 1)) <= s.n) ++b;
        s.hist[b] += 1;
    }
    const auto count_block = [&](int ni) {
        ++s.nblock; ++done;
        s.npart += ni;
        s.inter += (double)ni * (double)s.n;
        int b = 0;
        while ((1LL << (b + 1)) <= ni) ++b;
        s.hist[b] += 1;
    };
    // block steps, the loop on the device: one launch steps until t_end, the step budget, or a block too large for it;
    // such a block comes back selected and predicted, the library's sweep path computes its forces, and the loop resumes
    while (!s.shared && s.loop && !s.profile && s.t < t_end && (max_block_steps <= 0 || done < max_block_steps)) {
        HlStatus st;
        int rc = hd_loop_run(c, s, t_end, max_block_steps > 0 ? max_block_steps - done : 0, &st);
        if (rc) return rc;
        if (st.steps > 0) {
            s.t = st.t;
            s.last_ni = st.ni_last;
            s.nblock += st.steps; done += st.steps;
            s.npart += st.npart;
            s.inter += (double)st.npart * (double)s.n;
            for (int b = 0; b < 64; ++b) { s.hist[b] += st.hist[b]; s.loop_us[b] += 1e-3 * (double)st.ns[b]; }
            s.inline_steps += st.inline_steps;
        }
        if (st.reason != HL_BIG) {
            if (st.reason == HL_END || st.reason == HL_STEPS) continue;        // the loop condition ends it
            return fail(c, G6_ERR_CUDA, "device step loop returned reason %d", st.reason);
        }
        const int ni = st.ni_next;
        const double tn = st.tnext;
        if (ni < 1 || ni > s.n || !(tn > s.t)) return fail(c, G6_ERR_CUDA, "device step loop handed over ni = %d, t = %g", ni, tn);
        const auto b0 = std::chrono::steady_clock::now();
        rc = hd_force(c, s, ni, tn);
        if (rc) return rc;
        s.pending = true;                               // its corrector runs before the loop resumes (hd_finish)
        s.t = tn;
        s.last_ni = ni;
        count_block(ni);
        if (s.loop_profile) {
            CK(cudaStreamSynchronize(c.stream));
            int b = 0;
            while ((1LL << (b + 1)) <= ni) ++b;
            s.big_us[b] += 1e6 * std::chrono::duration<double>(std::chrono::steady_clock::now() - b0).count();
            s.big_n[b] += 1;
        }
    }
    while (!s.shared && s.t < t_end && (max_block_steps <= 0 || done < max_block_steps)) {
        if (s.profile) CK(cudaEventRecord(s.pe[0], c.stream));
        s.B.seq = ++s.seq;
        k_hd_select<<<nb, HD_THREADS, 0, c.stream>>>(s.S, s.B, hd_corr(c, s), s.pending ? 1 : 0);
        CK(cudaGetLastError());
        c.pred_valid = false;                           // phase 0 rewrote j-store records
        s.pending = false;
        if (s.profile) CK(cudaEventRecord(s.pe[1], c.stream));
        int ni = 0;
        double tn = 0;
        {
            int rcw = hd_wait_note(c, s, s.B.seq, ni, tn);      // the one host wait of the block step
            if (rcw) return rcw;
        }
        if (ni < 1 || ni > s.n || !(tn > s.t)) return fail(c, G6_ERR_CUDA, "block selection returned ni = %d, t = %g", ni, tn);
        if (ni > HD_GATHER_INLINE) {
            k_hd_gather<<<nb, HD_THREADS, 0, c.stream>>>(s.S, s.B);
            CK(cudaGetLastError());
        }
        int rc = hd_force(c, s, ni, tn);
        if (rc) return rc;
        s.pending = true;                               // its corrector is phase 0 of the next k_hd_select
        if (s.profile) {
            CK(cudaEventRecord(s.pe[2], c.stream));
            CK(cudaEventRecord(s.pe[3], c.stream));
            CK(cudaEventSynchronize(s.pe[3]));
            int bb = 0;
            while ((1LL << (bb + 1)) <= ni) ++bb;
            for (int q = 0; q < 3; ++q) {
                float ms = 0;
                CK(cudaEventElapsedTime(&ms, s.pe[q], s.pe[q + 1]));
                s.phase_us[q][bb] += 1e3 * ms;
            }
        }
        s.t = tn;
        s.last_ni = ni;
        ++s.nblock; ++done;
        s.npart += ni;
        s.inter += (double)ni * (double)s.n;
        int b = 0;
        while ((1LL << (b + 1)) <= ni) ++b;
        s.hist[b] += 1;
    }
    {
        int rcf = hd_finish(c, s);
        if (rcf) return rcf;
    }
    CK(cudaStreamSynchronize(c.stream));
    s.wall += std::chrono::duration<double>(std::chrono::steady_clock::now() - w0).count();
    return G6_OK;
}

int g6hd_set_shared_steps(g6hd_system *sp, int on)
{
    if (!sp) return G6_ERR_ARG;
    g6hd_system &s = *sp;
    GET_CLUSTER(s.cl);
    int rc = hd_finish(c, s);           // (never pending between calls; kept for safety)
    if (rc) return rc;
    if (on && !s.shared) {
        // the shared scheme predicts everybody from ONE time and gives everybody ONE new time: all particles must be at the
        // system time now (true at multiples of dt_max; not after a stop on max_block_steps or at another t_end)
        unsigned long long off = 0;
        k_hd_set_u64<<<1, 1, 0, c.stream>>>(s.shared_bits, 0ULL);
        k_hd_count_unsynchronised<<<(s.n + HD_THREADS - 1) / HD_THREADS, HD_THREADS, 0, c.stream>>>(s.S, s.t, s.shared_bits);
        CK(cudaGetLastError());
        CK(cudaMemcpyAsync(&off, s.shared_bits, sizeof(off), cudaMemcpyDeviceToHost, c.stream));
        CK(cudaStreamSynchronize(c.stream));
        if (off) return fail(c, G6_ERR_SEQUENCE, "shared time steps need all particles at the system time t = %g; %llu are not "
                             "(evolve to a multiple of dt_max first)", s.t, off);
    }
    s.shared = on != 0;
    return G6_OK;
}

int g6hd_get_state(g6hd_system *sp, double x[][3], double v[][3])
{
    if (!sp || !x || !v) return G6_ERR_ARG;
    g6hd_system &s = *sp;
    GET_CLUSTER(s.cl);
    // B.xi / B.vi are free between block steps
    k_hd_predict_all<<<(s.n + HD_THREADS - 1) / HD_THREADS, HD_THREADS, 0, c.stream>>>(s.S, s.t, s.B.xi, s.B.vi);
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(x, s.B.xi, 3 * (size_t)s.n * sizeof(double), cudaMemcpyDeviceToHost, c.stream));
    CK(cudaMemcpyAsync(v, s.B.vi, 3 * (size_t)s.n * sizeof(double), cudaMemcpyDeviceToHost, c.stream));
    CK(cudaStreamSynchronize(c.stream));
    return G6_OK;
}

int g6hd_get_particles(g6hd_system *sp, double x[][3], double v[][3], double a[][3], double adot[][3], double t[], double dt[])
{
    if (!sp) return G6_ERR_ARG;
    g6hd_system &s = *sp;
    GET_CLUSTER(s.cl);
    const size_t b3 = 3 * (size_t)s.n * sizeof(double), b1 = (size_t)s.n * sizeof(double);
    CK(cudaStreamSynchronize(c.stream));
    if (x) CK(cudaMemcpy(x, s.S.x, b3, cudaMemcpyDeviceToHost));
    if (v) CK(cudaMemcpy(v, s.S.v, b3, cudaMemcpyDeviceToHost));
    if (a) CK(cudaMemcpy(a, s.S.a, b3, cudaMemcpyDeviceToHost));
    if (adot) CK(cudaMemcpy(adot, s.S.ad, b3, cudaMemcpyDeviceToHost));
    if (t) CK(cudaMemcpy(t, s.S.t, b1, cudaMemcpyDeviceToHost));
    if (dt) CK(cudaMemcpy(dt, s.S.dt, b1, cudaMemcpyDeviceToHost));
    return G6_OK;
}

int g6hd_get_last_block(g6hd_system *sp, int maxn, int *ni, int act[], double xi[][3], double vi[][3], double acc[][3], double jerk[][3])
{
    if (!sp || !ni) return G6_ERR_ARG;
    g6hd_system &s = *sp;
    GET_CLUSTER(s.cl);
    *ni = s.last_ni;
    if (s.last_ni > maxn) return fail(c, G6_ERR_ARG, "last block has %d particles, buffer holds %d", s.last_ni, maxn);
    const size_t b3 = 3 * (size_t)s.last_ni * sizeof(double);
    CK(cudaStreamSynchronize(c.stream));
    if (act) CK(cudaMemcpy(act, s.B.act, s.last_ni * sizeof(int), cudaMemcpyDeviceToHost));
    if (xi) CK(cudaMemcpy(xi, s.B.xi, b3, cudaMemcpyDeviceToHost));
    if (vi) CK(cudaMemcpy(vi, s.B.vi, b3, cudaMemcpyDeviceToHost));
    if (acc) CK(cudaMemcpy(acc, s.a1, b3, cudaMemcpyDeviceToHost));
    if (jerk) CK(cudaMemcpy(jerk, s.ad1, b3, cudaMemcpyDeviceToHost));
    return G6_OK;
}

int g6hd_get_stats(g6hd_system *sp, double stats[8], long long ni_hist_log2[64])
{
    if (!sp || !stats) return G6_ERR_ARG;
    g6hd_system &s = *sp;
    GET_CLUSTER(s.cl);
    unsigned long long bits = 0;
    CK(cudaStreamSynchronize(c.stream));
    CK(cudaMemcpy(&bits, s.dt_min_bits, sizeof(bits), cudaMemcpyDeviceToHost));
    double dmin;
    memcpy(&dmin, &bits, sizeof(dmin));
    stats[0] = (double)s.nblock; stats[1] = (double)s.npart; stats[2] = s.t; stats[3] = dmin;
    stats[4] = s.inter; stats[5] = s.wall; stats[6] = 0; stats[7] = 0;
    if (s.profile)
        for (int b = 0; b < 64; ++b)
            if (s.hist[b])
                fprintf(stderr, "g6hd profile: n_i in [2^%d, 2^%d): %lld block steps, select %.1f us, force (from the host wait to its last kernel) %.1f us, correct %.1f us per step\n",
                        b, b + 1, s.hist[b], s.phase_us[0][b] / s.hist[b], s.phase_us[1][b] / s.hist[b], s.phase_us[2][b] / s.hist[b]);
    if (s.loop_profile) {
        fprintf(stderr, "g6hd loop profile: %lld launches of the step loop, %lld block steps inside it\n", s.loop_launches, s.loop_steps);
        fprintf(stderr, "  %lld of them predicted their i-block in every CTA (one exchange less)\n", s.inline_steps);
        if (s.loop_marks && s.prof) {
            unsigned long long pr[32];
            CK(cudaMemcpy(pr, s.prof, sizeof(pr), cudaMemcpyDeviceToHost));
            if (pr[15]) {
                const double n = (double)pr[15];
                fprintf(stderr, "  steps with n_i < 8 as CTA 0 walks them, SM cycles per step: publish %.0f | poll: own lane %.0f, all lanes %.0f | select %.0f | barrier %.0f | predict i, j %.0f | "
                        "pairs + shuffle tree %.0f | barrier %.0f | slice sums + partials out %.0f | gather + correct (if owner) %.0f\n",
                        pr[0] / n, pr[1] / n, pr[2] / n, pr[3] / n, pr[4] / n, pr[5] / n, pr[6] / n, pr[7] / n, pr[8] / n, pr[9] / n);
                fprintf(stderr, "    select in parts: counts per lane %.0f | scan over the lanes %.0f | offsets and active list %.0f | own list %.0f\n", pr[11] / n, pr[12] / n, pr[13] / n, pr[14] / n);
            }
            if (pr[31]) {
                const double n = (double)pr[31];
                fprintf(stderr, "  the CTAs that own an active particle of such a step (<= %d of them): gather poll %.0f | barrier %.0f | sum of the %d partials %.0f | corrector %.0f | "
                        "barrier + stores + release fence (an idle warp rescans the tile meanwhile) %.0f | closing barrier %.0f | to the top of the next step %.0f | publish %.0f\n",
                        HL_CQ, pr[16] / n, pr[17] / n, s.loop_G, pr[18] / n, pr[19] / n, pr[20] / n, pr[21] / n, (pr[22] + pr[23]) / n, pr[24] / n);
            }
        }
        for (int b = 0; b < 64; ++b)
            if (s.hist[b])
                fprintf(stderr, "  n_i in [2^%d, 2^%d): %lld block steps; in the loop %.1f us per step (device clock, %lld steps); handed to the host %lld steps, %.1f us each (wall, force only)\n",
                        b, b + 1, s.hist[b], (s.hist[b] - s.big_n[b]) ? s.loop_us[b] / (double)(s.hist[b] - s.big_n[b]) : 0.0, s.hist[b] - s.big_n[b],
                        s.big_n[b], s.big_n[b] ? s.big_us[b] / (double)s.big_n[b] : 0.0);
    }
    if (ni_hist_log2) memcpy(ni_hist_log2, s.hist, sizeof(s.hist));
    return G6_OK;
}

}  // extern "C"
