// g6_hermite.cpp -- host fp64 Hermite block-step driver on top of the g6_* C ABI (include/g6_hermite.h).
// Step a-7 of the path: O(n_i log N) host work per block step; all O(n_i N) work is in the library.
#include "../../include/g6_hermite.h"
#include "../../include/g6.h"

#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <utility>
#include <vector>

namespace {
constexpr int LEVELS = 1100;             // dt = 2^-k, k up to the smallest normal double
struct V3 { double c[3]; };
inline double norm(const V3 &a) { return std::sqrt(a.c[0] * a.c[0] + a.c[1] * a.c[1] + a.c[2] * a.c[2]); }
using Clock = std::chrono::steady_clock;
inline double secs(Clock::time_point a, Clock::time_point b) { return std::chrono::duration<double>(b - a).count(); }
}  // namespace

struct g6h_system {
    int cl = 0, n = 0;
    double eps2 = 0, eta = 0, dt_max = 0, t = 0, dt_min = 0;
    std::vector<V3> x, v, a, ad;     // state at each particle's own time
    std::vector<double> m, tp, dt;
    // Block scheduling in O(1) per particle step.  Steps are dt_max halved k times and a particle's time is always a
    // multiple of its step, so ALL particles of level k (dt = dt_max 2^-k) are due at every multiple of that step: the next
    // block time is t + (smallest step in use), and the block is the union of the levels whose step divides it.
    std::vector<int> lev[LEVELS];        // members of every level
    std::vector<int> pos, lvl;           // position in its level's list, level of every particle
    // per-block scratch
    std::vector<int> act;
    std::vector<V3> xi, vi, a1, ad1;
    std::vector<double> pot;
    long long nblock = 0, npart = 0, hist[64] = {};
    double inter = 0, wall = 0, wall_force = 0, wall_force_hist[64] = {};
    double wall_predict = 0, wall_correct = 0;       // where the host's own time goes (printed with env G6H_PROFILE)
};

namespace {

// Eq. 1-2 for one particle on the host ("The prediction of the i-particles is
// similarly implemented on the CPU")
inline void predict_one(const g6h_system &s, int p, double tn, V3 &xp, V3 &vp)
{
    const double h = tn - s.tp[p], h2 = h * h / 2, h3 = h * h * h / 6;
    for (int k = 0; k < 3; ++k) {
        xp.c[k] = s.x[p].c[k] + s.v[p].c[k] * h + s.a[p].c[k] * h2 + s.ad[p].c[k] * h3;
        vp.c[k] = s.v[p].c[k] + s.a[p].c[k] * h + s.ad[p].c[k] * h2;
    }
}

int send_j(const g6h_system &s, int p)
{
    double a2[3], j6[3];
    for (int k = 0; k < 3; ++k) { a2[k] = s.a[p].c[k] / 2; j6[k] = s.ad[p].c[k] / 6; }
    return g6_set_j_particle(s.cl, p, p, s.tp[p], s.dt[p], s.m[p], nullptr, j6, a2, s.v[p].c, s.x[p].c);
}

// forces on the block s.act (already predicted into s.xi, s.vi) -> s.a1, s.ad1, s.pot
int block_force(g6h_system &s, double tn)
{
    const int ni = (int)s.act.size(), np = g6_npipes();
    int rc = g6_set_ti(s.cl, tn);
    for (int i0 = 0; rc == 0 && i0 < ni; i0 += np) {
        const int c = std::min(np, ni - i0);
        rc = g6calc_firsthalf(s.cl, s.n, c, &s.act[i0], (const double(*)[3]) & s.xi[i0], (const double(*)[3]) & s.vi[i0],
                              nullptr, nullptr, nullptr, s.eps2, nullptr);
        if (rc) break;
        rc = g6calc_lasthalf(s.cl, s.n, c, &s.act[i0], (const double(*)[3]) & s.xi[i0], (const double(*)[3]) & s.vi[i0],
                             s.eps2, nullptr, (double(*)[3]) & s.a1[i0], (double(*)[3]) & s.ad1[i0], &s.pot[i0]);
    }
    return rc;
}

// k of dt = dt_max 2^-k (every step is dt_max halved k times)
inline int level_of(const g6h_system &s, double dt)
{
    int e;
    std::frexp(s.dt_max / dt, &e);       // the ratio is 2^k = 0.5 * 2^(k+1), exactly
    return e - 1;
}
inline double level_step(const g6h_system &s, int k) { return std::ldexp(s.dt_max, -k); }

void level_insert(g6h_system &s, int p, double dt)
{
    const int k = level_of(s, dt);
    s.lvl[p] = k;
    s.pos[p] = (int)s.lev[k].size();
    s.lev[k].push_back(p);
}

void level_move(g6h_system &s, int p, double dt)
{
    const int k = level_of(s, dt);
    if (k == s.lvl[p]) return;
    std::vector<int> &old = s.lev[s.lvl[p]];
    const int last = old.back();
    old[s.pos[p]] = last;                // swap-remove
    s.pos[last] = s.pos[p];
    old.pop_back();
    level_insert(s, p, dt);
}

double pow2_floor(double want, double cap)
{
    double d = cap;
    while (d > want && d > 1e-300) d *= 0.5;
    return d;
}

}  // namespace

extern "C" {

g6h_system *g6h_create(int clusterid, int n, const double x[][3], const double v[][3], const double m[],
                       double eps2, double eta, double eta_start, double dt_max)
{
    if (n < 1 || !x || !v || !m || !(eta > 0) || !(dt_max > 0)) return nullptr;
    g6h_system *s = new (std::nothrow) g6h_system;
    if (!s) return nullptr;
    try {
        s->cl = clusterid; s->n = n; s->eps2 = eps2; s->eta = eta; s->dt_max = dt_max; s->dt_min = dt_max;
        s->x.resize(n); s->v.resize(n); s->a.assign(n, V3{{0, 0, 0}}); s->ad.assign(n, V3{{0, 0, 0}});
        s->m.assign(m, m + n); s->tp.assign(n, 0.0); s->dt.assign(n, dt_max);
        s->pos.assign(n, 0); s->lvl.assign(n, 0);
        s->act.resize(n); s->xi.resize(n); s->vi.resize(n); s->a1.resize(n); s->ad1.resize(n); s->pot.resize(n);
    } catch (const std::bad_alloc &) { delete s; return nullptr; }
    std::memcpy(s->x.data(), x, sizeof(V3) * n);
    std::memcpy(s->v.data(), v, sizeof(V3) * n);
    // initial load (acc = jerk = 0 at t = 0: prediction to t = 0 is the identity), then a full sweep
    int rc = 0;
    for (int p = 0; rc == 0 && p < n; ++p) rc = send_j(*s, p);
    for (int p = 0; p < n; ++p) { s->act[p] = p; s->xi[p] = s->x[p]; s->vi[p] = s->v[p]; }
    if (rc == 0) rc = block_force(*s, 0.0);
    if (rc != 0) { delete s; return nullptr; }
    for (int p = 0; p < n; ++p) {
        s->a[p] = s->a1[p];
        s->ad[p] = s->ad1[p];
        const double na = norm(s->a[p]), nad = norm(s->ad[p]);
        s->dt[p] = pow2_floor(nad > 0 ? eta_start * na / nad : dt_max, dt_max);
        if (s->dt[p] < s->dt_min) s->dt_min = s->dt[p];
        if (level_of(*s, s->dt[p]) < 0 || level_of(*s, s->dt[p]) >= LEVELS) { delete s; return nullptr; }
        level_insert(*s, p, s->dt[p]);
    }
    for (int p = 0; rc == 0 && p < n; ++p) rc = send_j(*s, p);
    if (rc != 0) { delete s; return nullptr; }
    s->act.clear();
    return s;
}

void g6h_destroy(g6h_system *s) { delete s; }

static int evolve_body(g6h_system &s, double t_end, long long max_block_steps);

int g6h_evolve(g6h_system *sp, double t_end, long long max_block_steps)
{
    if (!sp) return G6_ERR_ARG;
    try {
        return evolve_body(*sp, t_end, max_block_steps);      // no C++ exception crosses the boundary (level lists grow)
    } catch (const std::bad_alloc &) {
        return G6_ERR_NOMEM;
    } catch (...) {
        return G6_ERR_ARG;
    }
}

static int evolve_body(g6h_system &s, double t_end, long long max_block_steps)
{
    const auto w0 = Clock::now();
    const double dt_floor = level_step(s, LEVELS - 1);      // the smallest step the level table holds
    long long done = 0;
    int rc = 0;
    while (s.t < t_end && (max_block_steps <= 0 || done < max_block_steps)) {
        int kmax = LEVELS - 1;
        while (kmax > 0 && s.lev[kmax].empty()) --kmax;                 // smallest step in use
        const double tn = s.t + level_step(s, kmax);
        s.act.clear();
        for (int k = kmax; k >= 0 && std::fmod(tn, level_step(s, k)) == 0.0; --k)
            s.act.insert(s.act.end(), s.lev[k].begin(), s.lev[k].end());
        const int ni = (int)s.act.size();
        const auto p0 = Clock::now();
        for (int k = 0; k < ni; ++k) predict_one(s, s.act[k], tn, s.xi[k], s.vi[k]);
        const auto f0 = Clock::now();
        s.wall_predict += secs(p0, f0);
        rc = block_force(s, tn);
        const double wf = secs(f0, Clock::now());
        s.wall_force += wf;
        if (rc) break;
        const auto c0 = Clock::now();
        for (int k = 0; k < ni; ++k) {
            const int p = s.act[k];
            const double h = s.dt[p], h2 = h * h, h3 = h2 * h, h4 = h3 * h, h5 = h4 * h;
            V3 a2n, a3;
            for (int c = 0; c < 3; ++c) {
                const double da = s.a[p].c[c] - s.a1[k].c[c];
                const double a2 = (-6 * da - h * (4 * s.ad[p].c[c] + 2 * s.ad1[k].c[c])) / h2;
                a3.c[c] = (12 * da + 6 * h * (s.ad[p].c[c] + s.ad1[k].c[c])) / h3;
                s.x[p].c[c] = s.xi[k].c[c] + h4 * a2 / 24 + h5 * a3.c[c] / 120;
                s.v[p].c[c] = s.vi[k].c[c] + h3 * a2 / 6 + h4 * a3.c[c] / 24;
                a2n.c[c] = a2 + h * a3.c[c];
            }
            s.a[p] = s.a1[k];
            s.ad[p] = s.ad1[k];
            s.tp[p] = tn;
            const double na = norm(s.a[p]), nad = norm(s.ad[p]), n2 = norm(a2n), n3 = norm(a3);
            const double den = nad * n3 + n2 * n2;
            const double want = den > 0 ? std::sqrt(s.eta * (na * n2 + nad * nad) / den) : s.dt_max;
            double d = h;
            if (want < d) {
                while (d > want && d > dt_floor) d *= 0.5;
                if (d > want) { rc = G6_ERR_ARG; break; }     // the step criterion asks for a step below 2^-1100 dt_max (want = 0 or NaN forces)
            } else if (want >= 2 * d && 2 * d <= s.dt_max && std::fmod(tn, 2 * d) == 0.0) {
                d *= 2;
            }
            s.dt[p] = d;
            if (d < s.dt_min) s.dt_min = d;
            level_move(s, p, d);
            rc = send_j(s, p);
            if (rc) break;
        }
        s.wall_correct += secs(c0, Clock::now());
        if (rc) break;
        s.t = tn;
        ++s.nblock; ++done;
        s.npart += ni;
        s.inter += (double)ni * (double)s.n;
        int b = 0;
        while ((1LL << (b + 1)) <= ni) ++b;
        s.hist[b] += 1;
        s.wall_force_hist[b] += wf;
    }
    s.wall += secs(w0, Clock::now());
    // (measured on C2: 3.4 s = force calls 2.3 + i-prediction 0.17 + corrector, level lists and g6_set_j_particle 0.87; computing the
    // corrector of large blocks on 8 threads and updating lists and j-particles afterwards was slower, 1.18 s: the scattered
    // particle state, not the arithmetic, is what costs)
    if (std::getenv("G6H_PROFILE"))
        std::fprintf(stderr, "g6h profile: wall %.3f s, force calls %.3f, i-prediction %.3f, corrector + level lists + g6_set_j_particle %.3f, block selection and the rest %.3f\n",
                     s.wall, s.wall_force, s.wall_predict, s.wall_correct, s.wall - s.wall_force - s.wall_predict - s.wall_correct);
    return rc;
}

int g6h_get_state(g6h_system *s, double x[][3], double v[][3])
{
    if (!s || !x || !v) return G6_ERR_ARG;
    for (int p = 0; p < s->n; ++p) {
        V3 xp, vp;
        predict_one(*s, p, s->t, xp, vp);
        std::memcpy(x[p], xp.c, sizeof(V3));
        std::memcpy(v[p], vp.c, sizeof(V3));
    }
    return 0;
}

int g6h_get_stats(g6h_system *s, double stats[8], long long ni_hist_log2[64])
{
    if (!s || !stats) return G6_ERR_ARG;
    stats[0] = (double)s->nblock; stats[1] = (double)s->npart; stats[2] = s->t; stats[3] = s->dt_min;
    stats[4] = s->inter; stats[5] = s->wall; stats[6] = s->wall_force; stats[7] = 0;
    if (ni_hist_log2) std::memcpy(ni_hist_log2, s->hist, sizeof(s->hist));
    return 0;
}

int g6h_get_force_wall_hist(g6h_system *s, double wall_s_log2[64])
{
    if (!s || !wall_s_log2) return G6_ERR_ARG;
    std::memcpy(wall_s_log2, s->wall_force_hist, sizeof(s->wall_force_hist));
    return 0;
}

}  // extern "C"
