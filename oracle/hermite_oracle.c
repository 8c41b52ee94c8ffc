/*
 * oracle/hermite_oracle.c -- CPU ORACLE of the host integrator.  TEST INFRASTRUCTURE ONLY.
 *
 * "standard 4th-order predictor-corrector Hermite integration scheme (Makino & Aarseth 1992)
 *  ... with block time steps" -- PAPER.md:31-33 (section 2); time-step criterion of Aarseth
 * 1985, accuracy parameter eta -- PAPER.md:156, :162.  The paper only cites these; the
 * formulas below are the textbook ones, SURVEY.md section 8(c) reading 16 / DESIGN.md:
 *
 *   predict (Eq. 1-2) every particle to the block time t;
 *   force on the active block {i : t_i + dt_i == t} from ALL predicted particles (orc_force);
 *   corrector, h = dt_i, (a0, adot0) old, (a1, adot1) new:
 *       a2 = [ -6 (a0 - a1) - h (4 adot0 + 2 adot1) ] / h^2
 *       a3 = [ 12 (a0 - a1) + 6 h (adot0 + adot1) ] / h^3
 *       x1 = x_p + h^4 a2 / 24 + h^5 a3 / 120 ,   v1 = v_p + h^3 a2 / 6 + h^4 a3 / 24
 *       a2' = a2 + h a3                                    (second derivative at the new time)
 *   step:  dt_want = sqrt( eta (|a1||a2'| + |adot1|^2) / (|adot1||a3| + |a2'|^2) )
 *       halve dt while dt > dt_want; double it (once) only if dt_want >= 2 dt, the new time is
 *       a multiple of 2 dt and 2 dt <= dt_max;
 *   start: dt = eta_start |a| / |adot| rounded down to a power of two, <= dt_max.
 *
 * orc_hermite_shared: the same with ONE step for all particles (reading 21), pinned by: identical to the block scheme
 * on a configuration whose particles all ask for the same step (rotating polygon), step counts, energy conservation.
 *
 * Plain fp64, one block step after the other, the whole system re-predicted every step.
 * Uses orc_force of g6_oracle.c for the forces (same oracle, same pins).  Pinned by
 * tests/test_oracle_pins.py: a circular binary returns to its start after one period, the
 * energy error falls as the 4th-order scheme predicts when eta shrinks, and all particles are
 * synchronised at multiples of dt_max.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

void orc_force(int ni, const int *index_i, const double (*xi)[3], const double (*vi)[3],
               int nj, const int *index_j, const double (*xj)[3], const double (*vj)[3],
               const double *mj, double eps2,
               double (*acc)[3], double (*jerk)[3], double *pot,
               int *nn_addr, int *nn_index, double *nn_r2);
void orc_predict(int n, double ti, const double *tj,
                 const double (*x0)[3], const double (*v0)[3],
                 const double (*a0)[3], const double (*j0)[3],
                 double (*xp)[3], double (*vp)[3]);

static double norm3(const double *a) { return sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]); }

static double pow2_floor(double x, double cap)
{
    /* largest power of two <= min(x, cap); cap is itself a power of two */
    double d = cap;
    while (d > x && d > 1e-300) d *= 0.5;
    return d;
}

/* Corrector of one particle (formulas in the header).  In: step h, predicted x_p, v_p, old
 * (a0, adot0), new (a1, adot1).  Out: corrected x1, v1, and a2' = a2 + h a3, a3.
 * Exact whenever the acceleration is a cubic polynomial in time (pinned that way). */
void orc_hermite_correct(double h, const double *xp, const double *vp,
                         const double *a0, const double *ad0, const double *a1, const double *ad1,
                         double *x1, double *v1, double *a2n, double *a3)
{
    double h2 = h * h, h3 = h2 * h, h4 = h3 * h, h5 = h4 * h;
    for (int c = 0; c < 3; ++c) {
        double da = a0[c] - a1[c];
        double a2 = (-6.0 * da - h * (4.0 * ad0[c] + 2.0 * ad1[c])) / h2;
        a3[c] = (12.0 * da + 6.0 * h * (ad0[c] + ad1[c])) / h3;
        x1[c] = xp[c] + h4 * a2 / 24.0 + h5 * a3[c] / 120.0;
        v1[c] = vp[c] + h3 * a2 / 6.0 + h4 * a3[c] / 24.0;
        a2n[c] = a2 + h * a3[c];
    }
}

/* Aarseth step wish (formula in the header) */
double orc_aarseth_dt(double eta, const double *a1, const double *ad1, const double *a2n, const double *a3,
                      double dt_max)
{
    double na = norm3(a1), nad = norm3(ad1), n2 = norm3(a2n), n3 = norm3(a3);
    double den = nad * n3 + n2 * n2;
    return den > 0 ? sqrt(eta * (na * n2 + nad * nad) / den) : dt_max;
}

/* stats: [0] block steps, [1] particle steps, [2] final time, [3] smallest dt used,
 *        [4] pairwise interactions (n_i * N per block step, self pair counted)
 * ni_hist_log2[b] counts block steps with 2^b <= n_i < 2^(b+1).
 * Stops at t_end (a multiple of dt_max, where every particle is synchronised) or after
 * max_block_steps block steps if that is > 0 (then the state is NOT synchronised:
 * x, v are returned as predicted to the last block time). */
/* shared != 0: the shared-time-step variant ("shared or block time steps"; reading 21): every
 * particle is advanced every step with one common step; after the corrector each particle applies the rule above to the
 * common step and the new common step is the smallest result (likewise at the start). */
static int hermite_impl(int n, double (*x)[3], double (*v)[3], const double *m,
                        double eps2, double eta, double eta_start, double dt_max, double t_end,
                        long long max_block_steps, long long *ni_hist_log2, double *stats, int shared)
{
    double (*a)[3] = malloc(sizeof(double[3]) * n), (*ad)[3] = malloc(sizeof(double[3]) * n);
    double (*xp)[3] = malloc(sizeof(double[3]) * n), (*vp)[3] = malloc(sizeof(double[3]) * n);
    double (*xi)[3] = malloc(sizeof(double[3]) * n), (*vi)[3] = malloc(sizeof(double[3]) * n);
    double (*a1)[3] = malloc(sizeof(double[3]) * n), (*ad1)[3] = malloc(sizeof(double[3]) * n);
    double *pot = malloc(sizeof(double) * n), *t = malloc(sizeof(double) * n), *dt = malloc(sizeof(double) * n);
    int *index = malloc(sizeof(int) * n), *act = malloc(sizeof(int) * n), *iidx = malloc(sizeof(int) * n);
    if (!a || !ad || !xp || !vp || !xi || !vi || !a1 || !ad1 || !pot || !t || !dt || !index || !act || !iidx) return -1;

    for (int p = 0; p < n; ++p) { index[p] = p; t[p] = 0.0; }
    /* initial forces: everything at t = 0 */
    orc_force(n, index, (const double (*)[3])x, (const double (*)[3])v, n, index,
              (const double (*)[3])x, (const double (*)[3])v, m, eps2, a, ad, pot, NULL, NULL, NULL);
    double dt_min = dt_max;
    for (int p = 0; p < n; ++p) {
        double na = norm3(a[p]), nad = norm3(ad[p]);
        double want = nad > 0 ? eta_start * na / nad : dt_max;
        dt[p] = pow2_floor(want, dt_max);
        if (dt[p] < dt_min) dt_min = dt[p];
    }
    if (shared) for (int p = 0; p < n; ++p) dt[p] = dt_min;

    long long nblock = 0, npart = 0;
    double inter = 0.0, tnow = 0.0;
    while (tnow < t_end && (max_block_steps <= 0 || nblock < max_block_steps)) {
        /* next block time and active block */
        double tn = INFINITY;
        for (int p = 0; p < n; ++p) if (t[p] + dt[p] < tn) tn = t[p] + dt[p];
        int ni = 0;
        for (int p = 0; p < n; ++p) if (t[p] + dt[p] == tn) act[ni++] = p;
        /* predictor, all particles (Eq. 1-2) */
        orc_predict(n, tn, t, (const double (*)[3])x, (const double (*)[3])v,
                    (const double (*)[3])a, (const double (*)[3])ad, xp, vp);
        for (int k = 0; k < ni; ++k) {
            int p = act[k];
            iidx[k] = p;
            memcpy(xi[k], xp[p], sizeof(double[3]));
            memcpy(vi[k], vp[p], sizeof(double[3]));
        }
        /* force on the active block */
        orc_force(ni, iidx, (const double (*)[3])xi, (const double (*)[3])vi, n, index,
                  (const double (*)[3])xp, (const double (*)[3])vp, m, eps2, a1, ad1, pot, NULL, NULL, NULL);
        /* corrector + new step */
        for (int k = 0; k < ni; ++k) {
            int p = act[k];
            double h = dt[p];
            double a3[3], a2n[3];
            orc_hermite_correct(h, xi[k], vi[k], a[p], ad[p], a1[k], ad1[k], x[p], v[p], a2n, a3);
            for (int c = 0; c < 3; ++c) { a[p][c] = a1[k][c]; ad[p][c] = ad1[k][c]; }
            t[p] = tn;
            double want = orc_aarseth_dt(eta, a[p], ad[p], a2n, a3, dt_max);
            double d = h;
            if (want < d) {
                while (d > want) d *= 0.5;
            } else if (want >= 2.0 * d && 2.0 * d <= dt_max && fmod(tn, 2.0 * d) == 0.0) {
                d *= 2.0;
            }
            dt[p] = d;
            if (d < dt_min) dt_min = d;
        }
        if (shared) {
            double dcommon = dt[act[0]];
            for (int k = 1; k < ni; ++k) if (dt[act[k]] < dcommon) dcommon = dt[act[k]];
            for (int k = 0; k < ni; ++k) dt[act[k]] = dcommon;
        }
        tnow = tn;
        ++nblock;
        npart += ni;
        inter += (double)ni * (double)n;
        int b = 0;
        while ((1LL << (b + 1)) <= ni) ++b;
        ni_hist_log2[b] += 1;
    }
    if (max_block_steps > 0 && tnow < t_end) {
        /* unsynchronised stop: hand back the state predicted to the last block time */
        orc_predict(n, tnow, t, (const double (*)[3])x, (const double (*)[3])v,
                    (const double (*)[3])a, (const double (*)[3])ad, xp, vp);
        memcpy(x, xp, sizeof(double[3]) * n);
        memcpy(v, vp, sizeof(double[3]) * n);
    }
    stats[0] = (double)nblock; stats[1] = (double)npart; stats[2] = tnow; stats[3] = dt_min; stats[4] = inter;
    free(a); free(ad); free(xp); free(vp); free(xi); free(vi); free(a1); free(ad1);
    free(pot); free(t); free(dt); free(index); free(act); free(iidx);
    return 0;
}

int orc_hermite(int n, double (*x)[3], double (*v)[3], const double *m,
                double eps2, double eta, double eta_start, double dt_max, double t_end,
                long long max_block_steps, long long *ni_hist_log2, double *stats)
{
    return hermite_impl(n, x, v, m, eps2, eta, eta_start, dt_max, t_end, max_block_steps, ni_hist_log2, stats, 0);
}

int orc_hermite_shared(int n, double (*x)[3], double (*v)[3], const double *m,
                       double eps2, double eta, double eta_start, double dt_max, double t_end,
                       long long max_block_steps, long long *ni_hist_log2, double *stats)
{
    return hermite_impl(n, x, v, m, eps2, eta, eta_start, dt_max, t_end, max_block_steps, ni_hist_log2, stats, 1);
}
