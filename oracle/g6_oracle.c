/*
 * oracle/g6_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, obviously-correct fp64 statement of what the Sapporo / GRAPE-6 force
 * path computes (arxiv 0902.4463).  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  It shares no
 * code with the CUDA path under paper_0902_4463_b200/csrc/ and is never a fallback for it.
 *
 * Everything here is the textbook definition written out pair by pair, in the order of
 * the j-addresses, one sqrt and one divide per pair, no blocking, no reordering, compiled
 * WITHOUT -ffast-math and with -ffp-contract=off.  Compile with -DORC_LONG_DOUBLE for the
 * `long double` (x87 80-bit) cross-check build of the same text (pin P7).
 *
 * Passages followed (PAPER.md line numbers; SURVEY.md section 8(c) for the readings where
 * the paper is silent):
 *   orc_predict   PAPER.md:55-64  (section 2.2, Eq. 1-2); dt = t_i - t_j  (reading 3)
 *   orc_force     PAPER.md:31, :41 fn.3, :80, :118, :126 (section 2.3, 2.5): "gravitational
 *                 accelerations, potentials and jerks", softening per i-block, nearest
 *                 neighbour.  The paper does not print the pair formulas; they are the
 *                 Hermite quantities of Makino & Aarseth 1992 which it cites (reading 1):
 *                     dx = x_j - x_i, dv = v_j - v_i, s2 = dx.dx + eps2
 *                     a    += m_j dx / s^3
 *                     adot += m_j [ dv / s^3 - 3 (dx.dv) dx / s^5 ]
 *                     phi  -= m_j / s
 *                 Self-interaction: a pair is skipped when index_j == index_i (reading 4);
 *                 a pair with s2 == 0 is skipped (reading 5); nearest neighbour = argmin of
 *                 the UNSOFTENED r2 = dx.dx, ties -> smallest j address (readings 6-8);
 *                 none -> address -1, index -1, r2 = +inf.
 *   orc_neighbours  neighbour lists, PAPER.md:206 (section 4): "a neighbour lists functionality ...
 *                 The maximum number of neighbours that a particle in a block can store is
 *                 configured at compile time (default is 256)".  The paper says no more; the
 *                 reading (reading 20) is the GRAPE-6 one: j is a neighbour of i when
 *                 the UNSOFTENED r2 = |x_j - x_i|^2 < h2_i (strict), index_j != index_i; the
 *                 list holds the j addresses in increasing order; count = all neighbours, the
 *                 stored list is its first `maxlen` entries (count > maxlen = overflow).
 *   orc_energy    total kinetic and (softened) potential energy, the quantity the paper's
 *                 accuracy test monitors (dE/E).
 *   orc_ds_*      double-single numbers, PAPER.md:68-74, :86 fn.5, and the truncated
 *                 DS difference Eq. 3, in IEEE binary32 (reading 12).
 *
 * Pins (tests/test_oracle_pins.py): two-body closed form, regular polygon, rigid rotation,
 * homologous expansion, Newton's third law, Plummer W = -1/2, 50-digit decimal brute force,
 * translation invariance, cubic-polynomial predictor, phi self-term, DS error bounds;
 * orc_neighbours: lattice shell counts (closed form), consistency with the nearest neighbour
 * of orc_force, overflow rule.
 * No function in this file is "parity unpinned".
 */
#include <math.h>
#include <stddef.h>

#ifdef ORC_LONG_DOUBLE
typedef long double real;
#define ORC_SQRT sqrtl
#else
typedef double real;
#define ORC_SQRT sqrt
#endif

/* ---- Eq. 1-2: j-particle predictor, dt_j = t_i - t_j ------------------ */
void orc_predict(int n, double ti, const double *tj,
                 const double (*x0)[3], const double (*v0)[3],
                 const double (*a0)[3], const double (*j0)[3],
                 double (*xp)[3], double (*vp)[3])
{
    for (int p = 0; p < n; ++p) {
        real dt = (real)ti - (real)tj[p];
        real dt2 = dt * dt;
        real dt3 = dt2 * dt;
        for (int k = 0; k < 3; ++k) {
            /* Eq. 1 */
            xp[p][k] = (double)((real)x0[p][k] + (real)v0[p][k] * dt
                                + (real)a0[p][k] * dt2 / 2 + (real)j0[p][k] * dt3 / 6);
            /* Eq. 2 */
            vp[p][k] = (double)((real)v0[p][k] + (real)a0[p][k] * dt
                                + (real)j0[p][k] * dt2 / 2);
        }
    }
}

/* ---- the force sum (section 2.3; formulas: reading 1) -------------------------- */
void orc_force(int ni, const int *index_i, const double (*xi)[3], const double (*vi)[3],
               int nj, const int *index_j, const double (*xj)[3], const double (*vj)[3],
               const double *mj, double eps2,
               double (*acc)[3], double (*jerk)[3], double *pot,
               int *nn_addr, int *nn_index, double *nn_r2)
{
#pragma omp parallel for schedule(static)
    for (int i = 0; i < ni; ++i) {
        real ax = 0, ay = 0, az = 0, jx = 0, jy = 0, jz = 0, phi = 0;
        real best = INFINITY;
        int best_addr = -1;
        for (int j = 0; j < nj; ++j) {
            if (index_j[j] == index_i[i]) continue;            /* reading 4 */
            real dx = (real)xj[j][0] - (real)xi[i][0];
            real dy = (real)xj[j][1] - (real)xi[i][1];
            real dz = (real)xj[j][2] - (real)xi[i][2];
            real dvx = (real)vj[j][0] - (real)vi[i][0];
            real dvy = (real)vj[j][1] - (real)vi[i][1];
            real dvz = (real)vj[j][2] - (real)vi[i][2];
            real r2 = dx * dx + dy * dy + dz * dz;
            real s2 = r2 + (real)eps2;
            if (s2 == 0) continue;                             /* reading 5 */
            if (r2 < best) { best = r2; best_addr = j; }       /* readings 6-7: strict <, first wins */
            real s = ORC_SQRT(s2);                             /* one sqrt, one divide per pair */
            real rinv = 1 / s;
            real rinv2 = rinv * rinv;
            real m = (real)mj[j];
            real mrinv = m * rinv;                             /* m / s   */
            real mrinv3 = mrinv * rinv2;                       /* m / s^3 */
            real rv = dx * dvx + dy * dvy + dz * dvz;
            real alpha = 3 * rv * rinv2;                       /* 3 (dx.dv) / s^2 */
            ax += mrinv3 * dx;
            ay += mrinv3 * dy;
            az += mrinv3 * dz;
            jx += mrinv3 * (dvx - alpha * dx);
            jy += mrinv3 * (dvy - alpha * dy);
            jz += mrinv3 * (dvz - alpha * dz);
            phi -= mrinv;
        }
        acc[i][0] = (double)ax;  acc[i][1] = (double)ay;  acc[i][2] = (double)az;
        jerk[i][0] = (double)jx; jerk[i][1] = (double)jy; jerk[i][2] = (double)jz;
        pot[i] = (double)phi;
        if (nn_addr)  nn_addr[i] = best_addr;
        if (nn_index) nn_index[i] = best_addr >= 0 ? index_j[best_addr] : -1;
        if (nn_r2)    nn_r2[i] = (double)best;
    }
}

/* ---- neighbour lists (reading 20) -------------------------------- */
void orc_neighbours(int ni, const int *index_i, const double (*xi)[3], const double *h2,
                    int nj, const int *index_j, const double (*xj)[3],
                    int maxlen, int *count, int *list_addr)
{
#pragma omp parallel for schedule(dynamic, 16)
    for (int i = 0; i < ni; ++i) {
        int n = 0;
        for (int j = 0; j < nj; ++j) {
            if (index_j[j] == index_i[i]) continue;
            real dx = (real)xj[j][0] - (real)xi[i][0];
            real dy = (real)xj[j][1] - (real)xi[i][1];
            real dz = (real)xj[j][2] - (real)xi[i][2];
            real r2 = dx * dx + dy * dy + dz * dz;
            if (r2 < (real)h2[i]) {
                if (n < maxlen) list_addr[(size_t)i * maxlen + n] = j;
                ++n;
            }
        }
        count[i] = n;
    }
}

/* ---- energies: T = 1/2 sum m v^2,  W = - sum_{i<j} m_i m_j / sqrt(r_ij^2 + eps2) -------- */
void orc_energy(int n, const double (*x)[3], const double (*v)[3], const double *m,
                double eps2, double *T_out, double *W_out)
{
    real T = 0, W = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : T, W)
    for (int i = 0; i < n; ++i) {
        T += (real)m[i] * ((real)v[i][0] * v[i][0] + (real)v[i][1] * v[i][1] + (real)v[i][2] * v[i][2]) / 2;
        real w = 0;
        for (int j = i + 1; j < n; ++j) {
            real dx = (real)x[j][0] - (real)x[i][0];
            real dy = (real)x[j][1] - (real)x[i][1];
            real dz = (real)x[j][2] - (real)x[i][2];
            w -= (real)m[j] / ORC_SQRT(dx * dx + dy * dy + dz * dz + (real)eps2);
        }
        W += (real)m[i] * w;
    }
    *T_out = (double)T;
    *W_out = (double)W;
}

/* ---- double-single numbers and Eq. 3 ----------- */
/* split: hi = nearest binary32 to x, lo = nearest binary32 to (x - hi)   (reading 12)      */
void orc_ds_split(int n, const double *x, float *hi, float *lo)
{
    for (int p = 0; p < n; ++p) {
        float h = (float)x[p];
        hi[p] = h;
        lo[p] = (float)(x[p] - (double)h);
    }
}

/* Eq. 3: dx = (xj_hi - xi_hi) + (xj_lo - xi_lo), three binary32 operations, result binary32 */
void orc_ds_diff(int n, const float *xj_hi, const float *xj_lo,
                 const float *xi_hi, const float *xi_lo, float *dx)
{
    for (int p = 0; p < n; ++p) {
        volatile float a = xj_hi[p] - xi_hi[p];
        volatile float b = xj_lo[p] - xi_lo[p];
        volatile float c = a + b;
        dx[p] = c;
    }
}

int orc_sizeof_real(void) { return (int)sizeof(real); }
