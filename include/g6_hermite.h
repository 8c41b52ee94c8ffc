/*
 * g6_hermite.h -- host-side 4th-order Hermite predictor-corrector with block time steps (fp64)
 * that drives libg6b200 through the g6_* calling sequence of g6.h, exactly as a GRAPE-6 host
 * code does (section 2; task split of Fig. 1: the host predicts
 * the i-particles and corrects, the device predicts the j-particles and computes the forces).
 *
 * The paper cites the scheme (Makino & Aarseth 1992) and the step criterion
 * (Aarseth 1985) without printing them; the textbook formulas used are
 * listed in DESIGN.md reading 16:
 *   corrector  a2 = [-6 (a0 - a1) - h (4 adot0 + 2 adot1)] / h^2,  a3 = [12 (a0 - a1) + 6 h (adot0 + adot1)] / h^3
 *              x1 = x_p + h^4 a2 / 24 + h^5 a3 / 120,  v1 = v_p + h^3 a2 / 6 + h^4 a3 / 24
 *   step       dt_want = sqrt(eta (|a1||a2'| + |adot1|^2) / (|adot1||a3| + |a2'|^2)),  a2' = a2 + h a3;
 *              power-of-two steps, halved while dt > dt_want, doubled only when dt_want >= 2 dt and the
 *              time is a multiple of 2 dt, dt <= dt_max; first step eta_start |a| / |adot| rounded down.
 *   dt_max     should be a POWER OF TWO (the configurations of BASELINE.json use 1/8): all steps are dt_max halved k times, so the
 *              particle times are then exact binary fractions and the particles of one step level share their block times bit for
 *              bit -- which is what "the same block" means in all three drivers.  Any other positive value is accepted and
 *              integrates correctly (the drivers agree with each other, tested by random comparison at dt_max = 0.1), but sums of
 *              steps are then rounded and particles that reached a time by different step sequences may not compare equal.
 *
 * All pointers are HOST pointers, [][3] arrays row-major fp64; the caller owns them.
 * Functions return 0 or a negative G6_ERR_* code (g6h_create: NULL on failure; the text is in
 * g6x_last_error(clusterid)).  The cluster must have been opened with g6_open and must not be
 * used by anything else while the system exists.  Particle p lives at j address p with index p.
 */
#ifndef G6_B200_HERMITE_H
#define G6_B200_HERMITE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct g6h_system g6h_system;

/* Load n particles (t = 0), compute initial acc/jerk on the device and the initial steps. */
g6h_system *g6h_create(int clusterid, int n, const double x[][3], const double v[][3], const double m[],
                       double eps2, double eta, double eta_start, double dt_max);

void g6h_destroy(g6h_system *s);

/* Advance block step by block step until t_end (a multiple of dt_max: all particles are then
 * synchronised) or for at most max_block_steps (> 0) block steps. */
int g6h_evolve(g6h_system *s, double t_end, long long max_block_steps);

/* Positions and velocities at the current system time: corrected values for particles that
 * are at that time, Eq. 1-2 predictions (host, fp64) for the others. */
int g6h_get_state(g6h_system *s, double x[][3], double v[][3]);

/* stats[0] block steps, [1] particle steps, [2] system time, [3] smallest step used,
 * [4] pairwise interactions (n_i * N per block step), [5] wall seconds spent in g6h_evolve,
 * [6] wall seconds of that inside the g6 force calls.  ni_hist_log2[b] = block steps with
 * 2^b <= n_i < 2^(b+1) (64 entries). */
int g6h_get_stats(g6h_system *s, double stats[8], long long ni_hist_log2[64]);

/* wall_s_log2[b] = wall seconds spent inside the g6 force calls of the block steps counted in
 * ni_hist_log2[b] (64 entries): where the time of a block-step run goes, by block size. */
int g6h_get_force_wall_hist(g6h_system *s, double wall_s_log2[64]);

/* ---- device-resident variant -----------------------------------------------
 * The same integrator with the particle state kept in device memory and the O(n_i) steps -- block
 * selection, prediction of the i-particles, corrector, step choice, j-store update --
 * run as CUDA kernels; the force is the library's own path.  The paper leaves these steps on the CPU
 * because GRAPE host codes did.
 * Block steps of up to 768 particles ("block sizes are typically small on average") run inside ONE persistent
 * cooperative kernel (g6_hermite_loop.cuh: j-tiles resident in shared memory, the CTAs meet through self-validating exchange
 * words) which returns to the host only for a larger block -- whose forces the library's sweep path
 * computes -- at t_end, or when the step budget is used up.  Needs n <= 4 x 256 x (number of SMs) particles; beyond that, or
 * with env G6_HD_LOOP = 0, every block step is two or three launches and one host wait for (n_i, t_next).
 * Environment (read by g6hd_create): G6_HD_LOOP (default 1), G6_HD_LOOP_MAXI (largest block stepped inside the loop, default
 * and at most 768), G6_HD_LOOP_PROFILE (1: the loop built with clock marks, 2: the production loop; both print the time per
 * block-size bin from g6hd_get_stats to stderr), G6_HD_PROFILE (CUDA-event phase times of the path without the loop).
 * Same formulas as above, fp64 (the device contracts a*b+c into FMAs, so results agree with g6h_* to
 * rounding, not bit for bit).  Same argument and error conventions; n <= the cluster's capacity. */
typedef struct g6hd_system g6hd_system;

g6hd_system *g6hd_create(int clusterid, int n, const double x[][3], const double v[][3], const double m[],
                         double eps2, double eta, double eta_start, double dt_max);
void g6hd_destroy(g6hd_system *s);
int g6hd_evolve(g6hd_system *s, double t_end, long long max_block_steps);
/* on != 0: shared time steps from now on ("shared or block time steps"; reading 21): every
 * particle takes every step with one common step, the smallest of the per-particle results of the step rule above
 * applied to the common step.  Call between g6hd_evolve calls; switching back to block steps is allowed.  Switching ON
 * needs every particle at the system time (true at t = 0 and after evolving to a multiple of dt_max): otherwise
 * G6_ERR_SEQUENCE and nothing changes. */
int g6hd_set_shared_steps(g6hd_system *s, int on);
/* as g6h_get_state (Eq. 1-2 predictions to the system time, evaluated on the device) */
int g6hd_get_state(g6hd_system *s, double x[][3], double v[][3]);
/* stats[0..5] as g6h_get_stats ([6], [7] unused) */
int g6hd_get_stats(g6hd_system *s, double stats[8], long long ni_hist_log2[64]);
/* Raw per-particle Hermite state (each at its own time t[p]); any pointer may be NULL.  For parity tests. */
int g6hd_get_particles(g6hd_system *s, double x[][3], double v[][3], double a[][3], double adot[][3], double t[], double dt[]);
/* The last block step's i-block: *ni particles, their addresses, predicted x/v and the forces the corrector
 * used (any array may be NULL; G6_ERR_ARG if *ni > maxn).  For parity tests of the corrector kernel. */
int g6hd_get_last_block(g6hd_system *s, int maxn, int *ni, int act[], double xi[][3], double vi[][3], double acc[][3], double jerk[][3]);

#ifdef __cplusplus
}
#endif
#endif
