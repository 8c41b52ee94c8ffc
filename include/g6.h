/*
 * g6.h -- C ABI of libg6b200: a GRAPE-6-style direct-summation force engine for NVIDIA B200
 * (sm_100a), after Sapporo (arxiv 0902.4463; cited below as PAPER.md:LINE).
 *
 * The paper reproduces "the calling sequence of the GRAPE-6 library" but
 * prints no prototypes, and the GRAPE-6 header is not available to this build.  The g6_* names
 * and argument ORDER below follow the historical convention as recalled (Taylor coefficients
 * are passed pre-divided: acc/2, jerk/6, snap/18); binary drop-in compatibility with the
 * original header is NOT claimed.  g6x_* are extensions of this library.
 *
 * What one force call computes (PAPER.md:31, :41 fn.3, :80-118, :126):
 * for every i-particle of the block, over all stored j-particles with address in [0, nj) and
 * index_j != index_i, predicted to the time set by g6_set_ti (Eq. 1-2),
 *     dx = x_j - x_i (double-single, Eq. 3), dv = v_j - v_i, s^2 = dx.dx + eps2
 *     acc  = sum m_j dx / s^3
 *     jerk = sum m_j [ dv / s^3 - 3 (dx.dv) dx / s^5 ]          (d acc / dt, physical, not /6)
 *     pot  = - sum m_j / s                                       (negative; no self term)
 *     nearest neighbour = argmin over j of the UNSOFTENED dx.dx, ties -> smallest address.
 * Units G = 1.  Arithmetic: FP32 with double-single separations, partial
 * sums folded into fp64.  All j-particles live on the device; only
 * i-particles and results cross the host-device link per call.
 *
 * General rules
 *  - Every function returns G6_OK (0) or a negative G6_ERR_* code; g6x_last_error() gives text.
 *    No C++ exception crosses this boundary and the library never aborts.
 *  - Pointers are HOST pointers unless the parameter name starts with d_ (DEVICE pointers,
 *    valid on the library's device, 8-byte aligned).  The caller owns every array; the library
 *    copies what it needs before returning and keeps no caller pointer, except that the d_
 *    outputs of g6x_calc_dev are written asynchronously on the library's stream.
 *  - [][3] arrays are C row-major (x,y,z per particle), fp64.
 *  - One host thread per clusterid (not thread-safe, like the original).  clusterid in [0, 4).
 *  - The library never falls back to a CPU path: without a usable CUDA device g6_open fails.
 */
#ifndef G6_B200_H
#define G6_B200_H

#ifdef __cplusplus
extern "C" {
#endif

#define G6_OK                0
#define G6_ERR_NOT_OPEN     -1   /* cluster not opened                                  */
#define G6_ERR_CLUSTER      -2   /* clusterid out of range                              */
#define G6_ERR_ADDRESS      -3   /* j address < 0 or >= capacity                        */
#define G6_ERR_NI           -4   /* ni < 1 or ni > g6_npipes()                          */
#define G6_ERR_NJ           -5   /* nj < 1 or nj > highest stored address + 1           */
#define G6_ERR_SEQUENCE     -6   /* lasthalf without firsthalf, firsthalf twice, ...    */
#define G6_ERR_CUDA         -7   /* a CUDA call failed (text in g6x_last_error)         */
#define G6_ERR_ARG          -8   /* NULL pointer / bad value / mismatch with firsthalf  */
#define G6_ERR_ALREADY_OPEN -9
#define G6_ERR_NOMEM        -10

/* ---- GRAPE-6 calling sequence ------------------------------------- */

/* Acquire device `G6_DEVICE` (env, default 0), a stream and pinned staging.  The j-particle store holds at most
 * env G6_NJMAX addresses (default 2^21; g6_getnjmax) and its device memory is GROWN ON DEMAND: it starts at env
 * G6_NJINIT addresses (default 16384, 1.9 MB) and doubles whenever a higher address is set (76 + 40 B per address). */
int g6_open(int clusterid);

/* Wait for outstanding work and free everything the cluster owns. */
int g6_close(int clusterid);

/* Largest ni accepted by one firsthalf/lasthalf pair.  The paper's library reports 256
 * "pipelines" (PAPER.md:132 fn.7: one 256-thread block of i-particles on a G80); the number a
 * host code should chunk its blocks by on a B200 is what fills the chip, 148 SMs x 3 resident
 * CTAs x 256 i-particles, rounded up to a power of two: G6_DEFAULT_NPIPES.  A host code that
 * chunks by g6_npipes() (as GRAPE-6 codes do) then hands over whole blocks; chunks of 256 cost
 * one call latency each.  env G6_NPIPES or g6x_set_npipes change it (1 .. 2^21); larger
 * blocks are tiled inside the library (the paper's "segments"). */
#define G6_DEFAULT_NPIPES 131072
int g6_npipes(void);

/* Store / overwrite j-memory slot `address` (x, v, a, j and time per particle).
 *   index      caller's particle id: what neighbour queries return and what self-exclusion
 *              compares against the i-particle's index
 *   tj         time at which x, v, acc, jerk are valid
 *   dtj        the particle's step; accepted, not used by the formulas (reading 3)
 *   snap_by18  accepted and ignored (4th-order scheme); may be NULL
 *   jerk_by6, acc_by2   jerk/6 and acc/2 at tj (GRAPE convention, reading 13)
 *   v, x       velocity and position at tj; x is kept in full fp64, the rest in FP32
 *
 * The data is copied before return; the device copy is refreshed at the next firsthalf. */
int g6_set_j_particle(int clusterid, int address, int index, double tj, double dtj, double mass,
                      const double snap_by18[3], const double jerk_by6[3], const double acc_by2[3],
                      const double v[3], const double x[3]);

/* Time to which the j-particles are predicted by the next force call (Eq. 1-2, dt = ti - tj). */
int g6_set_ti(int clusterid, double ti);

/* ---- the rest of the GRAPE-6 calling sequence ----------------------
 * "Sapporo ... emulate[s the] GRAPE6 interface as closely as possible (with the exception of some rarely used
 * functions)" (PAPER.md:196; :9 "simple relinking", :126).  The paper prints none of these calls; names, argument
 * order and meaning are RECALLED from the GRAPE-6 user library and UNVERIFIED (its header is not available to this
 * build), like DESIGN.md reading 13.  Fortran-callable aliases of the whole sequence are in g6_fortran.h. */

/* GRAPE-6 stores times and positions in fixed point; these set the binary scales (2^tunit, 2^xunit) of that format.
 * This library keeps positions in fp64 / double-single, so the values are recorded (g6x_get_units)
 * and have no effect.  Global, like the originals.  Always return 0. */
int g6_set_tunit(int newtunit);
int g6_set_xunit(int newxunit);

/* Forget every j-particle and any unfinished force call of the cluster: as after g6_open, allocations kept. */
int g6_reset(int clusterid);
/* GRAPE-6 resets its force-output FPGA here; nothing to do on a GPU.  Checks the cluster, returns 0. */
int g6_reset_fofpga(int clusterid);

/* The j-particles set by g6_set_j_particle are buffered on the host and sent at the next force call.
 * initialize: size that buffer for buf_size particles in advance (it also grows by itself).
 * flush: send the buffered particles to the device now (asynchronous). */
int g6_initialize_jp_buffer(int clusterid, int buf_size);
int g6_flush_jp_buffer(int clusterid);

/* Largest number of j addresses the cluster can hold (env G6_NJMAX); the largest ni per call is g6_npipes().
 * Returns the POSITIVE count or a negative error. */
int g6_getnjmax(int clusterid);

/* Read j-memory slot `address` back (0 <= address < highest address set + 1): the inverse of g6_set_j_particle.
 * Returns the values AS STORED: x and tj exactly (fp64), mass, v, acc_by2, jerk_by6 rounded to binary32 ("Only the
 * position is stored in DP, whereas the rest of the terms are stored in SP").  Any output pointer may
 * be NULL.  Buffered particles are flushed first; waits for the device. */
int g6_get_j_particle(int clusterid, int address, int *index, double *tj, double *mass, double jerk_by6[3],
                      double acc_by2[3], double v[3], double x[3]);

/* Start a force calculation on ni i-particles against j addresses [0, nj).
 *   index[ni]          ids of the i-particles (for self-exclusion)
 *   xi, vi [ni][3]     positions / velocities ALREADY PREDICTED to ti by the host
 *
 *   acc_old, jerk6_old, phi_old   GRAPE fixed-point scaling hints: ignored, may be NULL
 *   eps2               softening length squared for this block, >= 0
 *   h2[ni]             neighbour-sphere radius squared per i-particle, or NULL.  When given, the
 *                      call also builds neighbour lists ("neighbour lists functionality";
 *                      DESIGN.md reading 20): j is a neighbour of i when the UNSOFTENED
 *                      |x_j - x_i|^2 < h2[i] (strict; compared in binary32 on the double-single
 *                      separation, like the nearest neighbour) and index_j != index_i.  At most
 *                      `nb_maxlen` (option, default G6_NB_MAXLEN = 256, the paper's default)
 *                      neighbours are stored per i, those with the smallest j addresses; the count
 *                      keeps running (count > nb_maxlen = overflow).  Read with
 *                      g6_read_neighbour_list + g6_get_neighbour_list.
 * Copies the block to pinned staging, uploads j-particles changed since the last call, and
 * enqueues predictor -> force -> combine -> download.  Returns without waiting. */
int g6calc_firsthalf(int clusterid, int nj, int ni, const int index[],
                     const double xi[][3], const double vi[][3],
                     const double acc_old[][3], const double jerk6_old[][3], const double phi_old[],
                     double eps2, const double h2[]);

/* Wait for the matching firsthalf (same clusterid, nj, ni) and return its results:
 * acc[ni][3], jerk[ni][3] (physical d acc/dt), pot[ni].  index/xi/vi/eps2/h2 are accepted for
 * signature compatibility and not read. */
int g6calc_lasthalf(int clusterid, int nj, int ni, const int index[],
                    const double xi[][3], const double vi[][3], double eps2, const double h2[],
                    double acc[][3], double jerk[][3], double pot[]);

/* As g6calc_lasthalf, and also the nearest neighbour's index per i (-1 if none). */
int g6calc_lasthalf2(int clusterid, int nj, int ni, const int index[],
                     const double xi[][3], const double vi[][3], double eps2, const double h2[],
                     double acc[][3], double jerk[][3], double pot[], int nnb_index[]);

/* Make the neighbour results of the last completed host force call readable (copies the lists
 * device -> host when the call had h2 != NULL).  Returns 0, or the POSITIVE number of i-particles
 * whose list overflowed nb_maxlen (the caller then shrinks h2 and repeats, as GRAPE-6 codes do),
 * or a negative error. */
#define G6_NB_MAXLEN 256
int g6_read_neighbour_list(int clusterid);

/* Neighbour list of pipe `ipipe` (the ipipe-th i-particle of the last host force call): the
 * callers' INDICES of its neighbours in increasing j-address order, at most `maxlen` (>= 1) of
 * them into list[], their number into *n.  Returns 0, or 1 when neighbours were dropped (the
 * particle has more than nb_maxlen, or more than `maxlen`), or a negative error.
 * If the force call had h2 == NULL the "list" is the single nearest neighbour: *n = 1 and
 * list[0] = its index, or *n = 0. */
int g6_get_neighbour_list(int clusterid, int ipipe, int maxlen, int *n, int list[]);

/* ---- extensions ------------------------------------------------------------------------ */

/* Text of the last error of this cluster (never NULL; valid until the next call). */
const char *g6x_last_error(int clusterid);

/* Raise/lower g6_npipes() (1 .. 2^21).  Global, like g6_npipes itself. */
int g6x_set_npipes(int npipes);

/* Bulk loader, HOST arrays: addresses addr0 .. addr0+n-1.  acc and jerk are PHYSICAL here
 * (not pre-divided).  Same effect as n calls of g6_set_j_particle. */
int g6x_set_j_particles(int clusterid, int addr0, int n, const int index[], const double tj[],
                        const double mass[], const double jerk[][3], const double acc[][3],
                        const double v[][3], const double x[][3]);

/* Bulk read-back, HOST arrays: addresses addr0 .. addr0+n-1 as stored (see g6_get_j_particle); acc and jerk PHYSICAL
 * (2 x and 6 x the stored binary32 values, exact).  Any output pointer may be NULL. */
int g6x_get_j_particles(int clusterid, int addr0, int n, int index[], double tj[], double mass[], double jerk[][3],
                        double acc[][3], double v[][3], double x[][3]);

/* The values last given to g6_set_tunit / g6_set_xunit (0 until set). */
int g6x_get_units(int *tunit, int *xunit);

/* Bulk loader, DEVICE arrays (fp64, same shapes).  Asynchronous on the library's stream. */
int g6x_set_j_particles_dev(int clusterid, int addr0, int n, const int *d_index, const double *d_tj,
                            const double *d_mass, const double *d_jerk, const double *d_acc,
                            const double *d_v, const double *d_x);

/* Whole force call with DEVICE inputs and outputs (fp64 [ni][3] / [ni]; d_nn_index int32,
 * d_nn_r2 fp64, either may be NULL).  ni <= g6_npipes().  Asynchronous on the library's
 * stream; outputs are complete after g6x_synchronize (or any sync of that stream). */
int g6x_calc_dev(int clusterid, int nj, int ni, const int *d_index, const double *d_xi,
                 const double *d_vi, double eps2, double *d_acc, double *d_jerk, double *d_pot,
                 int *d_nn_index, double *d_nn_r2);

/* g6x_calc_dev for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): same arguments, same results (the same predictor, force and combine kernels, PAPER.md section
 * 2.3, :106), but the per-split partial sums go to a FIXED file-scope device array instead of the on-demand buffer
 * that g6x_calc_dev grows with cudaMalloc.  The call allocates and frees nothing, on host or device.
 *  - Limit: (j-splits chosen by the scheduler) x ni <= g6x_noalloc_max_rows() = 65536 rows (4 MiB, held by every GPU
 *    that loads the library until exit); the splits are capped to fit, ni > 65536 is G6_ERR_NI.
 *  - Always the sweep path (predictor, force kernel, combine), also for small blocks; no neighbour lists.
 *  - No j-particle update may be pending (G6_ERR_SEQUENCE): call g6_flush_jp_buffer first -- this call stages nothing.
 *  - The array is shared by all calls on a device and keeps the last call's partials (every row read is written first,
 *    nothing needs clearing).  Calls that OVERLAP on the GPU (two clusters / streams on one device) race on it.
 *  - g6x_noalloc_init resolves the array's device address for the cluster's device (cudaGetSymbolAddress, once per
 *    device); g6x_calc_dev_noalloc does it itself on first use, so call init before a capture begins. */
int g6x_calc_dev_noalloc(int clusterid, int nj, int ni, const int *d_index, const double *d_xi,
                         const double *d_vi, double eps2, double *d_acc, double *d_jerk, double *d_pot,
                         int *d_nn_index, double *d_nn_r2);
int g6x_noalloc_init(int clusterid);
int g6x_noalloc_max_rows(void);

/* g6x_calc_dev with neighbour lists: d_h2[ni] fp64 radii squared in; d_nb_count[ni] (all neighbours
 * found, may exceed nb_maxlen) and d_nb_list[ni][nb_maxlen] (callers' indices, increasing j address;
 * entries past min(count, nb_maxlen) are left untouched) out.  The three pointers are given
 * together or all NULL (= g6x_calc_dev). */
int g6x_calc_dev_nb(int clusterid, int nj, int ni, const int *d_index, const double *d_xi,
                    const double *d_vi, double eps2, double *d_acc, double *d_jerk, double *d_pot,
                    int *d_nn_index, double *d_nn_r2, const double *d_h2, int *d_nb_count, int *d_nb_list);

/* All neighbour lists of the last host force call at once: count[ni] = neighbours found (may exceed
 * what is stored), list[ni][maxlen] row-major = indices, padded with -1.  Returns like
 * g6_read_neighbour_list (number of truncated rows).  G6_ERR_SEQUENCE if that call had h2 == NULL. */
int g6x_get_neighbour_lists(int clusterid, int ni, int maxlen, int count[], int list[]);

/* Nearest neighbour of each i of the last completed host force call: index (-1 if none) and
 * UNSOFTENED squared distance (+inf if none). */
int g6x_get_nearest(int clusterid, int ni, int nn_index[], double nn_r2[]);

/* Use the caller's CUDA stream (a cudaStream_t / CUstream handle cast to void*, NULL for the
 * library's own) for all further work of this cluster.  The cluster must be idle. */
int g6x_set_stream(int clusterid, void *cuda_stream);

/* Block until all work of this cluster has finished. */
int g6x_synchronize(int clusterid);

/* Device times (microseconds, CUDA events) of the phases of the last completed force call:
 * us[0] j upload + scatter, [1] predictor, [2] force kernel, [3] combine, [4] download,
 * [5] whole call enqueue->done; [6] number of force-kernel CTAs, [7] j-splits S. */
int g6x_get_timers(int clusterid, double us[8]);

/* Variant switches (for experiments and tests).  Keys:
 *   "ds"      1 (default) double-single positions; 0 = pure FP32 positions (lo words dropped; the sweep kernel then
 *             forms each separation with 1 packed add instead of Eq. 3's 3: what "DS costs <~ 20 %", is measured against)
 *   "newton"  1 = one Newton step after rsqrt.approx, 0 = none
 *   "jsplit"  0 = automatic; S > 0 forces S j-splits
 *   "kernel"  0 = automatic; 1 = checked reference kernel everywhere; 2 = fast kernel
 *   "timers"  1 = record CUDA events per phase for g6x_get_timers; 0 (default, or env G6_TIMERS) = none:
 *             the event records cost ~10 us per force call, a third of a small block step
 *   "variant" 0 = automatic; threads*8 + i_per_thread forces a fast-kernel shape: one of 128*8+2, 128*8+1, 64*8+1,
 *             32*8+1, 256*8+1 (the automatic ones), 128*8+4, 64*8+2; anything else is G6_ERR_ARG
 *   "small"   largest n_i served by the block-step kernel (one launch: j update + predictor + force +
 *             combine); at most 64, 0 = off.  Until it is set the library uses 64: the kernel beats the
 *             three-launch sweep path at every block size it is built for (with neighbour lists: 28 below 65536
 *             j-particles, 40 below 262144, 64 above; g6x_get_option reports 32 until the option is set)
 *   "nb_maxlen" neighbours stored per i-particle (1 .. 4096, default G6_NB_MAXLEN = 256; compile-time
 *             in the paper); changing it discards the lists of the last call
 *   "last_kernel" (g6x_get_option only) the force kernel the last call took: 1 checked reference kernel,
 *             2 fast sweep kernel, 3 block-step kernel
 * Returns G6_ERR_ARG for an unknown key or value. */
int g6x_set_option(int clusterid, const char *key, int value);
int g6x_get_option(int clusterid, const char *key, int *value);

/* Predicted j-particles (Eq. 1-2 at the current ti) for addresses addr0..addr0+n-1, read back
 * from the device as fp64: xp = hi + lo, vp.  Runs the predictor if needed.  For parity tests. */
int g6x_get_predicted(int clusterid, int addr0, int n, double xp[][3], double vp[][3]);

/* ---- multi-GPU j-split ("n/Q j-particles per GPU", the same i-particles on every GPU) ----
 * Each process (one per GPU) loads its slice of the j-particles -- increasing address ranges by rank --
 * and calls g6x_calc_dev on the SAME i-block; the partial acc/jerk/pot are then SUMMED over the
 * processes and the nearest neighbour is the MINIMUM (ties -> lowest rank = lowest addresses).  The
 * collectives themselves (two allreduces on device buffers: MIN on int64 keys, then SUM on fp64) are the
 * caller's (NCCL through torch.distributed in paper_0902_4463_b200/sharding.py); these three calls are the
 * device-side halves of the nearest-neighbour exchange.  All pointers are DEVICE pointers, work is
 * asynchronous on the cluster's stream.  Neighbour lists are not exchanged.
 *   pack    d_key[i] = (binary32 bits of d_nn_r2[i]) << 32 | rank, INT64_MAX when d_nn_index[i] < 0
 *   select  d_index_f64[i] = d_nn_index[i] if this rank holds the minimum d_key_min[i], else 0
 *   unpack  final d_nn_index / d_nn_r2 (either may be NULL) from the reduced keys and the summed index */
int g6x_jsplit_pack_dev(int clusterid, int ni, int rank, const double *d_nn_r2, const int *d_nn_index, long long *d_key);
int g6x_jsplit_select_dev(int clusterid, int ni, int rank, const long long *d_key_min, const int *d_nn_index, double *d_index_f64);
int g6x_jsplit_unpack_dev(int clusterid, int ni, const long long *d_key_min, const double *d_index_sum, int *d_nn_index, double *d_nn_r2);

/* Library build information: a static string (arch, variant flags). */
const char *g6x_version(void);

#ifdef __cplusplus
}
#endif
#endif /* G6_B200_H */
