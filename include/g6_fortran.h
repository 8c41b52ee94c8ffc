/*
 * g6_fortran.h -- Fortran-callable aliases of the GRAPE-6 calling sequence of g6.h.
 *
 * The paper's library is meant to be relinked into existing GRAPE-6 host codes ("simple relinking",
 * :126, :196); several of those (NBODY4, phiGRAPE's Fortran ancestors) are Fortran programs.  The convention
 * provided here is the common one of Fortran 77 compilers on Unix: the C symbol is the lower-case name with ONE
 * trailing underscore, every argument is passed BY REFERENCE, and a Fortran array xi(3, ni) (column-major) is
 * the C array xi[ni][3] of g6.h.  Names and argument lists are those of g6.h, as recalled; binary compatibility
 * with the original GRAPE-6 library is not claimed (its header is not available to this build) -- "recalled,
 * unverified" like DESIGN.md reading 13.  Each alias only dereferences its arguments and calls the g6.h function
 * of the same name; return values are the same (functions, INTEGER in Fortran).
 */
#ifndef G6_B200_FORTRAN_H
#define G6_B200_FORTRAN_H

#ifdef __cplusplus
extern "C" {
#endif

int g6_open_(const int *clusterid);
int g6_close_(const int *clusterid);
int g6_npipes_(void);
int g6_set_tunit_(const int *newtunit);
int g6_set_xunit_(const int *newxunit);
int g6_reset_(const int *clusterid);
int g6_reset_fofpga_(const int *clusterid);
int g6_initialize_jp_buffer_(const int *clusterid, const int *buf_size);
int g6_flush_jp_buffer_(const int *clusterid);
int g6_getnjmax_(const int *clusterid);
int g6_set_j_particle_(const int *clusterid, const int *address, const int *index, const double *tj, const double *dtj,
                       const double *mass, const double snap_by18[3], const double jerk_by6[3], const double acc_by2[3],
                       const double v[3], const double x[3]);
int g6_get_j_particle_(const int *clusterid, const int *address, int *index, double *tj, double *mass, double jerk_by6[3],
                       double acc_by2[3], double v[3], double x[3]);
int g6_set_ti_(const int *clusterid, const double *ti);
int g6calc_firsthalf_(const int *clusterid, const int *nj, const int *ni, const int index[], const double xi[][3],
                      const double vi[][3], const double acc_old[][3], const double jerk6_old[][3], const double phi_old[],
                      const double *eps2, const double h2[]);
int g6calc_lasthalf_(const int *clusterid, const int *nj, const int *ni, const int index[], const double xi[][3],
                     const double vi[][3], const double *eps2, const double h2[], double acc[][3], double jerk[][3], double pot[]);
int g6calc_lasthalf2_(const int *clusterid, const int *nj, const int *ni, const int index[], const double xi[][3],
                      const double vi[][3], const double *eps2, const double h2[], double acc[][3], double jerk[][3], double pot[],
                      int nnb_index[]);
int g6_read_neighbour_list_(const int *clusterid);
int g6_get_neighbour_list_(const int *clusterid, const int *ipipe, const int *maxlen, int *n, int list[]);

#ifdef __cplusplus
}
#endif
#endif /* G6_B200_FORTRAN_H */
