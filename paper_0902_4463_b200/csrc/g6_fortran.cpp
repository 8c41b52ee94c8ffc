// g6_fortran.cpp -- Fortran-callable aliases (include/g6_fortran.h): dereference and forward, nothing else.
#include "../../include/g6_fortran.h"
#include "../../include/g6.h"

extern "C" {

int g6_open_(const int *clusterid) { return clusterid ? g6_open(*clusterid) : G6_ERR_ARG; }
int g6_close_(const int *clusterid) { return clusterid ? g6_close(*clusterid) : G6_ERR_ARG; }
int g6_npipes_(void) { return g6_npipes(); }
int g6_set_tunit_(const int *newtunit) { return newtunit ? g6_set_tunit(*newtunit) : G6_ERR_ARG; }
int g6_set_xunit_(const int *newxunit) { return newxunit ? g6_set_xunit(*newxunit) : G6_ERR_ARG; }
int g6_reset_(const int *clusterid) { return clusterid ? g6_reset(*clusterid) : G6_ERR_ARG; }
int g6_reset_fofpga_(const int *clusterid) { return clusterid ? g6_reset_fofpga(*clusterid) : G6_ERR_ARG; }
int g6_initialize_jp_buffer_(const int *clusterid, const int *buf_size)
{
    return (clusterid && buf_size) ? g6_initialize_jp_buffer(*clusterid, *buf_size) : G6_ERR_ARG;
}
int g6_flush_jp_buffer_(const int *clusterid) { return clusterid ? g6_flush_jp_buffer(*clusterid) : G6_ERR_ARG; }
int g6_getnjmax_(const int *clusterid) { return clusterid ? g6_getnjmax(*clusterid) : G6_ERR_ARG; }

int g6_set_j_particle_(const int *clusterid, const int *address, const int *index, const double *tj, const double *dtj,
                       const double *mass, const double snap_by18[3], const double jerk_by6[3], const double acc_by2[3],
                       const double v[3], const double x[3])
{
    if (!clusterid || !address || !index || !tj || !dtj || !mass) return G6_ERR_ARG;
    return g6_set_j_particle(*clusterid, *address, *index, *tj, *dtj, *mass, snap_by18, jerk_by6, acc_by2, v, x);
}

int g6_get_j_particle_(const int *clusterid, const int *address, int *index, double *tj, double *mass, double jerk_by6[3],
                       double acc_by2[3], double v[3], double x[3])
{
    if (!clusterid || !address) return G6_ERR_ARG;
    return g6_get_j_particle(*clusterid, *address, index, tj, mass, jerk_by6, acc_by2, v, x);
}

int g6_set_ti_(const int *clusterid, const double *ti) { return (clusterid && ti) ? g6_set_ti(*clusterid, *ti) : G6_ERR_ARG; }

int g6calc_firsthalf_(const int *clusterid, const int *nj, const int *ni, const int index[], const double xi[][3],
                      const double vi[][3], const double acc_old[][3], const double jerk6_old[][3], const double phi_old[],
                      const double *eps2, const double h2[])
{
    if (!clusterid || !nj || !ni || !eps2) return G6_ERR_ARG;
    return g6calc_firsthalf(*clusterid, *nj, *ni, index, xi, vi, acc_old, jerk6_old, phi_old, *eps2, h2);
}

int g6calc_lasthalf_(const int *clusterid, const int *nj, const int *ni, const int index[], const double xi[][3],
                     const double vi[][3], const double *eps2, const double h2[], double acc[][3], double jerk[][3], double pot[])
{
    if (!clusterid || !nj || !ni || !eps2) return G6_ERR_ARG;
    return g6calc_lasthalf(*clusterid, *nj, *ni, index, xi, vi, *eps2, h2, acc, jerk, pot);
}

int g6calc_lasthalf2_(const int *clusterid, const int *nj, const int *ni, const int index[], const double xi[][3],
                      const double vi[][3], const double *eps2, const double h2[], double acc[][3], double jerk[][3], double pot[],
                      int nnb_index[])
{
    if (!clusterid || !nj || !ni || !eps2) return G6_ERR_ARG;
    return g6calc_lasthalf2(*clusterid, *nj, *ni, index, xi, vi, *eps2, h2, acc, jerk, pot, nnb_index);
}

int g6_read_neighbour_list_(const int *clusterid) { return clusterid ? g6_read_neighbour_list(*clusterid) : G6_ERR_ARG; }

int g6_get_neighbour_list_(const int *clusterid, const int *ipipe, const int *maxlen, int *n, int list[])
{
    if (!clusterid || !ipipe || !maxlen) return G6_ERR_ARG;
    return g6_get_neighbour_list(*clusterid, *ipipe, *maxlen, n, list);
}

}  // extern "C"
