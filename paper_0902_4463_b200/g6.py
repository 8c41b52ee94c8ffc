"""Thin ctypes binding of libg6b200.so: the same names as include/g6.h, argument marshalling only.

Every step of the path (j-store update, predictor, force, combine) runs in the CUDA kernels
behind the C ABI; nothing here computes.  There is no CPU fallback: if the shared library is
missing or no CUDA device is usable, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libg6b200.so")

#: include/g6.h G6_DEFAULT_NPIPES
DEFAULT_NPIPES = 131072

#: every symbol include/g6.h declares (tests check that the library exports each of them)
SYMBOLS = [
    "g6_open", "g6_close", "g6_npipes", "g6_set_j_particle", "g6_set_ti", "g6calc_firsthalf",
    "g6calc_lasthalf", "g6calc_lasthalf2", "g6_read_neighbour_list", "g6_get_neighbour_list",
    "g6_set_tunit", "g6_set_xunit", "g6_reset", "g6_reset_fofpga", "g6_initialize_jp_buffer", "g6_flush_jp_buffer",
    "g6_getnjmax", "g6_get_j_particle", "g6x_get_j_particles", "g6x_get_units",
    "g6x_last_error", "g6x_set_npipes", "g6x_set_j_particles", "g6x_set_j_particles_dev", "g6x_calc_dev",
    "g6x_calc_dev_noalloc", "g6x_noalloc_init", "g6x_noalloc_max_rows",
    "g6x_calc_dev_nb", "g6x_get_neighbour_lists", "g6x_jsplit_pack_dev", "g6x_jsplit_select_dev", "g6x_jsplit_unpack_dev",
    "g6x_get_nearest", "g6x_set_stream", "g6x_synchronize", "g6x_get_timers", "g6x_set_option",
    "g6x_get_option", "g6x_get_predicted", "g6x_version",
    "g6h_create", "g6h_destroy", "g6h_evolve", "g6h_get_state", "g6h_get_stats", "g6h_get_force_wall_hist",
    "g6hd_create", "g6hd_destroy", "g6hd_evolve", "g6hd_get_state", "g6hd_get_stats", "g6hd_get_particles", "g6hd_get_last_block", "g6hd_set_shared_steps",
]

#: the Fortran-callable aliases include/g6_fortran.h declares (trailing underscore, arguments by reference)
FORTRAN_SYMBOLS = [
    "g6_open_", "g6_close_", "g6_npipes_", "g6_set_tunit_", "g6_set_xunit_", "g6_reset_", "g6_reset_fofpga_",
    "g6_initialize_jp_buffer_", "g6_flush_jp_buffer_", "g6_getnjmax_", "g6_set_j_particle_", "g6_get_j_particle_",
    "g6_set_ti_", "g6calc_firsthalf_", "g6calc_lasthalf_", "g6calc_lasthalf2_", "g6_read_neighbour_list_",
    "g6_get_neighbour_list_",
]

ERRORS = {0: "G6_OK", -1: "G6_ERR_NOT_OPEN", -2: "G6_ERR_CLUSTER", -3: "G6_ERR_ADDRESS", -4: "G6_ERR_NI",
          -5: "G6_ERR_NJ", -6: "G6_ERR_SEQUENCE", -7: "G6_ERR_CUDA", -8: "G6_ERR_ARG",
          -9: "G6_ERR_ALREADY_OPEN", -10: "G6_ERR_NOMEM"}


class G6Error(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"{ERRORS.get(code, code)}: {text}")
        self.code = code


_lib = None


def lib():
    """The loaded shared library (loaded on first use; raises if it has not been built)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(
                f"{LIB_PATH} is missing: build it with `python -m paper_0902_4463_b200.build` "
                "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.g6x_last_error.restype = C.c_char_p
        L.g6x_version.restype = C.c_char_p
        L.g6h_create.restype = C.c_void_p
        L.g6hd_create.restype = C.c_void_p
        _lib = L
    return _lib


def _chk(rc, clusterid=0):
    if rc < 0:
        raise G6Error(rc, lib().g6x_last_error(C.c_int(clusterid)).decode())
    return rc


def _f64(a, shape):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if a.shape != shape:
        raise ValueError(f"expected shape {shape}, got {a.shape}")
    return a


def _i32(a, shape):
    a = np.ascontiguousarray(a, dtype=np.int32)
    if a.shape != shape:
        raise ValueError(f"expected shape {shape}, got {a.shape}")
    return a


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int))


def _vec3(a):
    return _dp(_f64(a, (3,)))


# ---- GRAPE-6 calling sequence ------------------------------------------------------------------
def g6_open(clusterid=0):
    return _chk(lib().g6_open(C.c_int(clusterid)), clusterid)


def g6_close(clusterid=0):
    return _chk(lib().g6_close(C.c_int(clusterid)), clusterid)


def g6_npipes():
    return lib().g6_npipes()


def g6_set_j_particle(clusterid, address, index, tj, dtj, mass, snap_by18, jerk_by6, acc_by2, v, x):
    snap = _vec3(snap_by18) if snap_by18 is not None else None
    return _chk(lib().g6_set_j_particle(C.c_int(clusterid), C.c_int(address), C.c_int(index), C.c_double(tj),
                                        C.c_double(dtj), C.c_double(mass), snap, _vec3(jerk_by6), _vec3(acc_by2),
                                        _vec3(v), _vec3(x)), clusterid)


def g6_set_ti(clusterid, ti):
    return _chk(lib().g6_set_ti(C.c_int(clusterid), C.c_double(ti)), clusterid)


def g6_set_tunit(newtunit):
    return lib().g6_set_tunit(C.c_int(newtunit))


def g6_set_xunit(newxunit):
    return lib().g6_set_xunit(C.c_int(newxunit))


def g6x_get_units():
    t = C.c_int(0); x = C.c_int(0)
    lib().g6x_get_units(C.byref(t), C.byref(x))
    return t.value, x.value


def g6_reset(clusterid=0):
    return _chk(lib().g6_reset(C.c_int(clusterid)), clusterid)


def g6_reset_fofpga(clusterid=0):
    return _chk(lib().g6_reset_fofpga(C.c_int(clusterid)), clusterid)


def g6_initialize_jp_buffer(clusterid, buf_size):
    return _chk(lib().g6_initialize_jp_buffer(C.c_int(clusterid), C.c_int(buf_size)), clusterid)


def g6_flush_jp_buffer(clusterid=0):
    return _chk(lib().g6_flush_jp_buffer(C.c_int(clusterid)), clusterid)


def g6_getnjmax(clusterid=0):
    return _chk(lib().g6_getnjmax(C.c_int(clusterid)), clusterid)


def g6_get_j_particle(clusterid, address):
    """Returns dict(index, tj, mass, jerk_by6[3], acc_by2[3], v[3], x[3]) as stored."""
    idx = C.c_int(0); tj = C.c_double(0); mass = C.c_double(0)
    j6 = np.empty(3); a2 = np.empty(3); v = np.empty(3); x = np.empty(3)
    _chk(lib().g6_get_j_particle(C.c_int(clusterid), C.c_int(address), C.byref(idx), C.byref(tj), C.byref(mass),
                                 _dp(j6), _dp(a2), _dp(v), _dp(x)), clusterid)
    return dict(index=idx.value, tj=tj.value, mass=mass.value, jerk_by6=j6, acc_by2=a2, v=v, x=x)


def g6x_get_j_particles(clusterid, addr0, n):
    """Bulk read-back: dict(index[n], tj[n], mass[n], jerk[n,3], acc[n,3], v[n,3], x[n,3]); acc and jerk physical."""
    o = dict(index=np.empty(n, np.int32), tj=np.empty(n), mass=np.empty(n), jerk=np.empty((n, 3)), acc=np.empty((n, 3)),
             v=np.empty((n, 3)), x=np.empty((n, 3)))
    _chk(lib().g6x_get_j_particles(C.c_int(clusterid), C.c_int(addr0), C.c_int(n), _ip(o["index"]), _dp(o["tj"]), _dp(o["mass"]),
                                   _dp(o["jerk"]), _dp(o["acc"]), _dp(o["v"]), _dp(o["x"])), clusterid)
    return o


def g6calc_firsthalf(clusterid, nj, ni, index, xi, vi, acc_old=None, jerk6_old=None, phi_old=None, eps2=0.0, h2=None):
    index = _i32(index, (ni,)); xi = _f64(xi, (ni, 3)); vi = _f64(vi, (ni, 3))
    h2p = _dp(_f64(h2, (ni,))) if h2 is not None else None
    return _chk(lib().g6calc_firsthalf(C.c_int(clusterid), C.c_int(nj), C.c_int(ni), _ip(index), _dp(xi), _dp(vi),
                                       None, None, None, C.c_double(eps2), h2p), clusterid)


def g6calc_lasthalf(clusterid, nj, ni, index=None, xi=None, vi=None, eps2=0.0, h2=None):
    """Returns (acc[ni,3], jerk[ni,3], pot[ni])."""
    acc = np.empty((ni, 3)); jerk = np.empty((ni, 3)); pot = np.empty(ni)
    _chk(lib().g6calc_lasthalf(C.c_int(clusterid), C.c_int(nj), C.c_int(ni), None, None, None, C.c_double(eps2), None,
                               _dp(acc), _dp(jerk), _dp(pot)), clusterid)
    return acc, jerk, pot


def g6calc_lasthalf2(clusterid, nj, ni, index=None, xi=None, vi=None, eps2=0.0, h2=None):
    """Returns (acc, jerk, pot, nnb_index[ni])."""
    acc = np.empty((ni, 3)); jerk = np.empty((ni, 3)); pot = np.empty(ni); nn = np.empty(ni, np.int32)
    _chk(lib().g6calc_lasthalf2(C.c_int(clusterid), C.c_int(nj), C.c_int(ni), None, None, None, C.c_double(eps2), None,
                                _dp(acc), _dp(jerk), _dp(pot), _ip(nn)), clusterid)
    return acc, jerk, pot, nn


def g6_read_neighbour_list(clusterid):
    return _chk(lib().g6_read_neighbour_list(C.c_int(clusterid)), clusterid)


def g6_get_neighbour_list(clusterid, ipipe, maxlen=1):
    n = C.c_int(0)
    lst = np.zeros(max(maxlen, 1), np.int32)
    _chk(lib().g6_get_neighbour_list(C.c_int(clusterid), C.c_int(ipipe), C.c_int(maxlen), C.byref(n), _ip(lst)), clusterid)
    return lst[: n.value].copy()


def g6x_get_neighbour_lists(clusterid, ni, maxlen):
    """Returns (count[ni], list[ni, maxlen] padded with -1, number of truncated rows)."""
    count = np.empty(ni, np.int32); lst = np.empty((ni, maxlen), np.int32)
    over = _chk(lib().g6x_get_neighbour_lists(C.c_int(clusterid), C.c_int(ni), C.c_int(maxlen), _ip(count), _ip(lst)), clusterid)
    return count, lst, over


# ---- extensions ----------------------------------------------------------------------------------
def g6x_last_error(clusterid=0):
    return lib().g6x_last_error(C.c_int(clusterid)).decode()


def g6x_version():
    return lib().g6x_version().decode()


def g6x_set_npipes(npipes):
    rc = lib().g6x_set_npipes(C.c_int(npipes))
    if rc < 0:
        raise G6Error(rc, f"npipes = {npipes}")
    return rc


def g6x_set_j_particles(clusterid, addr0, index, tj, mass, jerk, acc, v, x):
    """Bulk loader, host arrays; acc and jerk physical."""
    n = len(index)
    index = _i32(index, (n,)); tj = _f64(tj, (n,)); mass = _f64(mass, (n,))
    jerk = _f64(jerk, (n, 3)); acc = _f64(acc, (n, 3)); v = _f64(v, (n, 3)); x = _f64(x, (n, 3))
    return _chk(lib().g6x_set_j_particles(C.c_int(clusterid), C.c_int(addr0), C.c_int(n), _ip(index), _dp(tj), _dp(mass),
                                          _dp(jerk), _dp(acc), _dp(v), _dp(x)), clusterid)


def _dev(t, dtype, numel):
    """device pointer of a torch CUDA tensor (torch is used for device memory only)."""
    import torch
    if t is None:
        return None
    if not (t.is_cuda and t.is_contiguous() and t.dtype == dtype and t.numel() == numel):
        raise ValueError(f"need a contiguous CUDA tensor of {dtype} with {numel} elements, got {t.dtype} {tuple(t.shape)} {t.device}")
    return C.c_void_p(t.data_ptr())


def g6x_set_j_particles_dev(clusterid, addr0, n, d_index, d_tj, d_mass, d_jerk, d_acc, d_v, d_x):
    import torch
    f, i = torch.float64, torch.int32
    return _chk(lib().g6x_set_j_particles_dev(C.c_int(clusterid), C.c_int(addr0), C.c_int(n), _dev(d_index, i, n),
                                              _dev(d_tj, f, n), _dev(d_mass, f, n), _dev(d_jerk, f, 3 * n),
                                              _dev(d_acc, f, 3 * n), _dev(d_v, f, 3 * n), _dev(d_x, f, 3 * n)), clusterid)


def g6x_calc_dev(clusterid, nj, ni, d_index, d_xi, d_vi, eps2, d_acc, d_jerk, d_pot, d_nn_index=None, d_nn_r2=None):
    import torch
    f, i = torch.float64, torch.int32
    return _chk(lib().g6x_calc_dev(C.c_int(clusterid), C.c_int(nj), C.c_int(ni), _dev(d_index, i, ni), _dev(d_xi, f, 3 * ni),
                                   _dev(d_vi, f, 3 * ni), C.c_double(eps2), _dev(d_acc, f, 3 * ni), _dev(d_jerk, f, 3 * ni),
                                   _dev(d_pot, f, ni), _dev(d_nn_index, i, ni), _dev(d_nn_r2, f, ni)), clusterid)


def g6x_calc_dev_noalloc(clusterid, nj, ni, d_index, d_xi, d_vi, eps2, d_acc, d_jerk, d_pot, d_nn_index=None, d_nn_r2=None):
    import torch
    f, i = torch.float64, torch.int32
    return _chk(lib().g6x_calc_dev_noalloc(C.c_int(clusterid), C.c_int(nj), C.c_int(ni), _dev(d_index, i, ni), _dev(d_xi, f, 3 * ni),
                                           _dev(d_vi, f, 3 * ni), C.c_double(eps2), _dev(d_acc, f, 3 * ni), _dev(d_jerk, f, 3 * ni),
                                           _dev(d_pot, f, ni), _dev(d_nn_index, i, ni), _dev(d_nn_r2, f, ni)), clusterid)


def g6x_noalloc_init(clusterid):
    return _chk(lib().g6x_noalloc_init(C.c_int(clusterid)), clusterid)


def g6x_noalloc_max_rows():
    return int(lib().g6x_noalloc_max_rows())


def g6x_calc_dev_nb(clusterid, nj, ni, d_index, d_xi, d_vi, eps2, d_acc, d_jerk, d_pot, d_nn_index, d_nn_r2, d_h2, d_nb_count, d_nb_list):
    import torch
    f, i = torch.float64, torch.int32
    return _chk(lib().g6x_calc_dev_nb(C.c_int(clusterid), C.c_int(nj), C.c_int(ni), _dev(d_index, i, ni), _dev(d_xi, f, 3 * ni),
                                      _dev(d_vi, f, 3 * ni), C.c_double(eps2), _dev(d_acc, f, 3 * ni), _dev(d_jerk, f, 3 * ni),
                                      _dev(d_pot, f, ni), _dev(d_nn_index, i, ni), _dev(d_nn_r2, f, ni), _dev(d_h2, f, ni),
                                      _dev(d_nb_count, i, ni), _dev(d_nb_list, i, d_nb_list.numel() if d_nb_list is not None else 0)),
                clusterid)


def g6x_get_nearest(clusterid, ni):
    idx = np.empty(ni, np.int32); r2 = np.empty(ni)
    _chk(lib().g6x_get_nearest(C.c_int(clusterid), C.c_int(ni), _ip(idx), _dp(r2)), clusterid)
    return idx, r2


def g6x_set_stream(clusterid, cuda_stream):
    return _chk(lib().g6x_set_stream(C.c_int(clusterid), C.c_void_p(cuda_stream or 0)), clusterid)


def g6x_synchronize(clusterid=0):
    return _chk(lib().g6x_synchronize(C.c_int(clusterid)), clusterid)


def g6x_get_timers(clusterid=0):
    us = np.zeros(8)
    _chk(lib().g6x_get_timers(C.c_int(clusterid), _dp(us)), clusterid)
    return dict(upload_us=us[0], predict_us=us[1], force_us=us[2], combine_us=us[3], download_us=us[4],
                total_us=us[5], force_ctas=int(us[6]), jsplits=int(us[7]))


def g6x_set_option(clusterid, key, value):
    return _chk(lib().g6x_set_option(C.c_int(clusterid), key.encode(), C.c_int(int(value))), clusterid)


def g6x_get_option(clusterid, key):
    v = C.c_int(0)
    _chk(lib().g6x_get_option(C.c_int(clusterid), key.encode(), C.byref(v)), clusterid)
    return v.value


def g6x_get_predicted(clusterid, addr0, n):
    xp = np.empty((n, 3)); vp = np.empty((n, 3))
    _chk(lib().g6x_get_predicted(C.c_int(clusterid), C.c_int(addr0), C.c_int(n), _dp(xp), _dp(vp)), clusterid)
    return xp, vp


def g6x_jsplit_pack_dev(clusterid, ni, rank, d_nn_r2, d_nn_index, d_key):
    import torch
    return _chk(lib().g6x_jsplit_pack_dev(C.c_int(clusterid), C.c_int(ni), C.c_int(rank), _dev(d_nn_r2, torch.float64, ni),
                                          _dev(d_nn_index, torch.int32, ni), _dev(d_key, torch.int64, ni)), clusterid)


def g6x_jsplit_select_dev(clusterid, ni, rank, d_key_min, d_nn_index, d_index_f64):
    import torch
    return _chk(lib().g6x_jsplit_select_dev(C.c_int(clusterid), C.c_int(ni), C.c_int(rank), _dev(d_key_min, torch.int64, ni),
                                            _dev(d_nn_index, torch.int32, ni), _dev(d_index_f64, torch.float64, ni)), clusterid)


def g6x_jsplit_unpack_dev(clusterid, ni, d_key_min, d_index_sum, d_nn_index, d_nn_r2):
    import torch
    return _chk(lib().g6x_jsplit_unpack_dev(C.c_int(clusterid), C.c_int(ni), _dev(d_key_min, torch.int64, ni),
                                            _dev(d_index_sum, torch.float64, ni), _dev(d_nn_index, torch.int32, ni),
                                            _dev(d_nn_r2, torch.float64, ni)), clusterid)


# ---- convenience (still only calls the functions above) ------------------------------------------
def force_host(clusterid, index, xi, vi, eps2, nj, h2=None):
    """firsthalf + lasthalf2 + nearest-neighbour distances through HOST buffers."""
    ni = len(index)
    g6calc_firsthalf(clusterid, nj, ni, index, xi, vi, eps2=eps2, h2=h2)
    acc, jerk, pot, nn = g6calc_lasthalf2(clusterid, nj, ni, eps2=eps2)
    _, r2 = g6x_get_nearest(clusterid, ni)
    return dict(acc=acc, jerk=jerk, pot=pot, nn_index=nn, nn_r2=r2)


# ---- host Hermite driver (include/g6_hermite.h) ---------------------------------------------------
class Hermite:
    """4th-order Hermite block-step integration driven through the g6_* ABI (g6h_* functions)."""

    def __init__(self, clusterid, x, v, m, eps2, eta, eta_start=0.01, dt_max=0.125):
        n = len(m)
        x = _f64(x, (n, 3)); v = _f64(v, (n, 3)); m = _f64(m, (n,))
        self.n, self.clusterid = n, clusterid
        self._h = lib().g6h_create(C.c_int(clusterid), C.c_int(n), _dp(x), _dp(v), _dp(m), C.c_double(eps2),
                                   C.c_double(eta), C.c_double(eta_start), C.c_double(dt_max))
        if not self._h:
            raise G6Error(-8, "g6h_create failed: " + g6x_last_error(clusterid))

    def evolve(self, t_end, max_block_steps=0):
        return _chk(lib().g6h_evolve(C.c_void_p(self._h), C.c_double(t_end), C.c_longlong(max_block_steps)), self.clusterid)

    def state(self):
        x = np.empty((self.n, 3)); v = np.empty((self.n, 3))
        _chk(lib().g6h_get_state(C.c_void_p(self._h), _dp(x), _dp(v)), self.clusterid)
        return x, v

    def stats(self):
        st = np.zeros(8); hist = np.zeros(64, np.int64)
        _chk(lib().g6h_get_stats(C.c_void_p(self._h), _dp(st), hist.ctypes.data_as(C.POINTER(C.c_longlong))), self.clusterid)
        wall = np.zeros(64)
        _chk(lib().g6h_get_force_wall_hist(C.c_void_p(self._h), _dp(wall)), self.clusterid)
        return dict(n_block_steps=int(st[0]), n_particle_steps=int(st[1]), t=st[2], dt_min=st[3], interactions=st[4],
                    wall_s=st[5], wall_force_s=st[6], ni_hist_log2=hist, force_wall_s_log2=wall)

    def close(self):
        if self._h:
            lib().g6h_destroy(C.c_void_p(self._h))
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class HermiteDev:
    """The device-resident Hermite block-step integrator (g6hd_* functions, include/g6_hermite.h): block
    selection, i-prediction, corrector and step choice are CUDA kernels; argument marshalling only here."""

    def __init__(self, clusterid, x, v, m, eps2, eta, eta_start=0.01, dt_max=0.125):
        n = len(m)
        x = _f64(x, (n, 3)); v = _f64(v, (n, 3)); m = _f64(m, (n,))
        self.n, self.clusterid = n, clusterid
        self._h = lib().g6hd_create(C.c_int(clusterid), C.c_int(n), _dp(x), _dp(v), _dp(m), C.c_double(eps2),
                                    C.c_double(eta), C.c_double(eta_start), C.c_double(dt_max))
        if not self._h:
            raise G6Error(-8, "g6hd_create failed: " + g6x_last_error(clusterid))

    def evolve(self, t_end, max_block_steps=0):
        return _chk(lib().g6hd_evolve(C.c_void_p(self._h), C.c_double(t_end), C.c_longlong(max_block_steps)), self.clusterid)

    def state(self):
        x = np.empty((self.n, 3)); v = np.empty((self.n, 3))
        _chk(lib().g6hd_get_state(C.c_void_p(self._h), _dp(x), _dp(v)), self.clusterid)
        return x, v

    def set_shared_steps(self, on=True):
        return _chk(lib().g6hd_set_shared_steps(C.c_void_p(self._h), C.c_int(1 if on else 0)), self.clusterid)

    def particles(self):
        """raw Hermite state, each particle at its own time: dict x, v, a, adot [n,3], t, dt [n]"""
        n = self.n
        o = dict(x=np.empty((n, 3)), v=np.empty((n, 3)), a=np.empty((n, 3)), adot=np.empty((n, 3)), t=np.empty(n), dt=np.empty(n))
        _chk(lib().g6hd_get_particles(C.c_void_p(self._h), _dp(o["x"]), _dp(o["v"]), _dp(o["a"]), _dp(o["adot"]), _dp(o["t"]), _dp(o["dt"])),
             self.clusterid)
        return o

    def last_block(self):
        """the last block step's i-block: dict act[ni], xi, vi, acc, jerk [ni,3]"""
        n = self.n
        ni = C.c_int(0)
        act = np.empty(n, np.int32); xi = np.empty((n, 3)); vi = np.empty((n, 3)); acc = np.empty((n, 3)); jerk = np.empty((n, 3))
        _chk(lib().g6hd_get_last_block(C.c_void_p(self._h), C.c_int(n), C.byref(ni), _ip(act), _dp(xi), _dp(vi), _dp(acc), _dp(jerk)), self.clusterid)
        k = ni.value
        return dict(act=act[:k].copy(), xi=xi[:k].copy(), vi=vi[:k].copy(), acc=acc[:k].copy(), jerk=jerk[:k].copy())

    def stats(self):
        st = np.zeros(8); hist = np.zeros(64, np.int64)
        _chk(lib().g6hd_get_stats(C.c_void_p(self._h), _dp(st), hist.ctypes.data_as(C.POINTER(C.c_longlong))), self.clusterid)
        return dict(n_block_steps=int(st[0]), n_particle_steps=int(st[1]), t=st[2], dt_min=st[3], interactions=st[4],
                    wall_s=st[5], ni_hist_log2=hist)

    def close(self):
        if self._h:
            lib().g6hd_destroy(C.c_void_p(self._h))
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
