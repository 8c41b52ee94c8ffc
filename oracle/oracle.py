"""ctypes front end of the CPU oracle (oracle/*.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this module.  It imports nothing from the CUDA package and the CUDA package
imports nothing from here.  No arithmetic of the method lives in this file: it compiles
the C sources with gcc (no -ffast-math, -ffp-contract=off) and marshals numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_BUILD = os.path.join(_HERE, "build")
_SOURCES = ["g6_oracle.c", "hermite_oracle.c"]
CFLAGS = ["-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-ffp-contract=off", "-fno-fast-math"]
_lock = threading.Lock()
_libs: dict = {}


def build(long_double: bool = False, force: bool = False) -> str:
    """Compile oracle/*.c into oracle/build/liboracle[_ld].so (rebuilt when a source is newer)."""
    os.makedirs(_BUILD, exist_ok=True)
    out = os.path.join(_BUILD, "liboracle_ld.so" if long_double else "liboracle.so")
    srcs = [os.path.join(_HERE, s) for s in _SOURCES if os.path.exists(os.path.join(_HERE, s))]
    stale = force or not os.path.exists(out) or any(
        os.path.getmtime(s) > os.path.getmtime(out) for s in srcs)
    if stale:
        cmd = ["gcc"] + CFLAGS + (["-DORC_LONG_DOUBLE"] if long_double else []) + srcs + ["-o", out + ".tmp", "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(out + ".tmp", out)
    return out


def _lib(long_double: bool = False):
    with _lock:
        if long_double not in _libs:
            _libs[long_double] = C.CDLL(build(long_double))
        return _libs[long_double]


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def _f64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        assert a.shape == shape, (a.shape, shape)
    return a


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def threads() -> int:
    """Number of OpenMP threads the oracle will use (OMP_NUM_THREADS or all cores)."""
    v = os.environ.get("OMP_NUM_THREADS")
    return int(v) if v else (os.cpu_count() or 1)


def predict(ti, tj, x0, v0, a0, j0, long_double=False):
    """Eq. 1-2.  Returns (x_pred, v_pred) as fp64 [n,3]."""
    n = len(tj)
    tj = _f64(tj, (n,)); x0 = _f64(x0, (n, 3)); v0 = _f64(v0, (n, 3))
    a0 = _f64(a0, (n, 3)); j0 = _f64(j0, (n, 3))
    xp = np.empty((n, 3)); vp = np.empty((n, 3))
    d = C.c_double
    _lib(long_double).orc_predict(C.c_int(n), d(float(ti)), _p(tj, d), _p(x0, d), _p(v0, d),
                                  _p(a0, d), _p(j0, d), _p(xp, d), _p(vp, d))
    return xp, vp


def force(index_i, xi, vi, index_j, xj, vj, mj, eps2, long_double=False):
    """Direct sum over all j with index_j != index_i.  Returns a dict with
    acc[ni,3], jerk[ni,3], pot[ni], nn_addr[ni], nn_index[ni], nn_r2[ni]."""
    ni, nj = len(index_i), len(index_j)
    index_i = _i32(index_i); index_j = _i32(index_j)
    xi = _f64(xi, (ni, 3)); vi = _f64(vi, (ni, 3))
    xj = _f64(xj, (nj, 3)); vj = _f64(vj, (nj, 3)); mj = _f64(mj, (nj,))
    acc = np.empty((ni, 3)); jerk = np.empty((ni, 3)); pot = np.empty(ni)
    nn_addr = np.empty(ni, np.int32); nn_index = np.empty(ni, np.int32); nn_r2 = np.empty(ni)
    d, i = C.c_double, C.c_int
    _lib(long_double).orc_force(i(ni), _p(index_i, i), _p(xi, d), _p(vi, d),
                                i(nj), _p(index_j, i), _p(xj, d), _p(vj, d), _p(mj, d), d(float(eps2)),
                                _p(acc, d), _p(jerk, d), _p(pot, d),
                                _p(nn_addr, i), _p(nn_index, i), _p(nn_r2, d))
    return dict(acc=acc, jerk=jerk, pot=pot, nn_addr=nn_addr, nn_index=nn_index, nn_r2=nn_r2)


def neighbours(index_i, xi, h2, index_j, xj, maxlen=256, long_double=False):
    """Neighbour lists (orc_neighbours): (count[ni], list_addr[ni, maxlen]); entries past
    min(count, maxlen) are -1.  j addresses in increasing order."""
    ni, nj = len(index_i), len(index_j)
    index_i = _i32(index_i); index_j = _i32(index_j)
    xi = _f64(xi, (ni, 3)); xj = _f64(xj, (nj, 3)); h2 = _f64(h2, (ni,))
    count = np.zeros(ni, np.int32); lst = np.full((ni, maxlen), -1, np.int32)
    d, i = C.c_double, C.c_int
    _lib(long_double).orc_neighbours(i(ni), _p(index_i, i), _p(xi, d), _p(h2, d), i(nj), _p(index_j, i), _p(xj, d),
                                     i(maxlen), _p(count, i), _p(lst, i))
    return count, lst


def energy(x, v, m, eps2, long_double=False):
    """(T, W): kinetic and softened potential energy."""
    n = len(m)
    x = _f64(x, (n, 3)); v = _f64(v, (n, 3)); m = _f64(m, (n,))
    T = C.c_double(); W = C.c_double()
    d = C.c_double
    _lib(long_double).orc_energy(C.c_int(n), _p(x, d), _p(v, d), _p(m, d), d(float(eps2)),
                                 C.byref(T), C.byref(W))
    return T.value, W.value


def ds_split(x):
    """double -> (hi, lo) binary32 pair (reading 12)."""
    x = _f64(x).ravel()
    hi = np.empty(x.size, np.float32); lo = np.empty(x.size, np.float32)
    _lib().orc_ds_split(C.c_int(x.size), _p(x, C.c_double), _p(hi, C.c_float), _p(lo, C.c_float))
    return hi, lo


def ds_diff(xj_hi, xj_lo, xi_hi, xi_lo):
    """Eq. 3 in binary32."""
    a = [np.ascontiguousarray(t, dtype=np.float32).ravel() for t in (xj_hi, xj_lo, xi_hi, xi_lo)]
    n = a[0].size
    out = np.empty(n, np.float32)
    f = C.c_float
    _lib().orc_ds_diff(C.c_int(n), _p(a[0], f), _p(a[1], f), _p(a[2], f), _p(a[3], f), _p(out, f))
    return out


class HermiteResult(dict):
    __getattr__ = dict.__getitem__


def hermite(x, v, m, eps2, eta, t_end, dt_max=0.125, eta_start=0.01, max_steps=0, shared=False):
    """Oracle-driven 4th-order Hermite block-step integration (oracle/hermite_oracle.c); shared=True:
    one common step for all particles.  Returns the final synchronised state and step statistics."""
    n = len(m)
    x = _f64(x, (n, 3)).copy(); v = _f64(v, (n, 3)).copy(); m = _f64(m, (n,))
    hist = np.zeros(64, np.int64)
    stats = np.zeros(8, np.float64)
    d = C.c_double
    lib = _lib()
    fn = lib.orc_hermite_shared if shared else lib.orc_hermite
    fn.restype = C.c_int
    rc = fn(C.c_int(n), _p(x, d), _p(v, d), _p(m, d), d(float(eps2)), d(float(eta)),
                         d(float(eta_start)), d(float(dt_max)), d(float(t_end)),
                         C.c_longlong(int(max_steps)), _p(hist, C.c_longlong), _p(stats, d))
    if rc != 0:
        raise RuntimeError(f"orc_hermite failed rc={rc}")
    return HermiteResult(x=x, v=v, n_block_steps=int(stats[0]), n_particle_steps=int(stats[1]),
                         t=float(stats[2]), dt_min=float(stats[3]), interactions=float(stats[4]),
                         ni_hist_log2=hist)


def hermite_correct(h, xp, vp, a0, ad0, a1, ad1):
    """One particle's corrector (oracle/hermite_oracle.c).  Returns x1, v1, a2_new, a3."""
    d = C.c_double
    arrs = [_f64(t, (3,)) for t in (xp, vp, a0, ad0, a1, ad1)]
    outs = [np.empty(3) for _ in range(4)]
    _lib().orc_hermite_correct(d(float(h)), *[_p(t, d) for t in arrs], *[_p(t, d) for t in outs])
    return outs


def aarseth_dt(eta, a1, ad1, a2n, a3, dt_max=0.125):
    d = C.c_double
    lib = _lib()
    lib.orc_aarseth_dt.restype = d
    arrs = [_f64(t, (3,)) for t in (a1, ad1, a2n, a3)]
    return lib.orc_aarseth_dt(d(float(eta)), *[_p(t, d) for t in arrs], d(float(dt_max)))
