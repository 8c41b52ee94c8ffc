"""The rest of the GRAPE-6 calling sequence through the C ABI on a live device:
j-particle read-back against what was stored, reset / flush / buffer calls, the nj-max query, on-demand growth of the
j-store, the Fortran-callable aliases, option validation."""
import ctypes as C

import numpy as np
import pytest

from helpers import check_forces, check_nn, load_j
from paper_0902_4463_b200 import g6, inputs

pytestmark = pytest.mark.gpu


@pytest.fixture()
def cluster():
    from paper_0902_4463_b200 import build
    build.build()
    g6.g6_open(0)
    yield 0
    g6.g6_close(0)
    g6.g6x_set_npipes(g6.DEFAULT_NPIPES)


def _f32(a):
    return np.asarray(a, np.float64).astype(np.float32).astype(np.float64)


def test_j_particle_readback_is_what_was_stored(cluster):
    """g6_get_j_particle / g6x_get_j_particles return the stored record: x and t exactly (fp64), m, v, acc/2, jerk/6 rounded
    to binary32 -- bit for bit, for particles set one by one, in bulk, overwritten, and not yet flushed."""
    rng = np.random.default_rng(11)
    n = 700                                              # three j-tiles, the last one ragged
    x = 1000.0 + rng.standard_normal((n, 3)); v = rng.standard_normal((n, 3))
    a = rng.standard_normal((n, 3)); j = 10 * rng.standard_normal((n, 3))
    m = rng.uniform(0.1, 1.0, n) / n; t = rng.integers(0, 64, n) / 1024.0
    idx = (np.arange(n, dtype=np.int32) * 7 + 3).astype(np.int32)
    g6.g6x_set_j_particles(0, 0, idx, t, m, j, a, v, x)
    got = g6.g6x_get_j_particles(0, 0, n)
    assert np.array_equal(got["index"], idx) and np.array_equal(got["x"], x) and np.array_equal(got["tj"], t)
    assert np.array_equal(got["mass"], _f32(m)) and np.array_equal(got["v"], _f32(v))
    assert np.array_equal(got["acc"], 2 * _f32(a / 2)) and np.array_equal(got["jerk"], 6 * _f32(j / 6))
    # one by one, pre-divided coefficients; an overwrite; read before any force call flushed the buffer
    p = 511
    g6.g6_set_j_particle(0, p, 99, 0.25, 0.125, 0.5, None, j[p] / 6, a[p] / 2, v[p], x[p] + 1.0)
    g6.g6_set_j_particle(0, p, 77, 0.5, 0.125, 0.75, None, j[0] / 6, a[0] / 2, v[0], x[0])
    one = g6.g6_get_j_particle(0, p)
    assert one["index"] == 77 and one["tj"] == 0.5 and one["mass"] == 0.75
    assert np.array_equal(one["x"], x[0]) and np.array_equal(one["v"], _f32(v[0]))
    assert np.array_equal(one["acc_by2"], _f32(a[0] / 2)) and np.array_equal(one["jerk_by6"], _f32(j[0] / 6))
    # neighbours of the overwritten slot are untouched
    again = g6.g6x_get_j_particles(0, p - 1, 3)
    assert np.array_equal(again["x"][[0, 2]], x[[p - 1, p + 1]]) and again["index"][1] == 77
    with pytest.raises(g6.G6Error) as e: g6.g6_get_j_particle(0, n)
    assert e.value.code == -3


def test_reset_flush_buffer_units_and_njmax(cluster, oracle):
    x, v, m, eps2 = inputs.config("C1", n=600)
    idx = load_j(x, v, m)
    g6.g6_set_ti(0, 0.0)
    ref = oracle.force(idx[:40], x[:40], v[:40], idx, x, v, m, eps2)
    check_forces(g6.force_host(0, idx[:40], x[:40], v[:40], eps2, 600), ref, "before reset")
    assert g6.g6_getnjmax(0) == 1 << 21                  # env G6_NJMAX default; the largest n_i is g6_npipes()
    assert g6.g6_set_tunit(51) == 0 and g6.g6_set_xunit(47) == 0 and g6.g6x_get_units() == (51, 47)
    assert g6.g6_reset_fofpga(0) == 0
    # reset forgets the particles: nj > 0 is refused until particles are stored again
    g6.g6calc_firsthalf(0, 600, 5, idx[:5], x[:5], v[:5], eps2=eps2)        # an unfinished call is dropped too
    g6.g6_reset(0)
    with pytest.raises(g6.G6Error) as e: g6.g6calc_firsthalf(0, 600, 5, idx[:5], x[:5], v[:5], eps2=eps2)
    assert e.value.code == -5
    # reload HALF the system one particle at a time through the buffer calls: the forces are those of the half system
    g6.g6_initialize_jp_buffer(0, 300)
    z = np.zeros(3)
    for p in range(300):
        g6.g6_set_j_particle(0, p, int(idx[p]), 0.0, 0.125, m[p], None, z, z, v[p], x[p])
    g6.g6_flush_jp_buffer(0)
    back = g6.g6x_get_j_particles(0, 0, 300)
    assert np.array_equal(back["x"], x[:300])
    half = oracle.force(idx[:40], x[:40], v[:40], idx[:300], x[:300], v[:300], m[:300], eps2)
    got = g6.force_host(0, idx[:40], x[:40], v[:40], eps2, 300)
    check_forces(got, half, "after reset")
    check_nn(got["nn_index"], half, idx[:300], x[:40], x[:300])


def test_j_store_grows_on_demand(cluster, oracle):
    """g6_open allocates for G6_NJINIT = 16384 addresses; setting higher addresses grows the device arrays and keeps what
    was stored."""
    x, v, m, eps2 = inputs.config("C1", n=40000)
    idx = np.arange(40000, dtype=np.int32)
    z3 = np.zeros((40000, 3))
    g6.g6x_set_j_particles(0, 0, idx[:10000], np.zeros(10000), m[:10000], z3[:10000], z3[:10000], v[:10000], x[:10000])
    z = np.zeros(3)
    for p in (16383, 16384, 39999, 20000):               # across the initial allocation, twice
        g6.g6_set_j_particle(0, p, p, 0.0, 0.125, m[p], None, z, z, v[p], x[p])
    g6.g6x_set_j_particles(0, 10000, idx[10000:], np.zeros(30000), m[10000:], z3[10000:], z3[10000:], v[10000:], x[10000:])
    back = g6.g6x_get_j_particles(0, 0, 40000)
    assert np.array_equal(back["x"], x) and np.array_equal(back["index"], idx)
    g6.g6_set_ti(0, 0.0)
    rows = np.array([0, 9999, 16384, 39999])
    ref = oracle.force(idx[rows], x[rows], v[rows], idx, x, v, m, eps2)
    check_forces(g6.force_host(0, idx[rows], x[rows], v[rows], eps2, 40000), ref, "grown store")


def test_fortran_aliases(cluster, oracle):
    """include/g6_fortran.h: trailing underscore, every argument by reference; same results as the C calls."""
    L = g6.lib()
    x, v, m, eps2 = inputs.config("C1", n=300)
    idx = np.arange(300, dtype=np.int32)
    ci = lambda k: C.byref(C.c_int(k)); cd = lambda k: C.byref(C.c_double(k))
    dp = lambda a: a.ctypes.data_as(C.POINTER(C.c_double)); ip = lambda a: a.ctypes.data_as(C.POINTER(C.c_int))
    assert L.g6_open_(ci(0)) == -9                       # already open (the fixture): the alias reports the same code
    assert L.g6_npipes_() == g6.g6_npipes()
    assert L.g6_reset_(ci(0)) == 0 and L.g6_reset_fofpga_(ci(0)) == 0
    assert L.g6_set_tunit_(ci(40)) == 0 and L.g6_set_xunit_(ci(41)) == 0 and g6.g6x_get_units() == (40, 41)
    assert L.g6_initialize_jp_buffer_(ci(0), ci(300)) == 0 and L.g6_getnjmax_(ci(0)) == 1 << 21
    z = np.zeros(3)
    for p in range(300):
        assert L.g6_set_j_particle_(ci(0), ci(p), ci(p), cd(0.0), cd(0.125), cd(m[p]), None, dp(z), dp(z), dp(np.ascontiguousarray(v[p])),
                                    dp(np.ascontiguousarray(x[p]))) == 0
    assert L.g6_flush_jp_buffer_(ci(0)) == 0
    xb = np.empty(3); mb = C.c_double(0); ib = C.c_int(0)
    assert L.g6_get_j_particle_(ci(0), ci(17), C.byref(ib), None, C.byref(mb), None, None, None, dp(xb)) == 0
    assert ib.value == 17 and np.array_equal(xb, x[17]) and mb.value == float(np.float32(m[17]))
    assert L.g6_set_ti_(ci(0), cd(0.0)) == 0
    ni = 20
    xi = np.ascontiguousarray(x[:ni]); vi = np.ascontiguousarray(v[:ni]); ii = np.ascontiguousarray(idx[:ni])
    h2 = np.full(ni, 0.05)
    assert L.g6calc_firsthalf_(ci(0), ci(300), ci(ni), ip(ii), dp(xi), dp(vi), None, None, None, cd(eps2), dp(h2)) == 0
    acc = np.empty((ni, 3)); jerk = np.empty((ni, 3)); pot = np.empty(ni); nn = np.empty(ni, np.int32)
    assert L.g6calc_lasthalf2_(ci(0), ci(300), ci(ni), ip(ii), dp(xi), dp(vi), cd(eps2), dp(h2), dp(acc), dp(jerk), dp(pot), ip(nn)) == 0
    ref = oracle.force(ii, xi, vi, idx, x, v, m, eps2)
    check_forces(dict(acc=acc, jerk=jerk, pot=pot), ref, "fortran aliases")
    check_nn(nn, ref, idx, xi, x)
    assert L.g6_read_neighbour_list_(ci(0)) == 0
    cnt = C.c_int(0); lst = np.empty(256, np.int32)
    assert L.g6_get_neighbour_list_(ci(0), ci(3), ci(256), C.byref(cnt), ip(lst)) == 0
    oc, ol = oracle.neighbours(ii, xi, h2, idx, x, maxlen=300)
    d2 = np.sum((x - xi[3]) ** 2, axis=1)
    sym = set(int(a) for a in lst[: cnt.value]) ^ set(int(a) for a in ol[3, : oc[3]])
    assert all(abs(d2[a] - h2[3]) <= 1e-6 * h2[3] for a in sym)
    assert L.g6calc_firsthalf_(ci(0), ci(300), ci(ni), ip(ii), dp(xi), dp(vi), None, None, None, cd(eps2), None) == 0
    assert L.g6calc_lasthalf_(ci(0), ci(300), ci(ni), ip(ii), dp(xi), dp(vi), cd(eps2), None, dp(acc), dp(jerk), dp(pot)) == 0
    assert L.g6_set_ti_(None, cd(0.0)) == -8             # a NULL reference is an argument error, not a crash


def test_option_values_are_validated(cluster):
    """the shapes option 'variant' accepts are exactly the built ones (anything else used to divide by zero later)"""
    for ok in (128 * 8 + 2, 128 * 8 + 1, 64 * 8 + 1, 32 * 8 + 1, 256 * 8 + 1, 128 * 8 + 4, 64 * 8 + 2, 0):
        g6.g6x_set_option(0, "variant", ok)
    for bad in (8, 3, 1, 7, 128 * 8, 128 * 8 + 3, 96 * 8 + 1, 256 * 8 + 2, 1 << 20):
        with pytest.raises(g6.G6Error) as e: g6.g6x_set_option(0, "variant", bad)
        assert e.value.code == -8, bad
    g6.g6x_set_option(0, "variant", 0)
