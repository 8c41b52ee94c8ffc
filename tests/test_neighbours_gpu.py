"""GPU parity of the neighbour lists (reading 20):
the CUDA path through the C ABI against oracle.neighbours on the same seeded inputs."""
import numpy as np
import pytest

from paper_0902_4463_b200 import g6, inputs
from helpers import check_forces, check_neighbours, check_nn, load_j

pytestmark = pytest.mark.gpu


@pytest.fixture()
def cluster():
    from paper_0902_4463_b200 import build
    build.build()
    g6.g6_open(0)
    g6.g6x_set_npipes(1 << 21)
    yield 0
    g6.g6_close(0)
    g6.g6x_set_npipes(g6.DEFAULT_NPIPES)


def radii(x, idx_i, seed, lo=0.2, hi=3.0):
    """h2 per i-particle: (lo..hi x the local mean spacing)^2, so that counts run from 0 to some tens"""
    rng = np.random.default_rng(seed)
    n = len(x)
    r = np.linalg.norm(x[idx_i], axis=1)
    a = 3 * np.pi / 16
    rho = 3 / (4 * np.pi * a ** 3) * (1 + (r / a) ** 2) ** -2.5 * n        # Plummer number density
    return (rng.uniform(lo, hi, len(idx_i)) * rho ** (-1.0 / 3)) ** 2


def run(idx_i, xi, vi, eps2, nj, h2, maxlen):
    got = g6.force_host(0, idx_i, xi, vi, eps2, nj, h2=h2)
    over = g6.g6_read_neighbour_list(0)
    cnt, lst, over2 = g6.g6x_get_neighbour_lists(0, len(idx_i), maxlen)
    assert over == int(np.sum(cnt > maxlen)) == over2
    return got, cnt, lst


@pytest.mark.parametrize("kernel", [0, 1, 2])
@pytest.mark.parametrize("jsplit", [0, 1, 3])
def test_c1_lists_every_particle(cluster, oracle, kernel, jsplit):
    x, v, m, eps2 = inputs.config("C1")
    n = len(m)
    idx = load_j(x, v, m)
    h2 = radii(x, idx, 5)
    g6.g6x_set_option(0, "kernel", kernel); g6.g6x_set_option(0, "jsplit", jsplit)
    g6.g6_set_ti(0, 0.0)
    got, cnt, lst = run(idx, x, v, eps2, n, h2, 256)
    oc, ol = oracle.neighbours(idx, x, h2, idx, x, maxlen=1024)
    assert oc.max() > 20 and (oc == 0).any()              # the recipe spans empty and well-filled lists
    nb = check_neighbours(cnt, lst, oc, ol, idx, x, x, h2, 256)
    # forces and nearest neighbour are unchanged by the list building
    ref = oracle.force(idx, x, v, idx, x, v, m, eps2)
    check_forces(got, ref, "C1 with lists"); check_nn(got["nn_index"], ref, idx, x, x)
    # the GRAPE-6 per-pipe call returns the same rows
    for i in (0, 5, 1023):
        row = g6.g6_get_neighbour_list(0, i, 256)
        assert list(row) == list(lst[i][lst[i] >= 0])
    print("C1 lists kernel", kernel, "jsplit", jsplit, "mean count", cnt.mean(), "max", cnt.max(), "borderline", nb)


@pytest.mark.parametrize("kernel", [1, 2])
def test_overflow_rule(cluster, oracle, kernel):
    x, v, m, eps2 = inputs.config("C1", n=3000)
    n = len(m)
    idx = load_j(x, v, m)
    h2 = radii(x, idx, 6, lo=1.0, hi=4.0)
    g6.g6x_set_option(0, "kernel", kernel); g6.g6x_set_option(0, "nb_maxlen", 8)
    g6.g6_set_ti(0, 0.0)
    got, cnt, lst = run(idx, x, v, eps2, n, h2, 8)
    oc, ol = oracle.neighbours(idx, x, h2, idx, x, maxlen=n)
    assert (oc > 8).sum() > 100 and (oc <= 8).sum() > 100
    check_neighbours(cnt, lst, oc, ol, idx, x, x, h2, 8)
    assert g6.g6_read_neighbour_list(0) == int((cnt > 8).sum()) > 0
    # per-pipe call: 1 = neighbours dropped
    i = int(np.argmax(cnt))
    n_out = g6.lib().g6_get_neighbour_list
    import ctypes as C
    nn = C.c_int(0); buf = (C.c_int * 8)()
    assert n_out(0, i, 8, C.byref(nn), buf) == 1 and nn.value == 8
    g6.g6x_set_option(0, "nb_maxlen", 256)


@pytest.mark.parametrize("n,ni", [(4097, 130), (1000, 1), (257, 257), (5000, 3), (70000, 40)])
def test_ragged_small_blocks_and_extremes(cluster, oracle, n, ni):
    x, v, m, eps2 = inputs.config("C1", n=n)
    idx = load_j(x, v, m)
    sel = inputs.active_subset(n, ni, 99 + ni)
    h2 = radii(x, sel, 7)
    h2[0] = 0.0                    # nothing is inside an empty sphere
    if ni > 2:
        h2[1] = 1e6                # everything but the particle itself is inside this one: overflow
    g6.g6_set_ti(0, 0.0)
    got, cnt, lst = run(idx[sel], x[sel], v[sel], eps2, n, h2, 256)
    oc, ol = oracle.neighbours(idx[sel], x[sel], h2, idx, x, maxlen=max(n, 256))
    check_neighbours(cnt, lst, oc, ol, idx, x[sel], x, h2, 256)
    assert cnt[0] == 0
    if ni > 2:
        assert cnt[1] == n - 1
    ref = oracle.force(idx[sel], x[sel], v[sel], idx, x, v, m, eps2)
    check_forces(got, ref, f"lists n={n} ni={ni}"); check_nn(got["nn_index"], ref, idx, x[sel], x)


def test_lists_with_ti_not_tj_and_foreign_indices(cluster, oracle):
    """i-particles that are also j-particles, predicted to a later time on both sides: the self pair
    must stay out of the list although its separation is not zero (reading 4)."""
    n, ni = 6000, 200
    x, v, m, eps2 = inputs.config("C1", n=n)
    tj, dtj, a0, j0 = inputs.taylor_state(n, 31)
    index = (np.arange(n, dtype=np.int32) * 7 + 3).astype(np.int32)           # ids are not addresses
    g6.g6x_set_j_particles(0, 0, index, tj, m, j0, a0, v, x)
    ti = 0.0625
    g6.g6_set_ti(0, ti)
    xp, vp = oracle.predict(ti, tj, x, v, a0, j0)
    sel = inputs.active_subset(n, ni, 12)
    h2 = radii(x, sel, 8, lo=0.5, hi=2.5)
    got, cnt, lst = run(index[sel], xp[sel], vp[sel], eps2, n, h2, 256)
    oc, ol = oracle.neighbours(index[sel], xp[sel], h2, index, xp, maxlen=n)
    # predicted positions differ by the FP32 Taylor increment: widen the borderline band accordingly
    check_neighbours(cnt, lst, oc, ol, index, xp[sel], xp, h2, 256, tol=1e-4)
    for k in range(ni):
        assert index[sel[k]] not in lst[k]


def test_c4_size_device_entry_sampled_block(cluster, oracle):
    """BASELINE.json's full size (N = 2^20) in the launch shape bench.py times: a 4096-block through
    g6x_calc_dev_nb, every row against the oracle."""
    import torch
    x, v, m, eps2 = inputs.config("C4")
    n = len(m)
    idx = np.arange(n, dtype=np.int32)
    dev = torch.device("cuda:0")
    t = lambda a, dt=torch.float64: torch.from_numpy(np.ascontiguousarray(a)).to(dev, dt)
    z3 = torch.zeros(n, 3, dtype=torch.float64, device=dev)
    g6.g6x_set_j_particles_dev(0, 0, n, t(idx, torch.int32), torch.zeros(n, dtype=torch.float64, device=dev), t(m), z3, z3, t(v), t(x))
    g6.g6_set_ti(0, 0.0)
    ni = 4096
    sel = inputs.active_subset(n, ni, 4040 + ni)
    h2 = radii(x, sel, 9, lo=0.3, hi=3.5)
    acc = torch.empty(ni, 3, dtype=torch.float64, device=dev); jerk = torch.empty_like(acc)
    pot = torch.empty(ni, dtype=torch.float64, device=dev); nn = torch.empty(ni, dtype=torch.int32, device=dev); r2 = torch.empty_like(pot)
    cnt = torch.zeros(ni, dtype=torch.int32, device=dev); lst = torch.full((ni, 256), -1, dtype=torch.int32, device=dev)
    g6.g6x_calc_dev_nb(0, n, ni, t(idx[sel], torch.int32), t(x[sel]), t(v[sel]), eps2, acc, jerk, pot, nn, r2, t(h2), cnt, lst)
    g6.g6x_synchronize(0)
    oc, ol = oracle.neighbours(idx[sel], x[sel], h2, idx, x, maxlen=8192)
    nb = check_neighbours(cnt.cpu().numpy(), lst.cpu().numpy(), oc, ol, idx, x[sel], x, h2, 256)
    ref = oracle.force(idx[sel], x[sel], v[sel], idx, x, v, m, eps2)
    got = dict(acc=acc.cpu().numpy(), jerk=jerk.cpu().numpy(), pot=pot.cpu().numpy())
    check_forces(got, ref, "C4 4096-block with lists")
    print("C4 lists: mean count", oc.mean(), "max", oc.max(), "borderline", nb)


def test_neighbour_abi_errors_and_maxlen_change(cluster, oracle):
    import ctypes as C
    x, v, m, eps2 = inputs.config("C1", n=600)
    n = len(m)
    idx = load_j(x, v, m)
    g6.g6_set_ti(0, 0.0)
    # a call without h2 builds no lists: the bulk getter refuses, the per-pipe getter returns the nearest neighbour
    got = g6.force_host(0, idx, x, v, eps2, n)
    assert g6.g6_read_neighbour_list(0) == 0
    with pytest.raises(g6.G6Error) as e:
        g6.g6x_get_neighbour_lists(0, n, 16)
    assert e.value.code == -6
    assert list(g6.g6_get_neighbour_list(0, 3, 4)) == [got["nn_index"][3]]
    # bad option values
    for bad in (0, 5000):
        with pytest.raises(g6.G6Error) as e:
            g6.g6x_set_option(0, "nb_maxlen", bad)
        assert e.value.code == -8
    # the three neighbour pointers of the device entry go together
    import torch
    d = torch.zeros(8, dtype=torch.float64, device="cuda:0")
    L = g6.lib()
    rc = L.g6x_calc_dev_nb(0, n, 1, C.c_void_p(d.data_ptr()), C.c_void_p(d.data_ptr()), C.c_void_p(d.data_ptr()), C.c_double(eps2),
                           C.c_void_p(d.data_ptr()), C.c_void_p(d.data_ptr()), C.c_void_p(d.data_ptr()), None, None,
                           C.c_void_p(d.data_ptr()), None, None)
    assert rc == -8
    # lists, then a different nb_maxlen: the old lists are gone (error), a new call works with the new length
    h2 = radii(x, idx, 3, lo=1.0, hi=2.0)
    run(idx, x, v, eps2, n, h2, 256)
    g6.g6x_set_option(0, "nb_maxlen", 4)
    got2, cnt, lst = run(idx, x, v, eps2, n, h2, 4)
    oc, ol = oracle.neighbours(idx, x, h2, idx, x, maxlen=n)
    check_neighbours(cnt, lst, oc, ol, idx, x, x, h2, 4)
    # caller's buffer shorter than the stored list: truncated, return value 1
    i = int(np.argmax(cnt))
    nn = C.c_int(0); buf = (C.c_int * 2)()
    assert L.g6_get_neighbour_list(0, i, 2, C.byref(nn), buf) == 1 and nn.value == 2
    assert [buf[0], buf[1]] == list(lst[i][:2])
    g6.g6x_set_option(0, "nb_maxlen", 256)


@pytest.mark.parametrize("n,ni,small", [(5000, 1, 32), (5000, 7, 32), (3000, 16, 32), (70000, 32, 32), (900, 64, 64), (300, 33, 64)])
def test_small_blocks_lists_from_the_block_step_kernel(cluster, oracle, n, ni, small):
    """n_i <= `small`: lists come from the fused block-step kernel (per-warp lists merged by address in its last CTA);
    the same call with the kernel switched off (sweep path) must give identical lists."""
    x, v, m, eps2 = inputs.config("C1", n=n)
    tj, dtj, a0, j0 = inputs.taylor_state(n, 41)
    index = (np.arange(n, dtype=np.int32) * 3 + 1).astype(np.int32)
    g6.g6x_set_j_particles(0, 0, index, tj, m, j0, a0, v, x)
    ti = 0.03125
    g6.g6_set_ti(0, ti)
    xp, vp = oracle.predict(ti, tj, x, v, a0, j0)
    sel = inputs.active_subset(n, ni, 7 + ni)
    h2 = radii(x, sel, 10, lo=0.5, hi=3.0)
    if ni > 2:
        h2[1] = 1e6                                # overflow: everybody is a neighbour
    h2[0] = 0.0
    g6.g6x_set_option(0, "small", small)
    got, cnt, lst = run(index[sel], xp[sel], vp[sel], eps2, n, h2, 256)
    assert g6.g6x_get_option(0, "last_kernel") == 3          # the block-step kernel served it
    oc, ol = oracle.neighbours(index[sel], xp[sel], h2, index, xp, maxlen=max(n, 256))
    check_neighbours(cnt, lst, oc, ol, index, xp[sel], xp, h2, 256, tol=1e-4)
    assert cnt[0] == 0
    if ni > 2:
        assert cnt[1] == n - 1 and (lst[1] >= 0).sum() == min(256, n - 1)
    ref = oracle.force(index[sel], xp[sel], vp[sel], index, xp, vp, m, eps2)
    assert np.abs(got["pot"] - ref["pot"]).max() / np.abs(ref["pot"]).max() < 1e-5
    g6.g6x_set_option(0, "small", 0)               # the sweep kernels on the same call
    got2, cnt2, lst2 = run(index[sel], xp[sel], vp[sel], eps2, n, h2, 256)
    assert g6.g6x_get_option(0, "last_kernel") == 2
    assert np.array_equal(cnt, cnt2) and np.array_equal(lst, lst2)
    g6.g6x_set_option(0, "small", 32)


@pytest.mark.parametrize("n,ni", [(5000, 5), (3000, 16), (40000, 32)])
def test_production_cycle_with_lists_and_inline_j_updates(cluster, oracle, n, ni):
    """The Hermite cycle with neighbour lists: g6_set_j_particle for the corrected particles (they ride in the launch of the
    block-step kernel), then firsthalf with h2 / lasthalf / read_neighbour_list; lists see the UPDATED positions and agree
    with the sweep kernels' lists for the same call."""
    from helpers import rel_err
    x, v, m, _ = inputs.config("C2", n=n)
    eps2 = 1e-8
    rng = np.random.default_rng(500 + ni)
    idx = rng.permutation(n).astype(np.int32)
    tj, dtj, a0, j0 = inputs.taylor_state(n, 300 + ni, dt_max=2.0**-6)
    load_j(x, v, m, index=idx, t=tj, acc=a0, jerk=j0)
    g6.g6x_set_option(0, "small", 32)
    t = 2.0**-8
    for step in range(3):
        blk = np.append(np.sort(rng.choice(n - 1, ni - 1, replace=False)), n - 1).astype(int)
        x[blk] += 1e-3 * rng.standard_normal((ni, 3)); v[blk] += 1e-3 * rng.standard_normal((ni, 3))
        a0[blk] = rng.standard_normal((ni, 3)); j0[blk] = rng.standard_normal((ni, 3)); tj[blk] = t
        for p in blk:
            g6.g6_set_j_particle(0, int(p), int(idx[p]), tj[p], dtj[p], m[p], None, j0[p] / 6, a0[p] / 2, v[p], x[p])
        t += 2.0**-9
        g6.g6_set_ti(0, t)
        xo, vo = oracle.predict(t, tj, x, v, a0, j0)
        nxt = np.sort(rng.choice(n, ni, replace=False))
        nxt[0] = blk[0]
        h2 = radii(x, nxt, 600 + step, lo=0.5, hi=2.5)
        got, cnt, lst = run(idx[nxt], xo[nxt], vo[nxt], eps2, n, h2, 256)
        assert g6.g6x_get_option(0, "last_kernel") == 3
        oc, ol = oracle.neighbours(idx[nxt], xo[nxt], h2, idx, xo, maxlen=n)
        check_neighbours(cnt, lst, oc, ol, idx, xo[nxt], xo, h2, 256, tol=1e-4)
        ref = oracle.force(idx[nxt], xo[nxt], vo[nxt], idx, xo, vo, m, eps2)
        assert rel_err(got["acc"], ref["acc"]).max() <= 1e-5 and rel_err(got["pot"], ref["pot"]).max() <= 1e-6
        g6.g6x_set_option(0, "kernel", 2)
        got2, cnt2, lst2 = run(idx[nxt], xo[nxt], vo[nxt], eps2, n, h2, 256)
        g6.g6x_set_option(0, "kernel", 0)
        assert np.array_equal(cnt, cnt2) and np.array_equal(lst, lst2)
