"""Seeded random force calls and block-step cycles against the oracle: sizes, block sizes, kernels, options, indices that differ from the
addresses, j-particles at their own times (Eq. 1-2 on the device), neighbour lists, j-particle updates between calls.  The fixed cases of
test_parity_gpu.py pin the configurations of BASELINE.json; these walk the space between them (a longer walk of the same generators, and
of the step loop against the path without it, was run once with other seeds: 60 + 40 + 36 cases, no disagreement)."""
import numpy as np
import pytest

from paper_0902_4463_b200 import g6, inputs
from helpers import check_forces, check_neighbours, check_nn

pytestmark = pytest.mark.gpu


@pytest.fixture()
def cluster():
    from paper_0902_4463_b200 import build
    build.build()
    g6.g6_open(0)
    yield 0
    for key in ("kernel", "bs_design"):
        g6.g6x_set_option(0, key, 0)
    g6.g6x_set_option(0, "newton", 1)
    g6.g6_close(0)
    g6.g6x_set_npipes(g6.DEFAULT_NPIPES)


def _system(rng, nj):
    x, v, m, _ = inputs.config("C2", n=max(nj, 2))
    x, v, m = x[:nj].copy(), v[:nj].copy(), m[:nj] / m[:nj].sum()
    tj, _dtj, a0, j0 = inputs.taylor_state(nj, seed=int(rng.integers(1 << 30)))
    return x, v, m, tj, 1e-2 * a0, 1e-2 * j0, rng.permutation(nj).astype(np.int32)


@pytest.mark.parametrize("seed", [101, 202, 303])
def test_random_force_calls(cluster, oracle, seed):
    rng = np.random.default_rng(seed)
    kernels = set()
    for case in range(10):
        nj = int(rng.choice([rng.integers(1, 300), rng.integers(300, 3000), rng.integers(3000, 30000)]))
        ni = int(min(nj, rng.choice([1, 2, 3, 7, 16, 17, 31, 33, 40, 64, 65, 100, 255, 256, 257, 600, 2500])))
        eps2 = float(rng.choice([1e-2, 1e-3, 1e-4])) ** 2
        kernel, bsd, newton = int(rng.choice([0, 0, 0, 1, 2])), int(rng.choice([0, 1, 2])), int(rng.choice([1, 1, 0]))
        with_lists = bool(rng.random() < 0.3)
        x, v, m, tj, a0, j0, idx = _system(rng, nj)
        ti = float(tj.max() + 2.0 ** -7)
        g6.g6x_set_option(0, "kernel", kernel); g6.g6x_set_option(0, "bs_design", bsd); g6.g6x_set_option(0, "newton", newton)
        g6.g6x_set_npipes(max(ni, 4096))
        g6.g6_reset(0)
        g6.g6x_set_j_particles(0, 0, idx, tj, m, j0, a0, v, x)
        g6.g6_set_ti(0, ti)
        sel = np.sort(rng.choice(nj, ni, replace=False))
        xp, vp = oracle.predict(ti, tj, x, v, a0, j0)
        h2 = np.full(ni, float(rng.choice([0.01, 0.05]))) if with_lists else None
        got = g6.force_host(0, idx[sel], xp[sel], vp[sel], eps2, nj, h2=h2)
        kernels.add(g6.g6x_get_option(0, "last_kernel"))
        what = f"seed {seed} case {case}: nj {nj} ni {ni} kernel {kernel} design {bsd} newton {newton} lists {with_lists}"
        if nj > 1:
            ref = oracle.force(idx[sel], xp[sel], vp[sel], idx, xp, vp, m, eps2)
            check_forces(got, ref, what=what)
            check_nn(got["nn_index"], ref, idx, xp[sel], xp)
        if with_lists:
            g6.g6_read_neighbour_list(0)
            cnt, lst, _ = g6.g6x_get_neighbour_lists(0, ni, 256)
            oc, ol = oracle.neighbours(idx[sel], xp[sel], h2, idx, xp, maxlen=max(nj, 1))
            check_neighbours(cnt, lst, oc, ol, idx, xp[sel], xp, h2, 256)
    assert kernels >= {2, 3}, kernels          # the walk met the sweep kernel and the block-step kernel


@pytest.mark.parametrize("seed", [11, 22])
def test_random_block_step_cycles_with_j_updates(cluster, oracle, seed):
    """force call -> the block's particles get a new state through g6_set_j_particle, one by one (the GRAPE-6 way) -> next call at a
    later time: the changed records ride in the next small-block launch (a-1) and must take effect"""
    rng = np.random.default_rng(seed)
    for case in range(6):
        nj = int(rng.choice([rng.integers(2, 300), rng.integers(300, 5000), rng.integers(5000, 80000)]))
        eps2 = float(rng.choice([1e-2, 1e-3, 1e-4])) ** 2
        x, v, m, tj, a0, j0, idx = _system(rng, nj)
        g6.g6x_set_option(0, "bs_design", int(rng.choice([0, 1, 2]))); g6.g6x_set_option(0, "newton", int(rng.choice([1, 1, 0])))
        g6.g6x_set_npipes(4096)
        g6.g6_reset(0)
        g6.g6x_set_j_particles(0, 0, idx, tj, m, j0, a0, v, x)
        ti = float(tj.max())
        for cyc in range(4):
            ti += 2.0 ** -int(rng.integers(6, 12))
            ni = int(min(nj, rng.choice([1, 2, 5, 16, 24, 32, 33, 48, 64, 100])))
            sel = np.sort(rng.choice(nj, ni, replace=False))
            g6.g6_set_ti(0, ti)
            xp, vp = oracle.predict(ti, tj, x, v, a0, j0)
            got = g6.force_host(0, idx[sel], xp[sel], vp[sel], eps2, nj)
            ref = oracle.force(idx[sel], xp[sel], vp[sel], idx, xp, vp, m, eps2)
            check_forces(got, ref, what=f"seed {seed} case {case} cycle {cyc}: nj {nj} ni {ni}")
            check_nn(got["nn_index"], ref, idx, xp[sel], xp)
            for a in sel:
                x[a] = xp[a] + 1e-6 * rng.normal(size=3); v[a] = vp[a]; tj[a] = ti
                a0[a] = 1e-2 * rng.normal(size=3); j0[a] = 1e-1 * rng.normal(size=3)
                g6.g6_set_j_particle(0, int(a), int(idx[a]), ti, 2.0 ** -8, m[a], None, j0[a] / 6, a0[a] / 2, v[a], x[a])


def test_random_neighbour_lists_with_overflow(cluster, oracle):
    """radii from a few neighbours to a large part of the cluster, list lengths from 4 to 1024: counts, stored entries (the smallest
    addresses on overflow) and their order against the oracle, through every kernel that builds lists"""
    rng = np.random.default_rng(9090)
    overflowed = 0
    try:
        for case in range(12):
            nj = int(rng.choice([rng.integers(2, 500), rng.integers(500, 6000), rng.integers(6000, 40000)]))
            ni = int(min(nj, rng.choice([1, 3, 16, 32, 33, 64, 65, 200, 256, 300, 1000])))
            maxlen = int(rng.choice([4, 8, 64, 256, 1024]))
            g6.g6x_set_option(0, "kernel", int(rng.choice([0, 0, 1, 2]))); g6.g6x_set_option(0, "bs_design", int(rng.choice([0, 1, 2])))
            g6.g6x_set_option(0, "nb_maxlen", maxlen)
            g6.g6x_set_npipes(max(ni, 4096))
            x, v, m, _ = inputs.config("C2", n=max(nj, 2))
            x, v, m = x[:nj].copy(), v[:nj].copy(), m[:nj] / m[:nj].sum()
            idx = rng.permutation(nj).astype(np.int32)
            z = np.zeros((nj, 3))
            g6.g6_reset(0)
            g6.g6x_set_j_particles(0, 0, idx, np.zeros(nj), m, z, z, v, x)
            g6.g6_set_ti(0, 0.0)
            sel = np.sort(rng.choice(nj, ni, replace=False))
            h2 = 10.0 ** rng.uniform(-3.5, -0.3, ni)
            g6.force_host(0, idx[sel], x[sel], v[sel], 1e-6, nj, h2=h2)
            g6.g6_read_neighbour_list(0)
            cnt, lst, _ = g6.g6x_get_neighbour_lists(0, ni, maxlen)
            oc, ol = oracle.neighbours(idx[sel], x[sel], h2, idx, x, maxlen=nj)
            check_neighbours(cnt, lst, oc, ol, idx, x[sel], x, h2, maxlen)
            overflowed += int((oc > maxlen).sum())
    finally:
        g6.g6x_set_option(0, "nb_maxlen", 256)
    assert overflowed > 0
