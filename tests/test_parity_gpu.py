"""GPU parity: the CUDA path, called through the C ABI, against the fp64 oracle on the same
seeded inputs, element by element (small sizes) or on sampled rows (BASELINE.json sizes)."""
import numpy as np
import pytest

from paper_0902_4463_b200 import g6, inputs
from helpers import (TOL_NN_TIE, check_forces, check_nn, load_j, rel_err)

pytestmark = pytest.mark.gpu


@pytest.fixture()
def cluster():
    from paper_0902_4463_b200 import build
    build.build()
    g6.g6_open(0)
    g6.g6x_set_npipes(1 << 21)
    g6.g6x_set_option(0, "timers", 1)          # off by default (two event records per phase cost ~10 us a step)
    yield 0
    g6.g6_close(0)
    g6.g6x_set_npipes(g6.DEFAULT_NPIPES)


KERNELS = [0, 1, 2]       # 0 = automatic (block-step kernel for n_i <= 32), 1 = checked reference kernel, 2 = fast kernel (FFMA2 + TMA)


# ------------------------------------------------------------------ C1: every particle
@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("newton", [1, 0])
def test_c1_full_parity(cluster, oracle, kernel, newton):
    x, v, m, eps2 = inputs.config("C1")
    idx = load_j(x, v, m)
    g6.g6x_set_option(0, "kernel", kernel); g6.g6x_set_option(0, "newton", newton)
    g6.g6_set_ti(0, 0.0)
    got = g6.force_host(0, idx, x, v, eps2, len(m))
    ref = oracle.force(idx, x, v, idx, x, v, m, eps2)
    st = check_forces(got, ref, f"C1 kernel={kernel} newton={newton}")
    check_nn(got["nn_index"], ref, idx, x, x)
    assert np.allclose(got["nn_r2"], ref["nn_r2"], rtol=1e-5)
    # neighbour-list calls of the GRAPE-6 sequence
    assert g6.g6_read_neighbour_list(0) == 0
    for i in (0, 17, 1023):
        assert list(g6.g6_get_neighbour_list(0, i, 4)) == [got["nn_index"][i]]
    print("C1", kernel, newton, st)


# ------------------------------------------------------------------ device entry == host entry
@pytest.mark.parametrize("kernel", KERNELS)
def test_device_entry_matches_host_entry_bitwise(cluster, kernel):
    import torch
    x, v, m, eps2 = inputs.config("C1", n=3000)
    n = len(m)
    g6.g6x_set_option(0, "kernel", kernel)
    idx = load_j(x, v, m)
    g6.g6_set_ti(0, 0.0)
    host = g6.force_host(0, idx, x, v, eps2, n)
    dev = torch.device("cuda:0")
    t = lambda a, dt=torch.float64: torch.from_numpy(np.ascontiguousarray(a)).to(dev, dt)
    z3 = torch.zeros(n, 3, dtype=torch.float64, device=dev)
    g6.g6x_set_j_particles_dev(0, 0, n, t(idx, torch.int32), torch.zeros(n, dtype=torch.float64, device=dev), t(m), z3, z3, t(v), t(x))
    acc = torch.empty(n, 3, dtype=torch.float64, device=dev); jerk = torch.empty_like(acc)
    pot = torch.empty(n, dtype=torch.float64, device=dev); nn = torch.empty(n, dtype=torch.int32, device=dev); r2 = torch.empty_like(pot)
    g6.g6x_calc_dev(0, n, n, t(idx, torch.int32), t(x), t(v), eps2, acc, jerk, pot, nn, r2)
    g6.g6x_synchronize(0)
    assert np.array_equal(acc.cpu().numpy(), host["acc"]) and np.array_equal(jerk.cpu().numpy(), host["jerk"])
    assert np.array_equal(pot.cpu().numpy(), host["pot"]) and np.array_equal(nn.cpu().numpy(), host["nn_index"])
    assert np.array_equal(r2.cpu().numpy(), host["nn_r2"])


# ------------------------------------------------------------------ predictor (Eq. 1-2)
def test_predictor_parity(cluster, oracle):
    n = 5000                                          # 19 full tiles + a ragged one
    x, v, m, _ = inputs.config("C1", n=n)
    tj, dtj, a0, j0 = inputs.taylor_state(n, 77)
    # first 300 through the GRAPE-6 call (pre-divided coefficients), the rest through the bulk loader
    for p in range(300):
        g6.g6_set_j_particle(0, p, p, tj[p], dtj[p], m[p], None, j0[p] / 6, a0[p] / 2, v[p], x[p])
    g6.g6x_set_j_particles(0, 300, np.arange(300, n, dtype=np.int32), tj[300:], m[300:], j0[300:], a0[300:], v[300:], x[300:])
    for ti in (0.0, 0.0625):
        g6.g6_set_ti(0, ti)
        xp, vp = g6.g6x_get_predicted(0, 0, n)
        xo, vo = oracle.predict(ti, tj, x, v, a0, j0)
        dt = (ti - tj)[:, None]
        # v0, a0, j0 are stored in binary32: each term carries 2^-24 relative error,
        # the FP32 Horner evaluation a few more; positions are double-single (2^-48 relative)
        terms_x = np.abs(v * dt) + np.abs(a0 * dt**2 / 2) + np.abs(j0 * dt**3 / 6)
        terms_v = np.abs(v) + np.abs(a0 * dt) + np.abs(j0 * dt**2 / 2)
        assert np.all(np.abs(xp - xo) <= 4 * 2.0**-24 * terms_x + 2.0**-46 * np.abs(xo))
        assert np.all(np.abs(vp - vo) <= 4 * 2.0**-24 * terms_v)
    # identity at dt = 0: positions come back to double-single accuracy, velocities to binary32
    sel = tj == 0.0
    g6.g6_set_ti(0, 0.0)
    xp, vp = g6.g6x_get_predicted(0, 0, n)
    assert np.all(np.abs(xp[sel] - x[sel]) <= 2.0**-47 * np.abs(x[sel]))
    assert np.array_equal(vp[sel], v[sel].astype(np.float32).astype(np.float64))


# ------------------------------------------------------------------ t_i != t_j, self-exclusion by index
@pytest.mark.parametrize("kernel", KERNELS)
def test_block_step_shape_parity(cluster, oracle, kernel):
    """The production shape: j-particles at their own times, the block predicted by the host in
    fp64, the same particles present as j (so the self pair has a tiny non-zero separation and
    must be excluded by index, reading 4); index != address."""
    n = 3000
    x, v, m, _ = inputs.config("C2", n=n)
    eps2 = 1e-8
    rng = np.random.default_rng(5)
    idx = (rng.permutation(n) + 1000).astype(np.int32)
    lev = rng.integers(6, 12, n)
    tj = -(2.0 ** -lev.astype(float)) * rng.integers(0, 2, n)
    a0 = rng.normal(0, 1, (n, 3)); j0 = rng.normal(0, 5, (n, 3))
    g6.g6x_set_option(0, "kernel", kernel)
    load_j(x, v, m, index=idx, t=tj, acc=a0, jerk=j0)
    ti = 2.0**-9
    g6.g6_set_ti(0, ti)
    xo, vo = oracle.predict(ti, tj, x, v, a0, j0)            # host-side fp64 prediction
    block = np.sort(rng.choice(n, 77, replace=False))
    got = g6.force_host(0, idx[block], xo[block], vo[block], eps2, n)
    ref = oracle.force(idx[block], xo[block], vo[block], idx, xo, vo, m, eps2)
    check_forces(got, ref, f"block kernel={kernel}")
    check_nn(got["nn_index"], ref, idx, xo[block], xo)
    # had the self pair been included, phi would be off by ~ -m/eps = -1/(3000 * 1e-4) = -3.3
    assert np.abs(got["pot"] - ref["pot"]).max() < 1e-5


# ------------------------------------------------------------------ j-split invariance, determinism
@pytest.mark.parametrize("kernel", KERNELS)
def test_jsplit_invariance_and_reproducibility(cluster, oracle, kernel):
    x, v, m, eps2 = inputs.config("C1", n=6000)
    n = len(m)
    idx = load_j(x, v, m)
    g6.g6x_set_option(0, "kernel", kernel)
    g6.g6_set_ti(0, 0.0)
    block = np.arange(0, n, 29, dtype=np.int32)
    ref = oracle.force(idx[block], x[block], v[block], idx, x, v, m, eps2)
    runs = {}
    for S in (1, 3, 24, 0):
        g6.g6x_set_option(0, "jsplit", S)
        a = g6.force_host(0, idx[block], x[block], v[block], eps2, n)
        b = g6.force_host(0, idx[block], x[block], v[block], eps2, n)
        for k in ("acc", "jerk", "pot", "nn_index", "nn_r2"):
            assert np.array_equal(a[k], b[k]), f"S={S}: {k} not bit-reproducible"
        check_forces(a, ref, f"S={S}")
        check_nn(a["nn_index"], ref, idx, x[block], x)
        runs[S] = a
        if S:
            assert g6.g6x_get_timers(0)["jsplits"] == S
    assert np.array_equal(runs[1]["nn_index"], runs[24]["nn_index"])      # tie rule independent of the split
    assert rel_err(runs[1]["acc"], runs[24]["acc"]).max() < 1e-6


# ------------------------------------------------------------------ ragged sizes and degenerate cases
@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("n,ni", [(1000, 1), (257, 257), (256, 3), (1, 1), (2, 2), (4097, 130), (777, 600)])
def test_ragged_and_tiny(cluster, oracle, kernel, n, ni):
    x, v, m, eps2 = inputs.config("C1", n=max(n, 2))
    x, v, m = x[:n], v[:n], m[:n]
    idx = load_j(x, v, m)
    g6.g6x_set_option(0, "kernel", kernel)
    g6.g6_set_ti(0, 0.0)
    got = g6.force_host(0, idx[:ni], x[:ni], v[:ni], eps2, n)
    ref = oracle.force(idx[:ni], x[:ni], v[:ni], idx, x, v, m, eps2)
    if n == 1:
        assert got["nn_index"][0] == -1 and np.isinf(got["nn_r2"][0])
        assert np.all(got["acc"] == 0) and got["pot"][0] == 0
        return
    check_forces(got, ref, f"n={n} ni={ni}")
    check_nn(got["nn_index"], ref, idx, x[:ni], x)


@pytest.mark.parametrize("kernel", KERNELS)
def test_nj_smaller_than_stored_and_foreign_i(cluster, oracle, kernel):
    """nj < stored particles: only addresses [0, nj) act; i-particles that are not in the j set."""
    x, v, m, eps2 = inputs.config("C1", n=2000)
    idx = load_j(x, v, m)
    g6.g6x_set_option(0, "kernel", kernel)
    g6.g6_set_ti(0, 0.0)
    nj = 1234
    sel = np.arange(1500, 1700)
    got = g6.force_host(0, idx[sel], x[sel], v[sel], eps2, nj)
    ref = oracle.force(idx[sel], x[sel], v[sel], idx[:nj], x[:nj], v[:nj], m[:nj], eps2)
    check_forces(got, ref, "nj<stored")
    check_nn(got["nn_index"], ref, idx[:nj], x[sel], x[:nj])


def test_eps2_zero_and_coincident_particles(cluster, oracle):
    """eps2 = 0 takes the checked path: distinct coincident particles are skipped (reading 5),
    no NaN/Inf; the nearest-neighbour tie rule picks the smaller address (reading 7)."""
    x, v, m, _ = inputs.config("C1", n=600)
    x[300] = x[10]; v[300] = v[10]                      # coincident distinct pair
    x[400] = x[20] + np.array([0.5, 0, 0]); x[401] = x[20] - np.array([0.5, 0, 0])   # exact tie for i = 20
    x[20] = np.round(x[20] * 64) / 64; x[400] = x[20] + np.array([0.5, 0, 0]); x[401] = x[20] - np.array([0.5, 0, 0])
    idx = load_j(x, v, m)
    g6.g6_set_ti(0, 0.0)
    got = g6.force_host(0, idx, x, v, 0.0, 600)
    ref = oracle.force(idx, x, v, idx, x, v, m, 0.0)
    assert np.all(np.isfinite(got["acc"])) and np.all(np.isfinite(got["jerk"])) and np.all(np.isfinite(got["pot"]))
    check_forces(got, ref, "eps2=0")
    check_nn(got["nn_index"], ref, idx, x, x)
    d = np.linalg.norm(x - x[20], axis=1); d[20] = np.inf
    if d.min() == 0.5:
        assert got["nn_index"][20] == 400 == ref["nn_index"][20]


# ------------------------------------------------------------------ block-step kernel (one launch: update + predictor + force + combine)
@pytest.mark.parametrize("n,ni,small", [(5000, 1, 16), (5000, 7, 16), (5000, 16, 16), (1000, 64, 64), (300, 33, 64), (40000, 3, 16),
                                        # blocks of 17..31 as two power-of-two chunks, 33..64 as 32 + the rest
                                        (5000, 17, 64), (5000, 24, 64), (3000, 31, 64), (3000, 40, 64),
                                        # the static quarter-tile schedule: full rounds and every shape of the last round
                                        # (7-8 and 13-14 tiles per CTA: warps with two quarters, one, none; an empty last round)
                                        (300000, 5, 16), (300000, 20, 64), (530000, 16, 16), (530000, 24, 64)])
def test_small_block_kernel_fused_predictor(cluster, oracle, n, ni, small):
    """n_i <= `small`: one pass over the raw j-store, Eq. 1-2 evaluated on the fly, t_i != t_j, the
    block's own particles present as j; must agree with the oracle and with the two-kernel path."""
    x, v, m, _ = inputs.config("C2", n=n)
    eps2 = 1e-8
    rng = np.random.default_rng(ni)
    idx = (rng.permutation(n) + 7).astype(np.int32)
    tj, dtj, a0, j0 = inputs.taylor_state(n, 100 + ni, dt_max=2.0**-6)
    load_j(x, v, m, index=idx, t=tj, acc=a0, jerk=j0)
    ti = 2.0**-8
    g6.g6_set_ti(0, ti)
    xo, vo = oracle.predict(ti, tj, x, v, a0, j0)
    block = np.sort(rng.choice(n, ni, replace=False))
    ref = oracle.force(idx[block], xo[block], vo[block], idx, xo, vo, m, eps2)
    g6.g6x_set_option(0, "small", small)
    got = g6.force_host(0, idx[block], xo[block], vo[block], eps2, n)
    tm = g6.g6x_get_timers(0)
    assert tm["jsplits"] == tm["force_ctas"] <= (n + 255) // 256   # one partial per persistent CTA: the block-step kernel ran
    again = g6.force_host(0, idx[block], xo[block], vo[block], eps2, n)
    for k in got:
        assert np.array_equal(got[k], again[k]), k          # bit-reproducible
    g6.g6x_set_option(0, "kernel", 2)                        # the two-kernel path: predictor, then the fast kernel
    two = g6.force_host(0, idx[block], xo[block], vo[block], eps2, n)
    g6.g6x_set_option(0, "kernel", 0)
    g6.g6x_set_option(0, "small", 32)
    if ni >= 16:
        check_forces(got, ref, f"small n={n} ni={ni}")
    assert rel_err(got["acc"], ref["acc"]).max() <= 1e-5 and rel_err(got["jerk"], ref["jerk"]).max() <= 1e-4
    assert rel_err(got["pot"], ref["pot"]).max() <= 1e-6
    check_nn(got["nn_index"], ref, idx, xo[block], xo)
    assert rel_err(got["acc"], two["acc"]).max() < 2e-6 and np.array_equal(got["nn_index"], two["nn_index"])
    # a second call at the same time reuses nothing stale: predicted positions read back are current
    xp, vp = g6.g6x_get_predicted(0, 0, n)
    assert np.abs(xp - xo).max() < 1e-7


@pytest.mark.parametrize("n,ni", [(5000, 1), (5000, 5), (3000, 16), (70000, 32), (900, 64)])
def test_block_step_cycle_with_j_updates(cluster, oracle, n, ni):
    """The production cycle (SURVEY.md call stack 1): g6_set_j_particle for the n_i particles corrected in the
    last step, g6_set_ti, firsthalf/lasthalf of the next block.  With n_i <= 32 the changed records ride in
    the launch of the block-step kernel (a-1 fused); they must act in THAT call, persist in the j-store
    for later calls, and agree with the staged path (kernel = 2) bit for bit in what is stored."""
    x, v, m, _ = inputs.config("C2", n=n)
    eps2 = 1e-8
    rng = np.random.default_rng(1000 + ni)
    idx = rng.permutation(n).astype(np.int32)
    tj, dtj, a0, j0 = inputs.taylor_state(n, 200 + ni, dt_max=2.0**-6)
    load_j(x, v, m, index=idx, t=tj, acc=a0, jerk=j0)
    g6.g6x_set_option(0, "small", 64)
    t = 2.0**-8
    for step in range(3):
        # "correct" a block: new state at time t for ni particles (addresses spread over tiles, one in the last, ragged tile)
        blk = np.sort(rng.choice(n - 1, ni - 1, replace=False)) if ni > 1 else np.array([], dtype=int)
        blk = np.append(blk, n - 1).astype(int)
        x[blk] += 1e-3 * rng.standard_normal((ni, 3)); v[blk] += 1e-3 * rng.standard_normal((ni, 3))
        a0[blk] = rng.standard_normal((ni, 3)); j0[blk] = rng.standard_normal((ni, 3)); tj[blk] = t
        for p in blk:
            g6.g6_set_j_particle(0, int(p), int(idx[p]), tj[p], dtj[p], m[p], None, j0[p] / 6, a0[p] / 2, v[p], x[p])
        t += 2.0**-9
        g6.g6_set_ti(0, t)
        xo, vo = oracle.predict(t, tj, x, v, a0, j0)
        nxt = np.sort(rng.choice(n, ni, replace=False))
        nxt[0] = blk[0]                                     # a just-updated particle is also active next
        ref = oracle.force(idx[nxt], xo[nxt], vo[nxt], idx, xo, vo, m, eps2)
        got = g6.force_host(0, idx[nxt], xo[nxt], vo[nxt], eps2, n)
        assert rel_err(got["acc"], ref["acc"]).max() <= 1e-5 and rel_err(got["jerk"], ref["jerk"]).max() <= 1e-4
        assert rel_err(got["pot"], ref["pot"]).max() <= 1e-6
        check_nn(got["nn_index"], ref, idx, xo[nxt], xo)
        # the j-store now holds the updates: the two-kernel path sees the same particles
        g6.g6x_set_option(0, "kernel", 2)
        two = g6.force_host(0, idx[nxt], xo[nxt], vo[nxt], eps2, n)
        g6.g6x_set_option(0, "kernel", 0)
        assert rel_err(got["acc"], two["acc"]).max() < 2e-6 and np.array_equal(got["nn_index"], two["nn_index"])
        xp, vp = g6.g6x_get_predicted(0, 0, n)
        assert np.abs(xp - xo).max() < 1e-7 and np.abs(vp - vo).max() < 1e-5
    g6.g6x_set_option(0, "small", 32)


# ------------------------------------------------------------------ P11: Eq. 3 bit for bit
def _pair_dx(kernel, xj, index_j, xi, index_i, eps2, ds=1):
    """Every pair's separation as the PRODUCTION pair code formed it: libg6b200_dbg.so instantiates k_force_fast /
    the block-step kernel (same headers) with their DBG template flag (csrc/debug/g6_debug_dx.cu)."""
    import ctypes as C
    from paper_0902_4463_b200 import build
    L = C.CDLL(build.build_debug())
    nj, ni = len(index_j), len(index_i)
    xj = np.ascontiguousarray(xj, np.float64); xi = np.ascontiguousarray(xi, np.float64)
    index_j = np.ascontiguousarray(index_j, np.int32); index_i = np.ascontiguousarray(index_i, np.int32)
    dx = np.empty((ni, nj, 3), np.float32)
    dp = lambda a: a.ctypes.data_as(C.POINTER(C.c_double)); ip = lambda a: a.ctypes.data_as(C.POINTER(C.c_int))
    rc = L.g6dbg_pair_dx(C.c_int(kernel), C.c_int(nj), C.c_int(ni), dp(xj), ip(index_j), dp(xi), ip(index_i),
                         C.c_double(eps2), C.c_int(ds), dx.ctypes.data_as(C.POINTER(C.c_float)))
    assert rc == 0, rc
    return dx


@pytest.mark.parametrize("kernel,ni", [(2, 700), (3, 37)])
def test_p11_ds_separation_bit_exact(oracle, kernel, ni):
    """Eq. 3 as the hot loops form it -- packed lanes of pair2 (sweep kernel: unchecked tiles, the checked
    tiles that hold the warp's own particles, the ragged last tile) and pair2_checked (block-step kernel) -- equals the
    binary32 CPU transcription bit for bit, for EVERY (i, j) pair, on the offset cluster where the lo words matter."""
    nj = 4000                                            # 15 full j-tiles and a ragged one
    x, v, m, eps2 = inputs.config("C5", n=nj)
    idx = np.arange(nj, dtype=np.int32)
    sel = np.sort(np.random.default_rng(3).choice(nj, ni, replace=False))
    dx = _pair_dx(kernel, x, idx, x[sel], idx[sel], eps2)
    assert not np.isnan(dx).any()                        # every pair was visited (the buffer starts as NaN)
    for k in range(3):
        ih, il = oracle.ds_split(x[sel, k]); jh, jl = oracle.ds_split(x[:, k])
        want = oracle.ds_diff(np.broadcast_to(jh, (ni, nj)).ravel(), np.broadcast_to(jl, (ni, nj)).ravel(),
                              np.repeat(ih, nj), np.repeat(il, nj)).reshape(ni, nj)
        assert np.array_equal(dx[:, :, k].view(np.uint32), want.view(np.uint32))
        exact = x[None, :, k] - x[sel, None, k]
        assert np.all(np.abs(dx[:, :, k] - exact) <= 3 * 2.0**-24 * np.abs(exact) + 2.0**-47 * 1001.0)
    # pure FP32 (lo words dropped): the separation is the single rounded difference of the hi words
    d0 = _pair_dx(kernel, x, idx, x[sel], idx[sel], eps2, ds=0)
    ih, _ = oracle.ds_split(x[sel, 0]); jh, _ = oracle.ds_split(x[:, 0])
    assert np.array_equal(d0[:, :, 0], (jh[None, :] - ih[:, None]).astype(np.float32))


# ------------------------------------------------------------------ C5: double-single vs pure FP32
@pytest.mark.parametrize("n", [8192, 65536])
def test_c5_double_single_beats_pure_fp32(cluster, oracle, n):
    x, v, m, eps2 = inputs.config("C5", n=n)
    idx = load_j(x, v, m)
    g6.g6_set_ti(0, 0.0)
    rows = np.arange(n) if n <= 8192 else np.sort(np.random.default_rng(55).choice(n, 8192, replace=False))
    ref = oracle.force(idx[rows], x[rows], v[rows], idx, x, v, m, eps2)
    g6.g6x_set_option(0, "ds", 1)
    ds = g6.force_host(0, idx[rows], x[rows], v[rows], eps2, n)
    st = check_forces(ds, ref, "C5 DS")
    check_nn(ds["nn_index"], ref, idx, x[rows], x)
    g6.g6x_set_option(0, "ds", 0)
    sp = g6.force_host(0, idx[rows], x[rows], v[rows], eps2, n)
    g6.g6x_set_option(0, "ds", 1)
    e_ds = rel_err(ds["acc"], ref["acc"]); e_sp = rel_err(sp["acc"], ref["acc"])
    j_ds = rel_err(ds["jerk"], ref["jerk"]); j_sp = rel_err(sp["jerk"], ref["jerk"])
    print(f"C5 n={n}: DS acc median {np.median(e_ds):.2e} max {e_ds.max():.2e} | FP32 acc median {np.median(e_sp):.2e} max {e_sp.max():.2e}"
          f" | DS jerk median {np.median(j_ds):.2e} | FP32 jerk median {np.median(j_sp):.2e}")
    assert np.median(e_sp) > 100 * np.median(e_ds)       # orders of magnitude
    assert e_sp.max() > 100 * e_ds.max()
    assert np.median(j_sp) > 100 * np.median(j_ds)


# ------------------------------------------------------------------ C3 / C4 at full size: sampled rows
def _sampled_full_sweep(oracle, name, nrows, seed):
    x, v, m, eps2 = inputs.config(name)
    n = len(m)
    idx = load_j(x, v, m)
    g6.g6_set_ti(0, 0.0)
    got = g6.force_host(0, idx, x, v, eps2, n)           # the full sweep, n_i = N, one call
    tm = g6.g6x_get_timers(0)
    rows = np.sort(np.random.default_rng(seed).choice(n, nrows, replace=False))
    ref = oracle.force(idx[rows], x[rows], v[rows], idx, x, v, m, eps2)
    sub = {k: got[k][rows] for k in got}
    st = check_forces(sub, ref, name)
    nd = check_nn(sub["nn_index"], ref, idx, x[rows], x)
    print(name, st, "nn ties:", nd, "force kernel: %.1f ms, %.3e interactions/s" % (tm["force_us"] / 1e3, n * float(n) / (tm["force_us"] * 1e-6)))
    # invariants that hold at any size: Newton's third law over the whole sweep, W ~ -1/2
    tot = np.linalg.norm((m[:, None] * got["acc"]).sum(0)) / (m * np.linalg.norm(got["acc"], axis=1)).sum()
    assert tot < 1e-6, tot
    W = 0.5 * np.sum(m * got["pot"])
    assert abs(W + 0.5) < 1.5 / np.sqrt(n) + 0.003, W
    return x, v, m, eps2, idx


def test_c3_full_sweep_sampled_rows(cluster, oracle):
    _sampled_full_sweep(oracle, "C3", 16384, 303)


def test_c4_full_sweep_and_ni_sweep(cluster, oracle):
    x, v, m, eps2, idx = _sampled_full_sweep(oracle, "C4", 4096, 404)
    n = len(m)
    for ni in (1, 16, 256, 4096, 65536):
        block = inputs.active_subset(n, ni, 4040 + ni)
        got = g6.force_host(0, idx[block], x[block], v[block], eps2, n)
        tm = g6.g6x_get_timers(0)
        rows = np.arange(ni) if ni <= 4096 else np.sort(np.random.default_rng(9).choice(ni, 1024, replace=False))
        ref = oracle.force(idx[block][rows], x[block][rows], v[block][rows], idx, x, v, m, eps2)
        sub = {k: got[k][rows] for k in got}
        check_forces(sub, ref, f"C4 ni={ni}") if ni >= 16 else None
        if ni < 16:                                      # medians over < 16 rows mean little: max bounds only
            assert rel_err(sub["acc"], ref["acc"]).max() <= 1e-5 and rel_err(sub["jerk"], ref["jerk"]).max() <= 1e-4
            assert rel_err(sub["pot"], ref["pot"]).max() <= 1e-6
        check_nn(sub["nn_index"], ref, idx, x[block][rows], x)
        print(f"C4 ni={ni}: force {tm['force_us']:.1f} us, predict {tm['predict_us']:.1f} us, S={tm['jsplits']}, CTAs={tm['force_ctas']}")


# ------------------------------------------------------------------ error behaviour of the ABI on a live device
def test_abi_errors_on_device(cluster):
    x, v, m, eps2 = inputs.config("C1", n=300)
    idx = load_j(x, v, m)
    g6.g6_set_ti(0, 0.0)
    E = g6.G6Error
    with pytest.raises(E) as e: g6.g6calc_lasthalf(0, 300, 10)
    assert e.value.code == -6
    with pytest.raises(E) as e: g6.g6calc_firsthalf(0, 301, 10, idx[:10], x[:10], v[:10], eps2=eps2)
    assert e.value.code == -5
    g6.g6x_set_npipes(256)
    with pytest.raises(E) as e: g6.g6calc_firsthalf(0, 300, 257, idx[:257], x[:257], v[:257], eps2=eps2)
    assert e.value.code == -4
    g6.g6x_set_npipes(1 << 21)
    with pytest.raises(E) as e: g6.g6_set_j_particle(0, 1 << 30, 0, 0.0, 0.0, 1.0, None, x[0], x[0], x[0], x[0])
    assert e.value.code == -3
    with pytest.raises(E) as e: g6.g6_open(0)
    assert e.value.code == -9
    g6.g6calc_firsthalf(0, 300, 10, idx[:10], x[:10], v[:10], eps2=eps2)
    with pytest.raises(E) as e: g6.g6calc_firsthalf(0, 300, 10, idx[:10], x[:10], v[:10], eps2=eps2)
    assert e.value.code == -6
    with pytest.raises(E) as e: g6.g6calc_lasthalf(0, 300, 11)
    assert e.value.code == -8
    g6.g6calc_lasthalf(0, 300, 10)
    with pytest.raises(E) as e: g6.g6x_set_option(0, "nonsense", 1)
    assert e.value.code == -8


def test_overwriting_a_j_particle_takes_effect(cluster, oracle):
    x, v, m, eps2 = inputs.config("C1", n=500)
    idx = load_j(x, v, m)
    g6.g6_set_ti(0, 0.0)
    g6.force_host(0, idx[:50], x[:50], v[:50], eps2, 500)
    x2 = x.copy(); x2[123] += 0.25; m2 = m.copy(); m2[123] *= 3
    z = np.zeros(3)
    g6.g6_set_j_particle(0, 123, 123, 0.0, 0.125, m2[123], None, z, z, v[123], x2[123])
    g6.g6_set_j_particle(0, 123, 123, 0.0, 0.125, m2[123], None, z, z, v[123], x2[123])   # twice: last one wins, no race
    got = g6.force_host(0, idx[:50], x[:50], v[:50], eps2, 500)
    ref = oracle.force(idx[:50], x[:50], v[:50], idx, x2, v, m2, eps2)
    check_forces(got, ref, "after overwrite")


def test_maximum_capacity(cluster, oracle):
    """The largest j-store the library holds by default (2^21 addresses): every address in use, the last one included;
    a 512-block through the sweep kernels and a 7-block through the block-step kernel against the oracle; one address
    past the end is refused."""
    n = 1 << 21
    x, v, m, eps2 = inputs.config("C4", n=n)
    idx = load_j(x, v, m)
    g6.g6_set_ti(0, 0.0)
    E = g6.G6Error
    with pytest.raises(E) as e: g6.g6_set_j_particle(0, n, 0, 0.0, 0.0, 1.0, None, x[0], x[0], x[0], x[0])
    assert e.value.code == -3
    for ni, kernel in ((512, 2), (7, 3)):
        sel = inputs.active_subset(n, ni, 77 + ni)
        sel[-1] = n - 1                                   # the last address is an i-particle too
        got = g6.force_host(0, idx[sel], x[sel], v[sel], eps2, n)
        assert g6.g6x_get_option(0, "last_kernel") == kernel
        ref = oracle.force(idx[sel], x[sel], v[sel], idx, x, v, m, eps2)
        check_forces(got, ref, f"capacity n_i={ni}")
        check_nn(got["nn_index"], ref, idx, x[sel], x)
