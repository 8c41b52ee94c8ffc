"""The host Hermite driver (g6h_*, step a-7) driving the CUDA library, against the oracle-driven
integrator (oracle/hermite_oracle.c) on the same seeded inputs."""
import time

import os

import numpy as np
import pytest

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


def _energy(oracle, x, v, m, eps2):
    T, W = oracle.energy(x, v, m, eps2)
    return T + W


def test_binary_period_through_the_library(cluster, oracle):
    """circular binary with period 1 (Kepler), integrated by the library-driven Hermite scheme"""
    d = (2 * np.pi) ** (-2.0 / 3.0)
    m = np.array([0.5, 0.5]); vrel = np.sqrt(1.0 / d)
    x = np.array([[-d / 2, 0, 0], [d / 2, 0, 0]]); v = np.array([[0, -vrel / 2, 0], [0, vrel / 2, 0]])
    h = g6.Hermite(0, x, v, m, 1e-12, 0.002)
    h.evolve(1.0)
    x1, v1 = h.state()
    st = h.stats()
    assert st["t"] == 1.0
    assert np.abs(x1 - x).max() < 5e-6 and np.abs(v1 - v).max() < 5e-5
    h.close()


@pytest.mark.parametrize("n,t_end", [(512, 0.25)])
def test_library_driven_vs_oracle_driven(cluster, oracle, n, t_end):
    x, v, m, _ = inputs.config("C2", n=n)
    eps2, eta = 1e-4 ** 2, 0.01
    E0 = _energy(oracle, x, v, m, eps2)
    ro = oracle.hermite(x, v, m, eps2, eta, t_end)
    dE_o = abs(_energy(oracle, ro.x, ro.v, m, eps2) - E0) / abs(E0)
    h = g6.Hermite(0, x, v, m, eps2, eta)
    h.evolve(t_end)
    xg, vg = h.state(); st = h.stats(); h.close()
    dE_g = abs(_energy(oracle, xg, vg, m, eps2) - E0) / abs(E0)
    print(f"N={n} t={t_end}: dE/E library-driven {dE_g:.3e}, oracle-driven {dE_o:.3e}; block steps {st['n_block_steps']} vs {ro.n_block_steps}; "
          f"particle steps {st['n_particle_steps']} vs {ro.n_particle_steps}")
    assert st["t"] == t_end == ro.t
    # north_star: energy drift within 2x of the oracle-driven run (plus the FP32 force floor ~1e-9..1e-8)
    assert dE_g <= 2 * dE_o + 2e-8
    # the step sequence is the same scheme: counts agree to a few per cent (FP32 forces shift a few steps)
    assert abs(st["n_particle_steps"] - ro.n_particle_steps) <= 0.03 * ro.n_particle_steps
    assert st["ni_hist_log2"].sum() == st["n_block_steps"]
    # trajectories still agree closely over a quarter time unit for most particles
    dx = np.linalg.norm(xg - ro.x, axis=1)
    assert np.median(dx) < 1e-6


def test_c2_short_run_energy_and_block_histogram(cluster, oracle):
    """C2 (N = 32768, eps = 1e-4, eta = 0.01) for a short stretch: energy conservation and the n_i
    histogram.  The full t = 0 -> 1 run is done by `python -m paper_0902_4463_b200.hermite_run`
    (report in profiles/); here the end time is kept short so the suite stays fast."""
    x, v, m, eps2 = inputs.config("C2")
    eta, t_end = 0.01, 2.0 ** -6
    E0 = _energy(oracle, x, v, m, eps2)
    t0 = time.perf_counter()
    h = g6.Hermite(0, x, v, m, eps2, eta)
    h.evolve(t_end)
    xg, vg = h.state(); st = h.stats(); h.close()
    wall = time.perf_counter() - t0
    dE = abs(_energy(oracle, xg, vg, m, eps2) - E0) / abs(E0)
    print(f"C2 to t={t_end}: dE/E={dE:.3e}, {st['n_block_steps']} block steps, {st['n_particle_steps']} particle steps, "
          f"{st['interactions']:.3e} interactions in {wall:.1f} s (force calls {st['wall_force_s']:.1f} s); "
          f"n_i histogram (log2 bins): {list(st['ni_hist_log2'][:16])}")
    assert st["t"] == t_end
    assert dE < 1e-6


def test_c2_full_run_vs_oracle_driven(cluster, oracle):
    """BASELINE.json config 2 in full: N = 32768, eps = 1e-4, eta = 0.01, t = 0 -> 1, driven by the host driver (g6h_*), by the
    device-resident driver (g6hd_*) and by the oracle (~1e12 fp64 pair evaluations: a few minutes on the GPU box's host cores).
    north_star: the library-driven energy drift stays within 2x the oracle-driven one."""
    import json, os
    t_end = float(os.environ.get("G6_C2_TEND", "1.0"))
    x, v, m, eps2 = inputs.config("C2")
    eta = 0.01
    E0 = _energy(oracle, x, v, m, eps2)
    rep = {"config": "C2", "n": len(m), "eta": eta, "eps2": eps2, "t_end": t_end, "E0": E0, "oracle_threads": oracle.threads()}
    for newton in ((1, 0) if os.environ.get("G6_C2_NEWTON0") else (1,)):
        g6.g6x_set_option(0, "newton", newton)
        t0 = time.perf_counter()
        h = g6.Hermite(0, x, v, m, eps2, eta)
        h.evolve(t_end)
        xg, vg = h.state(); st = h.stats(); h.close()
        wall = time.perf_counter() - t0
        dE = (_energy(oracle, xg, vg, m, eps2) - E0) / abs(E0)
        rep[f"library_newton{newton}"] = {"dE_over_E": dE, "block_steps": st["n_block_steps"], "particle_steps": st["n_particle_steps"],
                                          "interactions": st["interactions"], "wall_s": wall, "wall_force_calls_s": st["wall_force_s"],
                                          "dt_min": st["dt_min"], "ni_hist_log2": [int(c) for c in st["ni_hist_log2"][:20]],
                                          "force_wall_s_log2": [round(float(c), 4) for c in st["force_wall_s_log2"][:20]]}
        print(json.dumps({f"library_newton{newton}": rep[f"library_newton{newton}"]}), flush=True)
    g6.g6x_set_option(0, "newton", 1)
    t0 = time.perf_counter()
    hd = g6.HermiteDev(0, x, v, m, eps2, eta)
    hd.evolve(t_end)
    xd, vd = hd.state(); sd = hd.stats(); hd.close()
    wall = time.perf_counter() - t0
    dE = (_energy(oracle, xd, vd, m, eps2) - E0) / abs(E0)
    rep["device_resident_newton1"] = {"dE_over_E": dE, "block_steps": sd["n_block_steps"], "particle_steps": sd["n_particle_steps"],
                                      "interactions": sd["interactions"], "wall_s": wall, "wall_evolve_s": sd["wall_s"], "dt_min": sd["dt_min"],
                                      "ni_hist_log2": [int(c) for c in sd["ni_hist_log2"][:20]]}
    print(json.dumps({"device_resident_newton1": rep["device_resident_newton1"]}), flush=True)
    t0 = time.perf_counter()
    ro = oracle.hermite(x, v, m, eps2, eta, t_end)
    wall = time.perf_counter() - t0
    dE_o = (_energy(oracle, ro.x, ro.v, m, eps2) - E0) / abs(E0)
    rep["oracle_driven"] = {"dE_over_E": dE_o, "block_steps": ro.n_block_steps, "particle_steps": ro.n_particle_steps,
                            "interactions": ro.interactions, "wall_s": wall, "dt_min": ro.dt_min,
                            "ni_hist_log2": [int(c) for c in ro.ni_hist_log2[:20]]}
    print("C2_REPORT " + json.dumps(rep), flush=True)
    os.makedirs("gpurun_out", exist_ok=True)
    json.dump(rep, open("gpurun_out/c2_report.json", "w"), indent=1)
    assert abs(rep["library_newton1"]["dE_over_E"]) <= 2 * abs(dE_o) + 2e-8
    assert abs(rep["device_resident_newton1"]["dE_over_E"]) <= 2 * abs(dE_o) + 2e-8


# ------------------------------------------------------------------ device-resident integrator (NEXT-3, g6hd_*)
@pytest.mark.parametrize("loop", [1, 0])
def test_device_corrector_and_selection_against_oracle(cluster, oracle, monkeypatch, loop):
    """(loop = 1: the persistent step-loop kernel k_hd_loop, one step per launch here; loop = 0: k_hd_select / the library's
    force path / k_hd_correct with one host wait per step -- env G6_HD_LOOP, read by g6hd_create.)
    One block step at a time: the block the device selects is the set of particles with the smallest
    t + dt, in address order; its i-particles are Eq. 1-2 predictions (oracle.predict); the corrector kernel's
    new x, v equal oracle.hermite_correct and the new step follows oracle.aarseth_dt and the power-of-two
    rule, given the forces the device used."""
    n = 3000
    x, v, m, _ = inputs.config("C2", n=n)
    eps2, eta, dt_max = 1e-4 ** 2, 0.01, 0.125
    monkeypatch.setenv("G6_HD_LOOP", str(loop))
    h = g6.HermiteDev(0, x, v, m, eps2, eta)
    before = h.particles()
    assert np.all(before["t"] == 0) and np.all(before["dt"] <= dt_max) and np.all(np.log2(before["dt"]) % 1 == 0)
    seen = 0
    for step in range(40):
        tn_all = before["t"] + before["dt"]
        tnext = tn_all.min()
        want_act = np.nonzero(tn_all == tnext)[0]
        h.evolve(1.0, max_block_steps=1)
        blk = h.last_block()
        after = h.particles()
        assert np.array_equal(blk["act"], want_act.astype(np.int32))
        act = blk["act"]
        xp, vp = oracle.predict(tnext, before["t"][act], before["x"][act], before["v"][act], before["a"][act], before["adot"][act])
        assert np.allclose(blk["xi"], xp, rtol=1e-14, atol=1e-15) and np.allclose(blk["vi"], vp, rtol=1e-13, atol=1e-15)
        for k, p in enumerate(act):
            hh = before["dt"][p]
            x1, v1, a2n, a3 = oracle.hermite_correct(hh, blk["xi"][k], blk["vi"][k], before["a"][p], before["adot"][p], blk["acc"][k], blk["jerk"][k])
            assert np.allclose(after["x"][p], x1, rtol=1e-14, atol=1e-16) and np.allclose(after["v"][p], v1, rtol=1e-13, atol=1e-15)
            assert np.array_equal(after["a"][p], blk["acc"][k]) and np.array_equal(after["adot"][p], blk["jerk"][k])
            assert after["t"][p] == tnext
            want = oracle.aarseth_dt(eta, blk["acc"][k], blk["jerk"][k], a2n, a3, dt_max)
            d = hh
            if want < d:
                while d > want:
                    d *= 0.5
            elif want >= 2 * d and 2 * d <= dt_max and np.fmod(tnext, 2 * d) == 0.0:
                d *= 2
            # a wish within rounding of a power of two may fall on either side of it
            assert after["dt"][p] == d or abs(want / after["dt"][p] - 1) < 1e-12 or abs(want / (2 * after["dt"][p]) - 1) < 1e-12, (p, want, d, after["dt"][p])
        untouched = np.setdiff1d(np.arange(n), act)
        for key in ("x", "v", "a", "adot", "t", "dt"):
            assert np.array_equal(after[key][untouched], before[key][untouched])
        seen += len(act)
        before = after
    # the forces the device used are the library's: check one block against the oracle on the predicted system
    st = h.stats()
    assert st["n_block_steps"] == 40 and st["n_particle_steps"] == seen
    h.close()


@pytest.mark.parametrize("n,t_end", [(512, 0.25), (5000, 0.03125)])
def test_device_driven_vs_host_driven_vs_oracle_driven(cluster, oracle, n, t_end):
    x, v, m, _ = inputs.config("C2", n=n)
    eps2, eta = 1e-4 ** 2, 0.01
    E0 = _energy(oracle, x, v, m, eps2)
    ro = oracle.hermite(x, v, m, eps2, eta, t_end)
    dE_o = abs(_energy(oracle, ro.x, ro.v, m, eps2) - E0) / abs(E0)
    hd = g6.HermiteDev(0, x, v, m, eps2, eta)
    hd.evolve(t_end)
    xd, vd = hd.state(); sd = hd.stats(); hd.close()
    hh = g6.Hermite(0, x, v, m, eps2, eta)
    hh.evolve(t_end)
    xh, vh = hh.state(); sh = hh.stats(); hh.close()
    dE_d = abs(_energy(oracle, xd, vd, m, eps2) - E0) / abs(E0)
    print(f"N={n} t={t_end}: dE/E device-driven {dE_d:.3e}, oracle-driven {dE_o:.3e}; block steps device {sd['n_block_steps']} host {sh['n_block_steps']} "
          f"oracle {ro.n_block_steps}; particle steps {sd['n_particle_steps']} / {sh['n_particle_steps']} / {ro.n_particle_steps}")
    assert sd["t"] == t_end
    assert dE_d <= 2 * dE_o + 2e-8
    assert abs(sd["n_particle_steps"] - ro.n_particle_steps) <= 0.03 * ro.n_particle_steps
    assert abs(sd["n_particle_steps"] - sh["n_particle_steps"]) <= 0.01 * sh["n_particle_steps"]
    assert sd["ni_hist_log2"].sum() == sd["n_block_steps"]
    assert np.median(np.linalg.norm(xd - ro.x, axis=1)) < 1e-6
    assert np.median(np.linalg.norm(xd - xh, axis=1)) < 1e-7


@pytest.mark.parametrize("n", [1, 2, 1025, 2049])
def test_device_driver_edge_sizes_match_host_driver(cluster, oracle, n):
    """sizes around the selection kernel's 1024-particle thread blocks, and the degenerate N = 1, 2"""
    x, v, m, _ = inputs.config("C2", n=max(n, 2))
    x, v, m = x[:n], v[:n], m[:n] / m[:n].sum()
    eps2, eta, t_end = 1e-2 ** 2, 0.02, 0.125
    hd = g6.HermiteDev(0, x, v, m, eps2, eta)
    hd.evolve(t_end)
    xd, vd = hd.state(); sd = hd.stats(); hd.close()
    hh = g6.Hermite(0, x, v, m, eps2, eta)
    hh.evolve(t_end)
    xh, vh = hh.state(); sh = hh.stats(); hh.close()
    assert sd["t"] == t_end == sh["t"]
    assert abs(sd["n_particle_steps"] - sh["n_particle_steps"]) <= 0.01 * sh["n_particle_steps"] + 1
    assert np.abs(xd - xh).max() < 1e-7 and np.abs(vd - vh).max() < 1e-6
    if n == 1:          # a lone particle feels nothing: straight line
        assert np.allclose(xd, x + v * t_end, rtol=0, atol=1e-15)


@pytest.mark.parametrize("n", [257, 37889, 80000, 151552])
def test_step_loop_with_several_resident_tiles_per_cta(cluster, oracle, n):
    """The step loop at sizes around its tile bookkeeping: two CTAs, one of them with a single particle (N = 257); one tile more
    than there are SMs (N = 37889 = 148 x 256 + 1: 75 CTAs with two resident raw tiles each); three per CTA (N = 80000); the most
    it takes (N = 151552 = 4 x 256 x 148) -- the whole-CTA rescan, the per-tile records and the tile loops of the pair phase.
    Against the same run without the loop (G6_HD_LOOP = 0: k_hd_select / sweep path / k_hd_correct)."""
    x, v, m, _ = inputs.config("C2", n=n)
    eps2, eta, t_end = 1e-3 ** 2, 0.01, (2.0 ** -5 if n < 1000 else 2.0 ** -9 if n < 100000 else 2.0 ** -10)
    runs = {}
    for loop in (1, 0):
        os.environ["G6_HD_LOOP"] = str(loop)
        try:
            h = g6.HermiteDev(0, x, v, m, eps2, eta)
        finally:
            del os.environ["G6_HD_LOOP"]
        h.evolve(t_end)
        runs[loop] = (h.state(), h.stats(), h.particles(), h.last_block())
        h.close()
    (x1, v1), s1, p1, b1 = runs[1]
    (x0, v0), s0, p0, b0 = runs[0]
    assert s1["t"] == t_end == s0["t"] and s1["n_block_steps"] > 4
    # same block schedule (FP32 force differences between the two pair codes may move a borderline step)
    assert abs(s1["n_particle_steps"] - s0["n_particle_steps"]) <= 0.002 * s0["n_particle_steps"] + 2
    assert np.abs(x1 - x0).max() < 1e-8 and np.abs(v1 - v0).max() < 1e-6
    # the no-loop path is what the oracle-driven comparisons above pin; the last blocks of the two runs are the same particles
    if s1["n_block_steps"] == s0["n_block_steps"] and s1["n_particle_steps"] == s0["n_particle_steps"]:
        assert np.array_equal(b1["act"], b0["act"])
        rel = np.linalg.norm(b1["acc"] - b0["acc"], axis=1) / np.linalg.norm(b0["acc"], axis=1)
        assert rel.max() <= 2e-5 and np.allclose(b1["xi"], b0["xi"], rtol=0, atol=1e-8)


def test_step_loop_with_a_largest_step_that_is_not_a_power_of_two(cluster, oracle):
    """dt_max = 0.1: the steps are 0.1 / 2^k, sums of steps are rounded, and t_next - t is no longer bit for bit the stored step.
    The loop and the path without it must still take the same block steps (the loop's corrector once started from t_next - t:
    3709 block steps against 2186 on this case)."""
    n = 3426
    x, v, m, _ = inputs.config("C2", n=n)
    eps2, eta, dt_max, t_end = 1e-2 ** 2, 0.01, 0.1, 0.05
    runs = {}
    for loop in (1, 0):
        os.environ["G6_HD_LOOP"] = str(loop)
        try:
            h = g6.HermiteDev(0, x, v, m, eps2, eta, dt_max=dt_max)
        finally:
            del os.environ["G6_HD_LOOP"]
        h.evolve(t_end)
        runs[loop] = (h.state(), h.stats())
        h.close()
    (x1, v1), s1 = runs[1]
    (x0, v0), s0 = runs[0]
    assert s1["t"] == t_end == s0["t"]
    assert abs(s1["n_block_steps"] - s0["n_block_steps"]) <= 0.01 * s0["n_block_steps"] + 2
    assert abs(s1["n_particle_steps"] - s0["n_particle_steps"]) <= 0.005 * s0["n_particle_steps"] + 2
    assert np.abs(x1 - x0).max() < 1e-8 and np.abs(v1 - v0).max() < 1e-5


def test_step_loop_random_walk_against_the_path_without_it(cluster, oracle):
    """seeded random sizes, softenings, accuracies and largest steps (0.1 included): the two device paths take the same block steps and
    end in the same state"""
    rng = np.random.default_rng(20261105)
    for case in range(10):
        n = int(rng.choice([rng.integers(2, 600), rng.integers(600, 9000), rng.integers(9000, 70000)]))
        eps2 = float(rng.choice([1e-2, 1e-3, 1e-4])) ** 2
        eta = float(rng.choice([0.005, 0.01, 0.02, 0.03]))
        dt_max = float(rng.choice([0.125, 0.0625, 0.1]))
        t_end = dt_max * float(rng.choice([0.25, 0.5, 1.0])) if n < 9000 else dt_max / 16
        x, v, m, _ = inputs.config("C2", n=max(n, 2))
        x, v, m = x[:n], v[:n], m[:n] / m[:n].sum()
        res = {}
        for loop in (1, 0):
            os.environ["G6_HD_LOOP"] = str(loop)
            try:
                h = g6.HermiteDev(0, x, v, m, eps2, eta, dt_max=dt_max)
            finally:
                del os.environ["G6_HD_LOOP"]
            h.evolve(t_end)
            res[loop] = (h.state(), h.stats())
            h.close()
        (x1, v1), s1 = res[1]
        (x0, v0), s0 = res[0]
        what = (case, n, eps2, eta, dt_max, t_end, s1["n_block_steps"], s0["n_block_steps"])
        assert s1["t"] == s0["t"] == t_end, what
        assert abs(s1["n_particle_steps"] - s0["n_particle_steps"]) <= 0.005 * s0["n_particle_steps"] + 3, what
        assert abs(s1["n_block_steps"] - s0["n_block_steps"]) <= 0.15 * s0["n_block_steps"] + 3, what
        assert np.abs(x1 - x0).max() < 1e-7 and np.abs(v1 - v0).max() < 1e-5, what


@pytest.mark.parametrize("n,t_end", [(512, 0.0625), (3000, 0.015625)])
def test_device_shared_time_steps_vs_oracle(cluster, oracle, n, t_end):
    """shared-time-step variant (reading 21) on the device against the oracle's: every particle takes every
    step, the same sequence of common steps (FP32 forces may shift a step or two), the same energy behaviour"""
    x, v, m, _ = inputs.config("C2", n=n)
    eps2, eta = 1e-3 ** 2, 0.01
    E0 = _energy(oracle, x, v, m, eps2)
    ro = oracle.hermite(x, v, m, eps2, eta, t_end, shared=True)
    dE_o = abs(_energy(oracle, ro.x, ro.v, m, eps2) - E0) / abs(E0)
    hd = g6.HermiteDev(0, x, v, m, eps2, eta)
    hd.set_shared_steps(True)
    hd.evolve(t_end)
    pt = hd.particles()
    xd, vd = hd.state(); sd = hd.stats()
    dE_d = abs(_energy(oracle, xd, vd, m, eps2) - E0) / abs(E0)
    print(f"shared N={n}: steps device {sd['n_block_steps']} oracle {ro.n_block_steps}, dE/E device {dE_d:.3e} oracle {dE_o:.3e}, dt_min {sd['dt_min']} / {ro.dt_min}")
    assert sd["t"] == t_end == ro.t
    assert np.all(pt["t"] == t_end)                                            # everybody at the same time
    # after the corrector every particle holds its own result of the block rule applied to the common step h:
    # a power of two, at most dt_max, and at most 2 h (one doubling) -- so no two of them differ by more than h's halvings
    assert np.all(np.log2(pt["dt"]) % 1 == 0) and pt["dt"].max() <= 0.125 and pt["dt"].min() >= sd["dt_min"]
    assert sd["n_particle_steps"] == n * sd["n_block_steps"]
    b = int(np.log2(n))
    assert sd["ni_hist_log2"][b] == sd["n_block_steps"]
    # the common step is the SMALLEST wish: one particle near a power-of-two boundary moves the whole system, so FP32
    # forces shift the step sequence more than in the block scheme
    assert abs(sd["n_block_steps"] - ro.n_block_steps) <= 0.1 * ro.n_block_steps + 2
    assert sd["dt_min"] in (ro.dt_min, ro.dt_min / 2, ro.dt_min * 2)
    assert dE_d <= 2 * dE_o + 2e-8
    assert np.median(np.linalg.norm(xd - ro.x, axis=1)) < 1e-7
    # back to block steps: the run continues and stays synchronised at multiples of dt_max
    hd.set_shared_steps(False)
    hd.evolve(0.125)
    assert hd.stats()["t"] == 0.125 and hd.stats()["n_particle_steps"] < n * hd.stats()["n_block_steps"]
    hd.close()


def test_shared_steps_need_synchronised_particles(cluster):
    """g6hd_set_shared_steps(on) is refused while particles sit at different times (it would integrate wrongly without
    saying so): after a stop on max_block_steps -> G6_ERR_SEQUENCE; at a multiple of dt_max -> accepted."""
    x, v, m, _ = inputs.config("C2", n=700)
    hd = g6.HermiteDev(0, x, v, m, 1e-6, 0.01)
    hd.evolve(1.0, max_block_steps=5)
    pt = hd.particles()
    assert len(np.unique(pt["t"])) > 1
    with pytest.raises(g6.G6Error) as e:
        hd.set_shared_steps(True)
    assert e.value.code == -6
    hd.evolve(0.125)                                     # a multiple of dt_max: everybody is synchronised
    assert np.all(hd.particles()["t"] == 0.125)
    hd.set_shared_steps(True)
    hd.evolve(0.125 + 2.0 ** -10)
    assert hd.stats()["t"] >= 0.125 + 2.0 ** -10
    hd.close()
