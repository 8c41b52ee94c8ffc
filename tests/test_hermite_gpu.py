"""The host Hermite driver (g6h_*, step a-7) driving the CUDA library, against the oracle-driven
integrator (oracle/hermite_oracle.c) on the same seeded inputs."""
import time

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


@pytest.mark.skipif(not __import__("os").environ.get("G6_FULL_C2"), reason="minutes of CPU: set G6_FULL_C2=1 (results recorded in profiles/)")
def test_c2_full_run_vs_oracle_driven(cluster, oracle):
    """BASELINE.json config 2 in full: N = 32768, t = 0 -> 1, library-driven and oracle-driven."""
    import json, os
    t_end = float(os.environ.get("G6_C2_TEND", "1.0"))
    x, v, m, eps2 = inputs.config("C2")
    eta = 0.01
    E0 = _energy(oracle, x, v, m, eps2)
    rep = {"config": "C2", "n": len(m), "eta": eta, "eps2": eps2, "t_end": t_end, "E0": E0, "oracle_threads": oracle.threads()}
    for newton in (1, 0):
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
