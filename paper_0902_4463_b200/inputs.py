"""Seeded synthetic workloads (stand-ins for the paper's Plummer initial conditions).

This module holds NONE of the method's arithmetic (no forces, no prediction, no
double-single splitting): it only draws particle sets.  It is the one module the
oracle-side tests and the CUDA-side tests/bench share, so that both see the same
fp64 inputs.

Workloads follow PAPER.md:130, :138, :148 ("equal mass Plummer spheres" in N-body
units, G = M = 1, E = -1/4) and BASELINE.json `configs`; the construction is
SURVEY.md section 8(c) reading 17 and is restated in DESIGN.md ("Input recipe").
"""
from __future__ import annotations

import numpy as np

# Plummer scale length in N-body units: W = -3 pi M^2 / (32 a) = -1/2  =>  a = 3 pi / 16.
PLUMMER_A = 3.0 * np.pi / 16.0

#: the five configs of BASELINE.json (N, eps, seed); see DESIGN.md for what each is used for.
CONFIGS = {
    "C1": dict(n=1024, eps=1.0 / 256.0, seed=1024001, masses="equal"),
    "C2": dict(n=32768, eps=1.0e-4, seed=32768002, masses="equal"),
    "C3": dict(n=131072, eps=1.0e-4, seed=131072003, masses="equal"),
    "C4": dict(n=1048576, eps=1.0e-4, seed=1048576004, masses="equal"),
    "C5": dict(n=65536, eps=1.0e-5, seed=65536005, masses="salpeter",
               offset=(1000.0, 1000.0, 1000.0)),
}


def _isotropic(rng: np.random.Generator, n: int) -> np.ndarray:
    """n unit vectors, uniform on the sphere."""
    z = rng.uniform(-1.0, 1.0, n)
    phi = rng.uniform(0.0, 2.0 * np.pi, n)
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1)


def salpeter_masses(rng: np.random.Generator, n: int, m_lo: float = 0.1, m_hi: float = 100.0,
                    alpha: float = 2.35) -> np.ndarray:
    """dN/dm ~ m^-alpha on [m_lo, m_hi] by inverse transform (un-normalised masses)."""
    p = 1.0 - alpha                      # = -1.35
    u = rng.uniform(0.0, 1.0, n)
    return (m_lo ** p + u * (m_hi ** p - m_lo ** p)) ** (1.0 / p)


def plummer(n: int, seed: int, masses: str = "equal", offset=None):
    """Plummer sphere, total mass 1, scale a = 3 pi/16, no energy rescaling.

    Returns (x[n,3], v[n,3], m[n]) as fp64.  Radii by inverse transform of the
    cumulative mass M(r) = X with X ~ U(0, 0.999) (truncates r at ~22.8 a);
    speeds by von Neumann rejection on g(q) = q^2 (1-q^2)^(7/2), v = q v_esc(r);
    isotropic directions; centre of mass position and velocity removed.
    """
    rng = np.random.default_rng(seed)
    if masses == "equal":
        m = np.full(n, 1.0 / n)
    elif masses == "salpeter":
        m = salpeter_masses(rng, n)
        m = m / m.sum()
    else:
        raise ValueError(masses)

    X = rng.uniform(0.0, 0.999, n)
    X = np.maximum(X, 1e-300)
    r = PLUMMER_A / np.sqrt(X ** (-2.0 / 3.0) - 1.0)
    x = r[:, None] * _isotropic(rng, n)

    q = np.empty(n)
    todo = np.arange(n)
    while todo.size:
        qq = rng.uniform(0.0, 1.0, todo.size)
        yy = rng.uniform(0.0, 0.1, todo.size)          # max of g is ~0.092
        ok = yy < qq * qq * (1.0 - qq * qq) ** 3.5
        q[todo[ok]] = qq[ok]
        todo = todo[~ok]
    vesc = np.sqrt(2.0 / PLUMMER_A) * (1.0 + (r / PLUMMER_A) ** 2) ** (-0.25)
    v = (q * vesc)[:, None] * _isotropic(rng, n)

    mt = m.sum()
    x -= (m[:, None] * x).sum(axis=0) / mt
    v -= (m[:, None] * v).sum(axis=0) / mt
    if offset is not None:
        x = x + np.asarray(offset, dtype=np.float64)[None, :]
    return np.ascontiguousarray(x), np.ascontiguousarray(v), np.ascontiguousarray(m)


def config(name: str, n: int | None = None):
    """(x, v, m, eps2) of one BASELINE.json config; `n` overrides N (same seed) for reduced tests."""
    c = CONFIGS[name]
    x, v, m = plummer(n or c["n"], c["seed"], c["masses"], c.get("offset"))
    return x, v, m, c["eps"] ** 2


def active_subset(n: int, ni: int, seed: int) -> np.ndarray:
    """Random active block of ni distinct particle addresses (C4 n_i sweep), sorted."""
    rng = np.random.default_rng(seed)
    return np.sort(rng.choice(n, size=ni, replace=False)).astype(np.int32)


def taylor_state(n: int, seed: int, dt_max: float = 0.125):
    """Synthetic per-particle Hermite state for predictor tests: (t_j, a0, j0) with
    t_j on a power-of-two grid in (-dt_max, 0], a0 ~ O(1), j0 ~ O(10)."""
    rng = np.random.default_rng(seed)
    lev = rng.integers(3, 12, n)
    dtj = 2.0 ** (-lev.astype(np.float64))
    tj = -dtj * rng.integers(0, 2, n)
    a0 = rng.normal(0.0, 1.0, (n, 3))
    j0 = rng.normal(0.0, 10.0, (n, 3))
    return tj, dtj, a0, j0
