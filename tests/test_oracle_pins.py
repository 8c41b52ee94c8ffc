"""Pins of the CPU oracle (oracle/) against what the paper and the mathematics fix.

PAPER.md prints no worked example, so every expected value here is a closed form, an
invariant, an exact-arithmetic brute force or a bound the paper states (SURVEY.md 8(c),
pins P1-P12).  None of these tests touches the CUDA path.  Run with -m "not gpu".
"""
import os
from decimal import Decimal, getcontext
from fractions import Fraction

import numpy as np
import pytest

from paper_0902_4463_b200 import inputs

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")


def _golden():
    out = {}
    for line in open(GOLDEN):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        key, *vals = line.split()
        out[key] = [float(Fraction(v)) for v in vals]
    return out


def _rel(a, b):
    a = np.asarray(a, float); b = np.asarray(b, float)
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


# --------------------------------------------------------------------------- P1
@pytest.mark.parametrize("eps2", [0.0, 11.0])
def test_p1_two_body_closed_form(oracle, eps2):
    g = _golden()
    x = np.array([[0.0, 0, 0], [3.0, 4, 0]]); v = np.array([[0.0, 0, 0], [1.0, 0, 0]])
    m = np.array([1.0, 2.0]); idx = np.array([10, 20], np.int32)
    r = oracle.force(idx, x, v, idx, x, v, m, eps2)
    tag = f"twobody_eps2_{int(eps2)}_"
    for p in (0, 1):
        assert _rel(r["acc"][p], g[tag + f"acc{p+1}"]) < 1e-15
        assert _rel(r["jerk"][p], g[tag + f"jerk{p+1}"]) < 2e-15
        assert abs(r["pot"][p] - g[tag + f"pot{p+1}"][0]) < 1e-15 * abs(r["pot"][p])
    # each is the other's nearest neighbour; r2 is unsoftened whatever eps2 (reading 6)
    assert list(r["nn_index"]) == [20, 10] and list(r["nn_addr"]) == [1, 0]
    assert np.all(r["nn_r2"] == g["twobody_eps2_0_nn_r2"][0])


# --------------------------------------------------------------------------- P2
def test_p2_regular_polygon(oracle):
    g = _golden()
    for n, m, R in [(4, 0.5, 2.0), (7, 0.3, 1.7), (24, 1.0 / 24, 0.9)]:
        th = 2 * np.pi * np.arange(n) / n
        x = np.stack([R * np.cos(th), R * np.sin(th), np.zeros(n)], 1)
        v = np.zeros((n, 3)); idx = np.arange(n, dtype=np.int32)
        r = oracle.force(idx, x, v, idx, x, v, np.full(n, m), 0.0)
        S = np.sum(1.0 / np.sin(np.pi * np.arange(1, n) / n))
        amag = m / R**2 * 0.25 * S
        assert np.allclose(np.linalg.norm(r["acc"], axis=1), amag, rtol=1e-14)
        # pointing to the centre
        assert np.allclose(r["acc"], -amag * x / R, rtol=0, atol=1e-13 * amag)   # positions carry cos/sin rounding
        assert np.allclose(r["pot"], -m / (2 * R) * S, rtol=1e-14)
        assert np.abs(r["jerk"]).max() == 0.0
        if n == 4:
            assert abs(np.linalg.norm(r["acc"][0]) - g["polygon_n4_m0.5_R2_absacc"][0]) < 1e-14
            assert abs(r["pot"][0] - g["polygon_n4_m0.5_R2_pot"][0]) < 1e-14


# --------------------------------------------------------------------------- P3, P4
def _cloud(n, seed):
    rng = np.random.default_rng(seed)
    return rng.normal(size=(n, 3)), rng.uniform(0.5, 1.5, n) / n


@pytest.mark.parametrize("eps2", [0.0, 0.01])
def test_p3_rigid_rotation_plus_translation(oracle, eps2):
    """v = Omega x X + u  =>  adot = Omega x a: pins the dv term, the factor 3 and the sign."""
    x, m = _cloud(200, 3)
    Om = np.array([0.3, -1.1, 0.7]); u = np.array([5.0, -2.0, 1.0])
    v = np.cross(Om, x) + u
    idx = np.arange(len(m), dtype=np.int32)
    r = oracle.force(idx, x, v, idx, x, v, m, eps2)
    want = np.cross(Om, r["acc"])
    err = np.linalg.norm(r["jerk"] - want, axis=1) / np.linalg.norm(want, axis=1)
    assert err.max() < 1e-13


def test_p4_homologous_expansion(oracle):
    """v = H x, eps = 0  =>  adot = -2 H a."""
    x, m = _cloud(200, 4)
    H = 0.37
    idx = np.arange(len(m), dtype=np.int32)
    r = oracle.force(idx, x, H * x, idx, x, H * x, m, 0.0)
    err = np.linalg.norm(r["jerk"] + 2 * H * r["acc"], axis=1) / np.linalg.norm(r["acc"], axis=1)
    assert err.max() < 1e-13


# --------------------------------------------------------------------------- P5
def test_p5_newtons_third_law(oracle):
    x, v, m, eps2 = inputs.config("C5", n=2048)      # unequal masses, offset cluster
    x = x - 1000.0                                     # keep fp64 cancellation out of this pin
    idx = np.arange(len(m), dtype=np.int32)
    r = oracle.force(idx, x, v, idx, x, v, m, eps2)
    for q in ("acc", "jerk"):
        tot = np.linalg.norm((m[:, None] * r[q]).sum(0))
        scale = (m * np.linalg.norm(r[q], axis=1)).sum()
        assert tot / scale < 1e-13, (q, tot / scale)


# --------------------------------------------------------------------------- P6
@pytest.mark.parametrize("n,seed", [(4096, 11), (16384, 12)])
def test_p6_plummer_virial(oracle, n, seed):
    """Un-rescaled Plummer sphere in N-body units: W -> -1/2, T -> 1/4 (north_star)."""
    x, v, m = inputs.plummer(n, seed)
    eps2 = (1.0 / 256) ** 2 if n <= 4096 else 1e-8
    idx = np.arange(n, dtype=np.int32)
    r = oracle.force(idx, x, v, idx, x, v, m, eps2)
    W = 0.5 * np.sum(m * r["pot"])
    T, W2 = oracle.energy(x, v, m, eps2)
    assert abs(W - W2) < 1e-12 * abs(W)                 # two routes to W agree (pair sum vs phi sum)
    tol = 1.5 / np.sqrt(n) + 0.003
    assert abs(W + 0.5) < tol, W
    assert abs(T - 0.25) < tol, T
    assert abs(T + W + 0.25) < 1.5 * tol


# --------------------------------------------------------------------------- P7
def _decimal_force(index_i, xi, vi, index_j, xj, vj, mj, eps2):
    """Independent 50-digit brute force, written from the potential: a = -grad_i phi-sum etc.
    (explicit formulas in a different algebraic form: everything divided, nothing multiplied
    by reciprocals)."""
    getcontext().prec = 50
    D = lambda t: Decimal(repr(float(t)))
    ni, nj = len(index_i), len(index_j)
    acc = np.zeros((ni, 3)); jerk = np.zeros((ni, 3)); pot = np.zeros(ni)
    for i in range(ni):
        A = [Decimal(0)] * 3; J = [Decimal(0)] * 3; P = Decimal(0)
        for j in range(nj):
            if index_j[j] == index_i[i]:
                continue
            d = [D(xj[j][k]) - D(xi[i][k]) for k in range(3)]
            w = [D(vj[j][k]) - D(vi[i][k]) for k in range(3)]
            s2 = sum(t * t for t in d) + D(eps2)
            s = s2.sqrt()
            dw = sum(p * q for p, q in zip(d, w))
            mm = D(mj[j])
            P -= mm / s
            for k in range(3):
                A[k] += mm * d[k] / (s2 * s)
                J[k] += mm * w[k] / (s2 * s) - 3 * mm * dw * d[k] / (s2 * s2 * s)
        acc[i] = [float(t) for t in A]; jerk[i] = [float(t) for t in J]; pot[i] = float(P)
    return acc, jerk, pot


def test_p7_exact_brute_force(oracle):
    x, v, m, _ = inputs.config("C1", n=48)
    idx = np.arange(48, dtype=np.int32) * 3 + 1
    for eps2 in (0.0, (1.0 / 256) ** 2):
        acc, jerk, pot = _decimal_force(idx[:20], x[:20], v[:20], idx, x, v, m, eps2)
        for ld in (False, True):
            r = oracle.force(idx[:20], x[:20], v[:20], idx, x, v, m, eps2, long_double=ld)
            tol = 1e-13 if not ld else 2e-15
            assert max(_rel(r["acc"][i], acc[i]) for i in range(20)) < tol
            assert max(_rel(r["jerk"][i], jerk[i]) for i in range(20)) < 20 * tol
            assert np.max(np.abs(r["pot"] - pot) / np.abs(pot)) < tol


def test_p7_long_double_build_is_wider(oracle):
    from oracle import oracle as orc
    orc.build(True)
    assert orc._lib(True).orc_sizeof_real() > orc._lib(False).orc_sizeof_real()


# --------------------------------------------------------------------------- P8
def test_p8_translation_invariance(oracle):
    x, v, m, eps2 = inputs.config("C1", n=512)
    idx = np.arange(512, dtype=np.int32)
    r0 = oracle.force(idx, x, v, idx, x, v, m, eps2)
    c = 1024.0                                         # exactly representable shift
    xs = x + c
    r1 = oracle.force(idx, xs, v, idx, xs, v, m, eps2)
    # the shifted positions are re-rounded to fp64: relative separation error <= 2^-53 c / r_min
    rmin = np.sqrt(r0["nn_r2"].min())
    bound = 64 * 2.0**-53 * c / rmin
    err = np.linalg.norm(r1["acc"] - r0["acc"], axis=1) / np.linalg.norm(r0["acc"], axis=1)
    assert err.max() < bound
    assert err.max() > 0.0                             # and the shift really changed the inputs
    assert np.array_equal(r0["nn_index"], r1["nn_index"])


# --------------------------------------------------------------------------- P9
def test_p9_predictor_is_the_cubic(oracle):
    """Eq. 1-2 against exact rational arithmetic; dt = t_i - t_j (reading 3); dt = 0 is the identity."""
    n = 64
    rng = np.random.default_rng(9)
    x0 = rng.normal(size=(n, 3)); v0 = rng.normal(size=(n, 3))
    tj, dtj, a0, j0 = inputs.taylor_state(n, 9)
    ti = 0.0625
    xp, vp = oracle.predict(ti, tj, x0, v0, a0, j0)
    F = Fraction
    for p in range(n):
        dt = F(ti) - F(float(tj[p]))
        for k in range(3):
            ex = F(float(x0[p, k])) + F(float(v0[p, k])) * dt + F(float(a0[p, k])) * dt**2 / 2 + F(float(j0[p, k])) * dt**3 / 6
            ev = F(float(v0[p, k])) + F(float(a0[p, k])) * dt + F(float(j0[p, k])) * dt**2 / 2
            assert abs(xp[p, k] - float(ex)) <= 4e-16 * max(1.0, abs(float(ex)))
            assert abs(vp[p, k] - float(ev)) <= 4e-16 * max(1.0, abs(float(ev)))
    xq, vq = oracle.predict(0.25, np.full(n, 0.25), x0, v0, a0, j0)
    assert np.array_equal(xq, x0) and np.array_equal(vq, v0)
    # a swapped a0/j0, a missing 1/2 or 1/6 each move the result by far more than the tolerance
    xw, _ = oracle.predict(ti, tj, x0, v0, j0, a0)
    assert np.abs(xw - xp).max() > 1e-6


# --------------------------------------------------------------------------- P10
def test_p10_phi_self_term_and_index_exclusion(oracle):
    """Exclusion is by INDEX (reading 4): the same i-particles handed in under indices that
    match no j see their own copy at zero distance -> phi shifts by exactly -m_i/eps, a and
    adot do not move (dx = 0), and the nearest neighbour becomes the particle itself."""
    x, v, m, eps2 = inputs.config("C5", n=256)
    idx = np.arange(256, dtype=np.int32) + 100
    r = oracle.force(idx, x, v, idx, x, v, m, eps2)
    rs = oracle.force(idx + 10000, x, v, idx, x, v, m, eps2)
    assert np.allclose(rs["pot"] - r["pot"], -m / np.sqrt(eps2), rtol=1e-9)
    assert np.allclose(rs["acc"], r["acc"], rtol=1e-12, atol=0)
    assert np.array_equal(rs["nn_index"], idx) and np.all(rs["nn_r2"] == 0.0)
    assert not np.any(r["nn_index"] == idx)


def test_nearest_neighbour_rules(oracle):
    """argmin of unsoftened r2 (reading 6), ties -> smallest address (7), none -> -1 / inf (8),
    coincident distinct particles with eps = 0 are skipped (5)."""
    x, v, m, _ = inputs.config("C1", n=300)
    idx = (np.arange(300, dtype=np.int32) * 7) % 300 + 5     # a permutation, index != address
    r = oracle.force(idx, x, v, idx, x, v, m, 1.0)            # huge softening must not matter
    d2 = ((x[:, None, :] - x[None, :, :]) ** 2).sum(-1)
    np.fill_diagonal(d2, np.inf)
    assert np.array_equal(r["nn_addr"], d2.argmin(1))
    assert np.array_equal(r["nn_index"], idx[d2.argmin(1)])
    assert np.allclose(r["nn_r2"], d2.min(1), rtol=1e-15)
    # tie: i at the origin, two j at the same distance -> the smaller address wins
    xi = np.zeros((1, 3)); xj = np.array([[2.0, 0, 0], [0, 1.0, 0], [0, 0, -1.0], [1.0, 0, 0]])
    z = np.zeros_like(xj)
    t = oracle.force([99], xi, xi, [3, 2, 1, 0], xj, z, np.ones(4), 0.25)
    assert t["nn_addr"][0] == 1 and t["nn_index"][0] == 2 and t["nn_r2"][0] == 1.0
    # none: the only j is the particle itself
    t = oracle.force([7], xi, xi, [7], xi, xi, np.ones(1), 0.25)
    assert t["nn_index"][0] == -1 and t["nn_addr"][0] == -1 and np.isinf(t["nn_r2"][0])
    assert t["pot"][0] == 0.0 and np.all(t["acc"] == 0.0)
    # coincident distinct particle, eps = 0: skipped, no NaN
    t = oracle.force([7], xi, xi, [8, 9], np.array([[0.0, 0, 0], [0, 3.0, 4.0]]), np.zeros((2, 3)), np.ones(2), 0.0)
    assert t["nn_index"][0] == 9 and np.isclose(t["pot"][0], -0.2) and np.all(np.isfinite(t["acc"]))


# --------------------------------------------------------------------------- P11 (CPU half)
def test_p11_double_single(oracle):
    """DS split invariants and the accuracy of Eq. 3."""
    rng = np.random.default_rng(11)
    x = np.concatenate([rng.normal(size=4000), 1000.0 + rng.normal(size=4000) * 1e-3,
                        [0.0, 1.0, -1.0, 2.0**-30, 1e6 + 2.0**-20, 16777217.0]])
    hi, lo = oracle.ds_split(x)
    assert hi.dtype == np.float32 and lo.dtype == np.float32
    ulp = np.spacing(np.abs(hi))
    assert np.all(np.abs(lo.astype(np.float64)) <= 0.5 * ulp.astype(np.float64))      # |lo| <= ulp(hi)/2
    back = hi.astype(np.float64) + lo.astype(np.float64)
    nz = x != 0
    # 24 + 24 = 48 bits of mantissa ("48 bits in DS"): relative error <= 2^-48
    assert np.max(np.abs(back[nz] - x[nz]) / np.abs(x[nz])) <= 2.0**-48
    # Eq. 3 on an offset cluster: "one part in ten millions or better"
    xi = 1000.0 + rng.normal(size=20000) * 1e-2
    xj = 1000.0 + rng.normal(size=20000) * 1e-2
    ih, il = oracle.ds_split(xi); jh, jl = oracle.ds_split(xj)
    dx = oracle.ds_diff(jh, jl, ih, il).astype(np.float64)
    exact = xj - xi
    bound = 3 * 2.0**-24 * np.abs(exact) + 2.0**-47 * np.maximum(np.abs(xi), np.abs(xj))
    assert np.all(np.abs(dx - exact) <= bound)
    big = np.abs(exact) > 1e-4
    assert np.max(np.abs(dx[big] - exact[big]) / np.abs(exact[big])) < 1e-7
    # and pure single precision is orders of magnitude worse there (the paper's motivation, :110)
    sp = (jh - ih).astype(np.float64)
    assert np.median(np.abs(sp - exact)) > 100 * np.median(np.abs(dx - exact))
    # hand-checked example: x = 1 + 2^-30 -> hi = 1, lo = 2^-30
    h, l = oracle.ds_split(np.array([1.0 + 2.0**-30]))
    assert h[0] == 1.0 and l[0] == np.float32(2.0**-30)


# --------------------------------------------------------------------------- P12 (generators)
def test_p12_salpeter_and_plummer_generators():
    rng = np.random.default_rng(12)
    m = inputs.salpeter_masses(rng, 400000)
    assert m.min() >= 0.1 and m.max() <= 100.0
    # closed forms for dN/dm ~ m^-2.35 on [0.1, 100]
    p = -1.35
    lo, hi = 0.1**p, 100.0**p
    median = (lo + 0.5 * (hi - lo)) ** (1 / p)
    mean = (p / (p + 1)) * (100.0 ** (p + 1) - 0.1 ** (p + 1)) / (hi - lo)
    assert abs(median - 0.16709) < 1e-4 and abs(mean - 0.35137) < 1e-4     # SURVEY P12 numbers
    assert abs(np.median(m) - median) < 0.01 * median
    x, v, mm = inputs.plummer(20000, 5)
    assert abs(mm.sum() - 1) < 1e-12
    assert np.abs((mm[:, None] * x).sum(0)).max() < 1e-12 and np.abs((mm[:, None] * v).sum(0)).max() < 1e-12
    # half-mass radius of a Plummer sphere: a / sqrt(2^(2/3) - 1) = 1.3048 a (truncation shifts it < 1%)
    r = np.sort(np.linalg.norm(x, axis=1))
    assert abs(r[len(r) // 2] / inputs.PLUMMER_A - 1.3048) < 0.04
    assert r.max() < 22.9      # X < 0.999 cuts r at a / sqrt(0.999^(-2/3) - 1) = 22.8
    # determinism
    x2, _, _ = inputs.plummer(20000, 5)
    assert np.array_equal(x, x2)


# --------------------------------------------------------------------------- Hermite oracle
def _binary(d, e=0.0):
    """two equal masses 1/2, separation d at apocentre, eccentricity e, in the x-y plane."""
    m = np.array([0.5, 0.5])
    vrel = np.sqrt((1 - e) / d)               # apocentre speed for semi-major axis a = d/(1+e), M = 1
    x = np.array([[-d / 2, 0, 0], [d / 2, 0, 0]])
    v = np.array([[0, -vrel / 2, 0], [0, vrel / 2, 0]])
    return x, v, m


def test_hermite_oracle_circular_binary_period(oracle):
    """Kepler: P = 2 pi sqrt(a^3 / M).  With a = (2 pi)^(-2/3) the period is exactly 1."""
    d = (2 * np.pi) ** (-2.0 / 3.0)
    x, v, m = _binary(d)
    r = oracle.hermite(x, v, m, 0.0, 0.002, 1.0)
    assert r.t == 1.0
    assert np.abs(r.x - x).max() < 2e-6 and np.abs(r.v - v).max() < 2e-5
    # half a period: positions swapped
    r = oracle.hermite(x, v, m, 0.0, 0.002, 0.5)
    assert np.abs(r.x + x).max() < 2e-6


def test_hermite_oracle_fourth_order_and_blocks(oracle):
    """Energy error of an eccentric binary falls ~ eta^2 (4th-order scheme: dE ~ dt^4 ~ eta^2)."""
    a = (2 * np.pi) ** (-2.0 / 3.0); e = 0.5
    x, v, m = _binary(a * (1 + e), e)
    E0 = sum(oracle.energy(x, v, m, 0.0))
    assert abs(E0 + 0.125 / a) < 1e-13 * abs(E0)          # two-body energy -m1 m2 / (2a) with m1 = m2 = 1/2
    errs = []
    for eta in (0.04, 0.01):
        r = oracle.hermite(x, v, m, 0.0, eta, 1.0)
        errs.append(abs(sum(oracle.energy(r.x, r.v, m, 0.0)) - E0) / abs(E0))
        assert r.t == 1.0 and r.n_particle_steps == 2 * r.n_block_steps   # both always in the same block
    assert errs[1] < errs[0] / 6 and errs[1] < 1e-6, errs
    # a small cluster: block steps are hierarchical, stats are consistent, energy conserved
    x, v, m, eps2 = inputs.config("C1", n=128)
    E0 = sum(oracle.energy(x, v, m, eps2))
    r = oracle.hermite(x, v, m, eps2, 0.01, 0.125)
    assert r.t == 0.125 and r.n_particle_steps >= 128 and r.ni_hist_log2.sum() == r.n_block_steps
    assert np.log2(r.dt_min) == np.round(np.log2(r.dt_min)) and r.dt_min <= 0.125
    assert abs(sum(oracle.energy(r.x, r.v, m, eps2)) - E0) / abs(E0) < 1e-7


def test_hermite_corrector_exact_for_cubic_acceleration(oracle):
    """The corrector reproduces x(h), v(h) exactly when a(t) is a cubic in t (then x is a
    quintic): pins every coefficient (1/6, 1/24, 1/120, the -6/4/2 and 12/6 of a2, a3)."""
    F = Fraction
    rng = np.random.default_rng(16)
    for h in (0.125, 2.0**-7):
        c = [[F(float(t)) for t in rng.integers(-8, 9, 3)] for _ in range(6)]   # x0 v0 a0 ad0 a2 a3
        hh = F(h)
        fact = [1, 1, 2, 6, 24, 120]
        def poly(first, k):      # derivative `first` of x at time hh, component k
            return sum(c[n][k] * hh ** (n - first) / fact[n - first] for n in range(first, 6))
        xp = [float(sum(c[n][k] * hh**n / fact[n] for n in range(4))) for k in range(3)]   # Eq. 1
        vp = [float(sum(c[n][k] * hh**(n - 1) / fact[n - 1] for n in range(1, 4))) for k in range(3)]
        a0 = [float(c[2][k]) for k in range(3)]; ad0 = [float(c[3][k]) for k in range(3)]
        a1 = [float(poly(2, k)) for k in range(3)]; ad1 = [float(poly(3, k)) for k in range(3)]
        x1, v1, a2n, a3 = oracle.hermite_correct(h, xp, vp, a0, ad0, a1, ad1)
        for k in range(3):
            assert abs(x1[k] - float(poly(0, k))) <= 1e-14 * max(1, abs(float(poly(0, k))))
            assert abs(v1[k] - float(poly(1, k))) <= 1e-13 * max(1, abs(float(poly(1, k))))
            assert abs(a3[k] - float(c[5][k])) <= 1e-9 * max(1, abs(float(c[5][k]))) / h
            assert abs(a2n[k] - float(poly(4, k))) <= 1e-9 * max(1, abs(float(poly(4, k)))) / h


def test_aarseth_step_closed_form(oracle):
    """a(t) = A exp(lambda t) along one axis: every ratio of successive derivatives is lambda,
    so the criterion gives dt = sqrt(eta) / lambda."""
    A, lam, eta = 2.5, 7.0, 0.01
    e = np.array([1.0, 0, 0])
    dt = oracle.aarseth_dt(eta, A * e, lam * A * e, lam**2 * A * e, lam**3 * A * e)
    assert abs(dt - np.sqrt(eta) / lam) < 1e-15


# ---- P13: neighbour lists (reading 20) -------------------------------------
def test_p13_neighbour_lists_lattice_shell_counts(oracle):
    """On the integer lattice the number of points at squared distance n from a lattice point is
    r3(n), the number of representations of n as a sum of three squares: 6, 12, 8, 6, 24, 24, 0, 12, 30
    for n = 1..9 (number theory, e.g. OEIS A005875).  Strict '<': a point AT h2 is not a neighbour."""
    g = np.arange(-4, 5)
    X = np.array(np.meshgrid(g, g, g, indexing="ij"), dtype=float).reshape(3, -1).T + np.array([10.0, -7.0, 3.0])
    n = len(X)
    idx = np.arange(n, dtype=np.int32)
    c = int(np.nonzero((X == np.array([10.0, -7.0, 3.0])).all(axis=1))[0][0])
    r3 = [6, 12, 8, 6, 24, 24, 0, 12, 30]
    want = np.cumsum(r3)
    for k in range(9):
        cnt, lst = oracle.neighbours(idx[c:c + 1], X[c:c + 1], [k + 1.5], idx, X, maxlen=256)
        assert cnt[0] == want[k]
        got = lst[0, :cnt[0]]
        assert (np.diff(got) > 0).all() and c not in got                       # increasing addresses, self excluded by index
        d2 = ((X[got] - X[c]) ** 2).sum(axis=1)
        assert (d2 < k + 1.5).all()
        cnt_eq, _ = oracle.neighbours(idx[c:c + 1], X[c:c + 1], [float(k + 1)], idx, X, maxlen=256)
        assert cnt_eq[0] == (want[k - 1] if k else 0)                         # strict inequality
    # same answer from the long-double build
    cnt_l, lst_l = oracle.neighbours(idx[c:c + 1], X[c:c + 1], [6.5], idx, X, maxlen=256, long_double=True)
    cnt_d, lst_d = oracle.neighbours(idx[c:c + 1], X[c:c + 1], [6.5], idx, X, maxlen=256)
    assert cnt_l[0] == cnt_d[0] == 80 and (lst_l == lst_d).all()


def test_p13_neighbour_lists_brute_force_overflow_and_nearest(oracle):
    rng = np.random.default_rng(13)
    n = 400
    X = rng.normal(size=(n, 3)); V = rng.normal(size=(n, 3)); m = np.full(n, 1.0 / n)
    idx = rng.permutation(n).astype(np.int32) + 1000                          # index != address
    h2 = rng.uniform(0.05, 0.6, size=n)
    cnt, lst = oracle.neighbours(idx, X, h2, idx, X, maxlen=8)
    for i in range(n):                                                        # numpy brute force, pair by pair
        d2 = ((X - X[i]) ** 2).sum(axis=1)
        want = np.nonzero((d2 < h2[i]) & (idx != idx[i]))[0]
        assert cnt[i] == len(want)
        k = min(len(want), 8)
        assert (lst[i, :k] == want[:k]).all() and (lst[i, k:] == -1).all()   # overflow: count keeps counting, list = first maxlen
    assert (cnt > 8).any() and (cnt < 8).any()
    # the nearest neighbour of orc_force heads the set: with h2 just above its distance the list is exactly that particle
    f = oracle.force(idx, X, V, idx, X, V, m, 0.0)
    cnt1, lst1 = oracle.neighbours(idx, X, f["nn_r2"] * (1 + 1e-12), idx, X, maxlen=4)
    assert (cnt1 == 1).all() and (lst1[:, 0] == f["nn_addr"]).all()
    cnt0, _ = oracle.neighbours(idx, X, f["nn_r2"], idx, X, maxlen=4)          # at the distance itself: nobody (strict)
    assert (cnt0 == 0).all()
    # same index, different address (an i-particle that is also stored as a j): excluded by INDEX, not position
    Xs = X.copy(); Xs[7] += 0.01
    cnt2, lst2 = oracle.neighbours(idx[7:8], Xs[7:8], [0.5], idx, X, maxlen=64)
    assert 7 not in lst2[0, :cnt2[0]]


def test_hermite_oracle_shared_steps(oracle):
    """Shared-time-step variant (reading 21; "shared or block time steps").
    (i) A square of equal masses on a circular orbit: the four particles are images of one another under 90-degree
    rotations, which only permute and negate coordinates, so they ask for bit-identical steps and the shared scheme
    must reproduce the (pinned) block scheme bit for bit.  (ii) On a cluster every particle takes every step, the
    common step is never larger than the block scheme's smallest, and the energy is conserved at least as well."""
    R, mass = 1.0, 0.25
    x = np.array([[R, 0, 0], [0, R, 0], [-R, 0, 0], [0, -R, 0]], float)
    a = mass / R ** 2 * 0.25 * sum(1 / np.sin(np.pi * k / 4) for k in range(1, 4))      # polygon closed form (pin P2)
    vc = np.sqrt(a * R)
    v = np.array([[0, vc, 0], [-vc, 0, 0], [0, -vc, 0], [vc, 0, 0]], float)
    m = np.full(4, mass)
    rb = oracle.hermite(x, v, m, 0.0, 0.01, 0.5)
    rs = oracle.hermite(x, v, m, 0.0, 0.01, 0.5, shared=True)
    assert np.array_equal(rb.x, rs.x) and np.array_equal(rb.v, rs.v)
    assert rb.n_block_steps == rs.n_block_steps and rs.n_particle_steps == 4 * rs.n_block_steps
    assert np.allclose(np.linalg.norm(rs.x, axis=1), R, rtol=1e-7)                        # still on the circle
    # (ii)
    x, v, m, eps2 = inputs.config("C1", n=64)
    E0 = sum(oracle.energy(x, v, m, eps2))
    rb = oracle.hermite(x, v, m, eps2, 0.01, 0.125)
    rs = oracle.hermite(x, v, m, eps2, 0.01, 0.125, shared=True)
    assert rs.t == 0.125 and rs.n_particle_steps == 64 * rs.n_block_steps
    assert rs.ni_hist_log2[6] == rs.n_block_steps and rs.ni_hist_log2.sum() == rs.n_block_steps
    assert rs.dt_min <= rb.dt_min and rs.n_particle_steps > rb.n_particle_steps
    dEs = abs(sum(oracle.energy(rs.x, rs.v, m, eps2)) - E0) / abs(E0)
    dEb = abs(sum(oracle.energy(rb.x, rb.v, m, eps2)) - E0) / abs(E0)
    assert dEs < 1e-7 and dEs <= 2 * dEb + 1e-12, (dEs, dEb)
