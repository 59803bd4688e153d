"""Pins for the CPU oracle (oracle/top_oracle.c) and its direct solvers -- all `not gpu`.

Each test checks the oracle against something the paper or the mathematics fixes and that is NOT the
oracle's own formula retyped: textbook closed forms (tests/golden/closed_forms.json), a dense KKT solve,
the optimality conditions as a banded system, scipy's SLSQP on a tiny constrained instance, the KKT
certificate of the converged iterate, and per-iterate invariants of the projections.
SURVEY.md section 8(c) pins P1..P11.
"""
import json
import os

import numpy as np
import pytest
import scipy.integrate
import scipy.optimize

from oracle import direct
from oracle.top_oracle import Oracle, eval_poly
from paper_2507_10290_b200 import workloads as W

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "closed_forms.json")))


def scaled(c, T):
    """c^_k = c_k T^k (metres): the norm in which coefficients are compared (reading A12)."""
    n = c.shape[-1]
    return c * (np.asarray(T)[:, None, None] ** np.arange(n)[None, None, :])


def relerr(a, b, T):
    return np.abs(scaled(a - b, T)).max() / np.abs(scaled(b, T)).max()


# ---------------------------------------------------------------- P1 / P2: closed forms from the golden file
@pytest.mark.parametrize("s,key", [(3, "jerk"), (4, "snap")])
def test_P1_closed_form_single_segment(s, key):
    L, T = 3.0, 2.0
    unit = np.array(GOLD[key + "_unit_coeffs"], dtype=float)
    want = L * unit / T ** np.arange(2 * s)
    want_cost = GOLD[key + "_cost_factor"] * L * L / T ** GOLD[key + "_cost_T_power"]
    wp = np.array([[0.0, 1.0, -2.0], [L, 1.0, -2.0]])
    # direct solvers
    for solver in (direct.dense_kkt, direct.banded_optimality):
        c = solver(wp, np.array([T]), s)
        assert np.abs(c[0, 0] - want).max() < 1e-11
        assert np.abs(c[0, 1] - np.eye(2 * s)[0] * 1.0).max() < 1e-11      # constant dimension
        assert abs(direct.objective(c, [T], s) - want_cost) < 1e-9 * want_cost
    cf, cost = direct.closed_form_rest_to_rest(s, L, T)
    assert np.allclose(cf, want) and abs(cost - want_cost) < 1e-12 * want_cost
    # the CADMM oracle: N=1, z_0 and z_1 fixed (method of multipliers on one segment)
    for mode in ("hard", "pinned_z"):
        o = Oracle(wp, np.array([T]), s, rho=100.0, mode=mode)
        o.sweep(3000)
        c = o.get("coeffs")
        assert np.abs(c[0, 0] - want).max() < 1e-9, mode
        assert abs(o.objective() - want_cost) < 1e-8 * want_cost
        assert o.residuals()["r_p"] < 1e-9


def test_P2_Q_textbook_block_and_quadrature():
    T = 1.7
    o = Oracle(np.zeros((2, 3)) + np.array([[0.0], [1.0]]), np.array([T]), 3, rho=1.0)
    Q = o.get("Q")[0]
    coeff = np.array(GOLD["Q_jerk_block_coeff"], dtype=float)
    power = np.array(GOLD["Q_jerk_block_power"], dtype=float)
    assert np.allclose(Q[3:, 3:], coeff * T ** power, rtol=1e-14)
    assert np.all(Q[:3, :] == 0) and np.all(Q[:, :3] == 0)
    # independent check for s=4 by numerical quadrature of beta^(4) beta^(4)'
    o4 = Oracle(np.zeros((2, 3)) + np.array([[0.0], [1.0]]), np.array([T]), 4, rho=1.0)
    Q4 = o4.get("Q")[0]
    for j in range(8):
        for l in range(8):
            f = lambda t: direct.beta(8, 4, t)[j] * direct.beta(8, 4, t)[l]
            val, _ = scipy.integrate.quad(f, 0.0, T, epsabs=1e-10, epsrel=1e-12)
            assert abs(Q4[j, l] - val) <= 1e-9 * max(1.0, abs(val))


def test_M_and_E_rows_are_derivatives_of_the_polynomial():
    """M c and E_k c must equal numpy.polynomial derivatives at 0, T and the sample times t_j = T j/(Ms+1)."""
    rng = np.random.default_rng(0)
    T, s, Ms = 1.3, 4, 8
    o = Oracle(rng.normal(size=(2, 3)), np.array([T]), s, 1.0, samples=Ms, vmax=1.0, amax=1.0,
               box_lo=-np.ones((1, 3)) * 9, box_hi=np.ones((1, 3)) * 9)
    M, E = o.get("M")[0], [o.get("E%d" % k)[0] for k in range(3)]
    c = rng.normal(size=8)
    P = np.polynomial.Polynomial(c)
    for k in range(s):
        assert np.isclose(M[k] @ c, P.deriv(k)(0.0) if k else P(0.0))
        assert np.isclose(M[s + k] @ c, P.deriv(k)(T) if k else P(T))
    for k in range(3):
        for j in range(Ms):
            t = T * (j + 1) / (Ms + 1)
            assert np.isclose(E[k][j] @ c, P.deriv(k)(t) if k else P(t))


# ---------------------------------------------------------------- P3 / P4' / P5 / P6: direct solvers
@pytest.mark.parametrize("s", [3, 4])
@pytest.mark.parametrize("N", [2, 3, 4, 50])
def test_P3_P4_dense_kkt_equals_banded_optimality(s, N):
    rng = np.random.default_rng(10 * N + s)
    wp = np.cumsum(rng.normal(size=(N + 1, 3)), axis=0)
    T = rng.uniform(0.5, 2.5, size=N)
    sd, ed = rng.normal(size=(s - 1, 3)), rng.normal(size=(s - 1, 3))
    a = direct.dense_kkt(wp, T, s, sd, ed)
    b = direct.banded_optimality(wp, T, s, sd, ed)
    assert relerr(a, b, T) < 1e-10
    # P5: emergent smoothness -- the KKT solution (which only imposed C^{s-1}) is C^{2s-2}
    for k in range(2 * s - 1):
        end = eval_poly(a, T, k, [1.0])[:-1, 0]
        start = eval_poly(a, T, k, [0.0])[1:, 0]
        scale = max(1.0, np.abs(end).max())
        assert np.abs(end - start).max() < 1e-7 * scale, k
    # boundary states
    for k in range(1, s):
        assert np.allclose(eval_poly(a, T, k, [0.0])[0, 0], sd[k - 1], atol=1e-9)
        assert np.allclose(eval_poly(a, T, k, [1.0])[-1, 0], ed[k - 1], atol=1e-9)


@pytest.mark.parametrize("s,key", [(3, "jerk"), (4, "snap")])
def test_P6_single_polynomial_invariant(s, key):
    """Waypoints sampled from ONE rest-to-rest optimal polynomial at the knot times: every piece must be its Taylor shift."""
    Ttot, L = 6.0, 5.0
    unit = np.array(GOLD[key + "_unit_coeffs"], dtype=float)
    big = np.polynomial.Polynomial(L * unit / Ttot ** np.arange(2 * s))
    knots = np.array([0.0, 0.9, 2.2, 3.1, 4.7, 6.0])
    wp = np.stack([big(knots), -2 * big(knots), 0 * knots + 1.0], axis=1)
    T = np.diff(knots)
    for solver in (direct.dense_kkt, direct.banded_optimality):
        c = solver(wp, T, s)
        for i in range(T.size):
            taylor = np.array([big.deriv(k)(knots[i]) if k else big(knots[i]) for k in range(2 * s)]) \
                     / np.array([float(np.prod(np.arange(1, k + 1))) for k in range(2 * s)])
            assert np.abs((c[i, 0] - taylor) * T[i] ** np.arange(2 * s)).max() < 1e-10


# ---------------------------------------------------------------- P7: CADMM -> direct solution
@pytest.mark.parametrize("mode,tol", [("hard", 1e-8), ("pinned_z", 1e-6)])
def test_P7_config1_converges_to_direct_solution(mode, tol):
    w = W.config1()
    o = Oracle(w.waypoints[0], w.durations[0], w.s, w.rho, mode=mode)
    o.sweep(w.sweeps)
    ref = direct.dense_kkt(w.waypoints[0], w.durations[0], w.s)
    assert relerr(o.get("coeffs"), ref, w.durations[0]) < tol
    r = o.residuals()
    assert r["r_p"] < 1e-5 and r["r_p_gap"] < 1e-5
    # C^{s-1} continuity at every junction follows from r_p -> 0
    c = o.get("coeffs")
    for k in range(w.s):
        gap = eval_poly(c, w.durations[0], k, [1.0])[:-1, 0] - eval_poly(c, w.durations[0], k, [0.0])[1:, 0]
        assert np.abs(gap).max() < 1e-5


@pytest.mark.parametrize("s,N", [(3, 2), (3, 4), (4, 3)])
def test_P7_small_N_brute_force(s, N):
    rng = np.random.default_rng(100 + N)
    wp = np.cumsum(rng.uniform(-2, 2, size=(N + 1, 3)), axis=0)
    T = rng.uniform(0.8, 1.6, size=N)
    o = Oracle(wp, T, s, rho=10.0)
    o.solve(1e-11, 400000, use_rd_norm=True)
    assert relerr(o.get("coeffs"), direct.dense_kkt(wp, T, s), T) < 1e-8
    # FREE mode (paper's Alg. 1 verbatim) must NOT reach the fixed-waypoint solution: its unconstrained
    # limit is the single rest-to-rest polynomial from p_0 to p_N (waypoints are free)
    f = Oracle(wp, T, s, rho=10.0, mode="free")
    f.solve(1e-10, 2000000, use_rd_norm=True)
    one = direct.dense_kkt(np.stack([wp[0], wp[-1]]), np.array([T.sum()]), s)
    tk = np.concatenate([[0.0], np.cumsum(T)])
    got = eval_poly(f.get("coeffs"), T, 0, [0.0])[:, 0]
    want = eval_poly(one, [T.sum()], 0, tk[:-1] / T.sum())[0]
    assert np.abs(got - want).max() < 1e-6


def test_P11_residuals_decrease_and_nonexpansive():
    w = W.config3(N=60)
    o = Oracle(w.waypoints[0], w.durations[0], w.s, rho=10.0)
    hist = []
    for _ in range(12):
        o.sweep(50)
        hist.append(o.residuals()["r_p"])
    assert all(b < a for a, b in zip(hist, hist[1:]))
    ref = direct.banded_optimality(w.waypoints[0], w.durations[0], w.s)
    o.sweep(3000)
    assert relerr(o.get("coeffs"), ref, w.durations[0]) < 1e-9


def test_fp64_oracle_vs_long_double_oracle():
    """Bounds the fp64 oracle's own rounding error on the worst-conditioned config (cfg 1, T up to 9.5 s)."""
    w = W.config1()
    a = Oracle(w.waypoints[0], w.durations[0], w.s, w.rho)
    b = Oracle(w.waypoints[0], w.durations[0], w.s, w.rho, long_double=True)
    for k in (1, 9, 90, 200):
        a.sweep(k); b.sweep(k)
        assert relerr(a.get("coeffs"), b.get("coeffs"), w.durations[0]) < 2e-11
        ua, ub = a.get("u"), b.get("u")
        der = [r for r in range(2 * w.s) if r % w.s != 0]
        assert np.abs(ua[:, der] - ub[:, der]).max() <= 2e-11 * max(1.0, np.abs(ub).max())
        # HARD mode: the position rows of M c - z~ are identically 0 in exact arithmetic, so u's position rows
        # only collect rounding noise (it is annihilated by Pm and never reaches c); bound it, do not compare it.
        assert np.abs(ua[:, [0, w.s]]).max() < 1e-8 and np.abs(ub[:, [0, w.s]]).max() < 1e-11
    w = W.small_constrained(N=23)
    args = (w.waypoints[0], w.durations[0], w.s, w.rho, w.samples, w.box_lo[0], w.box_hi[0], w.vmax, w.amax)
    a, b = Oracle(*args), Oracle(*args, long_double=True)
    a.sweep(300); b.sweep(300)
    assert relerr(a.get("coeffs"), b.get("coeffs"), w.durations[0]) < 1e-10
