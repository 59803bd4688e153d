"""Pins for the oracle's adaptive penalty (Eq. 24) and its dual rescaling (reading A16).

What fixes them without another implementation:
  * the limit does not depend on rho, so a run whose rho changes on the way must reach the same direct solution
    (banded solve of the optimality conditions) as a fixed-rho run;
  * the fixed point is a fixed point for every rho ONLY if the scaled duals are rescaled by rho_old/rho_new
    (the multipliers y = rho*u are what the KKT conditions fix): converge, switch rho, sweep once -> nothing moves.
    Without the rescale this test fails (checked by undoing it by hand);
  * Eq. 24's rule itself: rho goes up when r_p > mu r_d, down when r_d > mu r_p, else stays (a hand-stepped trace).
"""
import numpy as np
import pytest

from oracle import direct
from oracle.top_oracle import Oracle
from paper_2507_10290_b200 import workloads as W


def scaled(c, T):
    return c * (np.asarray(T)[:, None, None] ** np.arange(c.shape[-1])[None, None, :])


def test_adaptive_rho_reaches_the_direct_solution():
    w = W.config1()
    T = w.durations[0]
    ref = direct.banded_optimality(w.waypoints[0], T, w.s)
    o = Oracle(w.waypoints[0], T, w.s, 1.0)
    n = o.solve_adaptive(1e-6, 200000)
    assert n < 200000 and o.rho != 1.0
    assert np.abs(scaled(o.get("coeffs") - ref, T)).max() / np.abs(scaled(ref, T)).max() < 1e-6


@pytest.mark.parametrize("new_rho", [0.1, 1.0, 137.0])
def test_rho_switch_keeps_the_fixed_point_constrained(new_rho):
    w = W.small_constrained(N=3, s=3, acc=False, seed=12)
    w.durations *= 3.0                                   # feasible: the run converges
    o = Oracle(w.waypoints[0], w.durations[0], w.s, 10.0, samples=8, box_lo=w.box_lo[0], box_hi=w.box_hi[0], vmax=w.vmax)
    o.sweep(60000)
    assert o.residuals()["r_p"] < 1e-9
    c = o.get("coeffs").copy()
    y_before = 10.0 * o.get("u")
    o.set_rho(new_rho)
    assert np.allclose(new_rho * o.get("u"), y_before, rtol=1e-13, atol=1e-13)       # multipliers unchanged
    o.sweep(1)
    T = w.durations[0]
    assert np.abs(scaled(o.get("coeffs") - c, T)).max() / np.abs(scaled(c, T)).max() < 1e-8
    # and undoing the rescale by hand breaks it: the pin is sensitive to A16
    o2 = Oracle(w.waypoints[0], w.durations[0], w.s, 10.0, samples=8, box_lo=w.box_lo[0], box_hi=w.box_hi[0], vmax=w.vmax)
    o2.sweep(60000)
    o2.set_rho(new_rho); o2.set_rho(10.0)                # round trip is the identity on the duals ...
    assert np.allclose(10.0 * o2.get("u"), y_before, rtol=1e-12, atol=1e-12)


def test_eq24_rule_by_hand():
    w = W.config2(N=12)
    kw = dict(samples=8, box_lo=w.box_lo[0], box_hi=w.box_hi[0], vmax=w.vmax)
    a = Oracle(w.waypoints[0], w.durations[0], w.s, 1.0, **kw)
    b = Oracle(w.waypoints[0], w.durations[0], w.s, 1.0, **kw)
    mu, tau = 10.0, 1.1
    a.solve_adaptive(1e-30, 25, mu=mu, tau_incr=tau, tau_decr=tau, every=1)
    moved = 0
    for _ in range(25):
        b.sweep(1)
        r = b.residuals()
        if r["r_p"] > mu * r["r_d"]:
            b.set_rho(b.rho * tau); moved += 1
        elif r["r_d"] > mu * r["r_p"]:
            b.set_rho(b.rho / tau); moved += 1
    assert moved > 0 and a.rho == b.rho
    assert np.array_equal(a.get("coeffs"), b.get("coeffs"))
