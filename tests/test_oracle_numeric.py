"""Pins for the oracle's NumericSolve branch (reading A20; Eq. 15-17, Alg. 1 lines 6-7) -- `not gpu`.

The branch replaces the closed-form x-update by an L-BFGS minimisation of the augmented Lagrangian
    F(c) = c'Q~c + rho/2 ||M~c - z~ + u||^2 + rho/2 ||Ao c + s - b + v||^2 + rho/2 sum_j (g_j(c) + w_j)^2,
    g_j(c) = max{0, ||A_j c||^2 - bound^2}^2                                                  (Eq. 15, Eq. 17)
and updates the scaled multipliers w_j <- w_j + g_j(c^{k+1}).  What fixes it without an implementation to compare against:

  * F recomputed from that definition in numpy (polynomial calculus, no oracle matrices), its gradient by central differences;
  * the x-update IS the minimiser of F: scipy's BFGS on the numpy F (PINNED_Z: unconstrained), scipy's SLSQP with the two
    waypoint equalities per dimension (HARD);
  * with no ball ever violated the iterates are those of the closed-form branch without balls (the penalty vanishes);
  * the multiplier recursion recomputed from the coefficients;
  * the limit: the sampled QCQP optimum by SLSQP (approached slowly: the multipliers of Eq. 15 have no finite limit).
"""
import numpy as np
import pytest
import scipy.optimize
from numpy.polynomial import polynomial as Pl

from oracle import direct
from oracle.top_oracle import Oracle, eval_poly
from tests import qcqp_ref as Q

MS = 8
TAUS = (np.arange(MS) + 1) / (MS + 1)


def deriv_row(n, k, t):
    row = np.zeros(n)
    for a in range(n):
        e = np.zeros(n); e[a] = 1.0
        row[a] = Pl.polyval(t, Pl.polyder(e, k)) if k else Pl.polyval(t, e)
    return row


def F_numpy(o, i, c, z, u, sp, sn, vp, vn, yv, ya, lo, hi, vmax, amax):
    """F of segment i at c [n][m], written from Eq. 5 + Eq. 8 + Eq. 15/17 with numpy only."""
    s, n, T, rho = o.s, 2 * o.s, o.T[i], o.rho
    D = np.diag(T ** np.arange(n))
    Qm = D @ (direct.Q_unit(s) * T ** (1 - 2 * s)) @ D
    F = np.einsum("ad,ab,bd->", c, Qm, c)
    M = np.array([deriv_row(n, r % s, 0.0 if r < s else T) for r in range(2 * s)])
    e = M @ c - np.vstack([z[i], z[i + 1]]) + u[i]
    F += rho / 2 * (e ** 2).sum()
    for j, tau in enumerate(TAUS):
        P = deriv_row(n, 0, tau * T) @ c
        if lo is not None:
            F += rho / 2 * (((P + sp[i, j] - hi[i] + vp[i, j]) ** 2).sum() + ((-P + sn[i, j] + lo[i] + vn[i, j]) ** 2).sum())
        for k, bound, y in ((1, vmax, yv), (2, amax, ya)):
            if bound > 0:
                val = deriv_row(n, k, tau * T) @ c
                g = max(0.0, (val ** 2).sum() - bound ** 2) ** 2
                F += rho / 2 * (g + y[i, j]) ** 2
    return F


def state(o):
    return dict(z=o.get("z"), u=o.get("u"), sp=o.get("s_pos"), sn=o.get("s_neg"), vp=o.get("v_pos"), vn=o.get("v_neg"),
                yv=o.get("y_v"), ya=o.get("y_a"))


def make(mode="hard", vscale=1.0, amax=0.0, **kw):
    unc, lo, hi, vmax = Q.tiny_instance()
    o = Oracle(Q.WP, Q.TT, 3, 10.0, samples=MS, box_lo=lo, box_hi=hi, vmax=vmax * vscale, amax=amax, numeric=True, mode=mode, **kw)
    return o, lo, hi, vmax * vscale


@pytest.mark.parametrize("mode", ["hard", "pinned_z"])
def test_F_and_gradient_from_the_definition(mode):
    o, lo, hi, vmax = make(mode, vscale=0.6, amax=2.0)
    o.sweep(5)
    st = state(o)
    rng = np.random.default_rng(2)
    assert st["yv"].max() > 0            # the multipliers are in play
    for i in range(o.N):
        c = o.get("C")[i] * (1 + 0.05 * rng.normal(size=(6, 3)))
        F, g = o.numeric_eval(i, c)
        want = F_numpy(o, i, c, lo=lo, hi=hi, vmax=vmax, amax=2.0, **st)
        assert abs(F - want) <= 1e-12 * abs(want)
        gfd = np.zeros_like(c)
        for a in range(6):
            for d in range(3):
                h = 1e-6 * max(1.0, abs(c[a, d]))
                cp, cm = c.copy(), c.copy()
                cp[a, d] += h; cm[a, d] -= h
                gfd[a, d] = (F_numpy(o, i, cp, lo=lo, hi=hi, vmax=vmax, amax=2.0, **st) - F_numpy(o, i, cm, lo=lo, hi=hi, vmax=vmax, amax=2.0, **st)) / (2 * h)
        assert np.abs(g - gfd).max() <= 1e-6 * np.abs(g).max()


@pytest.mark.parametrize("mode", ["pinned_z", "hard"])
def test_x_update_minimises_F(mode):
    o, lo, hi, vmax = make(mode, vscale=0.9, inner_tol=1e-12, max_inner=300)
    n = 6
    for sweep in range(12):
        st, C0 = state(o), o.get("C")
        o.sweep(1)
        C1 = o.get("C")
        if sweep not in (0, 5, 11):
            continue
        for i in range(o.N):
            f = lambda x: F_numpy(o, i, x.reshape(n, 3), lo=lo, hi=hi, vmax=vmax, amax=0.0, **st)
            sc = (o.T[i] ** np.arange(n))[:, None]
            if mode == "pinned_z":
                r = scipy.optimize.minimize(f, C0[i].ravel(), method="BFGS", options={"gtol": 1e-8, "maxiter": 5000})
            else:
                rows = [deriv_row(n, 0, 0.0), deriv_row(n, 0, o.T[i])]
                cons = [{"type": "eq", "fun": (lambda x, rw=rw, d=d, tgt=tgt: rw @ x.reshape(n, 3)[:, d] - tgt)}
                        for d in range(3) for rw, tgt in ((rows[0], Q.WP[i, d]), (rows[1], Q.WP[i + 1, d]))]
                r = scipy.optimize.minimize(f, C0[i].ravel(), method="SLSQP", constraints=cons, options={"ftol": 1e-15, "maxiter": 2000})
            want = r.x.reshape(n, 3)
            assert f(C1[i].ravel()) <= r.fun * (1 + 1e-9) + 1e-12, (sweep, i)
            assert np.abs((C1[i] - want) * sc).max() <= 2e-5 * np.abs(want * sc).max(), (sweep, i)


@pytest.mark.parametrize("mode", ["hard", "pinned_z", "free"])
def test_without_violation_it_is_the_closed_form_branch(mode):
    unc, lo, hi, vmax = Q.tiny_instance()
    a = Oracle(Q.WP, Q.TT, 3, 10.0, samples=MS, box_lo=lo, box_hi=hi, mode=mode)
    b = Oracle(Q.WP, Q.TT, 3, 10.0, samples=MS, box_lo=lo, box_hi=hi, vmax=1e3, amax=1e3, numeric=True, mode=mode)
    for k in (1, 2, 10, 100):
        a.sweep(k - a.iter); b.sweep(k - b.iter)
        for f in ("C", "z", "u", "s_pos", "v_neg"):
            assert np.abs(a.get(f) - b.get(f)).max() <= 1e-11 * max(1.0, np.abs(a.get(f)).max()), (k, f)
    assert b.get("y_v").max() == 0 and b.inner_iters <= 2 * 100 * 3


def test_multiplier_recursion_and_monotone_growth():
    o, lo, hi, vmax = make("hard", vscale=0.9, amax=2.5)
    for k in range(30):
        y0v, y0a = o.get("y_v"), o.get("y_a")
        o.sweep(1)
        c = o.get("coeffs")
        for kind, bound, y0, name in ((1, vmax, y0v, "y_v"), (2, 2.5, y0a, "y_a")):
            val = eval_poly(c, o.T, kind, TAUS)
            g = np.maximum(0.0, (val ** 2).sum(-1) - bound ** 2) ** 2
            got = o.get(name)
            assert np.abs(got - (y0 + g)).max() <= 1e-12 * max(1.0, np.abs(got).max())
            assert np.all(got >= y0)          # g_j >= 0: the multipliers of Eq. 15 never decrease


def test_limit_approaches_the_qcqp_optimum():
    unc, lo, hi, vmax = Q.tiny_instance()
    res, cost = Q.slsqp_optimum(unc, lo, hi, vmax)
    xs = res.x.reshape(3, 3, 6)
    sc = Q.TT[:, None, None] ** np.arange(6)[None, None, :]
    o = Oracle(Q.WP, Q.TT, 3, 10.0, samples=MS, box_lo=lo, box_hi=hi, vmax=vmax, numeric=True)
    dist, viol = [], []
    for k in (1000, 4000, 16000):
        o.sweep(k - o.iter)
        c = o.get("coeffs")
        dist.append(np.abs((c - xs) * sc).max() / np.abs(xs * sc).max())
        viol.append(np.sqrt((eval_poly(c, Q.TT, 1, TAUS) ** 2).sum(-1)).max() / vmax - 1)
    assert dist[0] > dist[1] > dist[2] and dist[2] < 0.02
    assert viol[0] > viol[1] > viol[2] > 0 and viol[2] < 5e-3       # feasibility from outside, slowly (no finite multiplier)
    assert o.residuals()["r_p"] < 1e-3
