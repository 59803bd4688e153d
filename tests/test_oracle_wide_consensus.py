"""Pins for the oracle's paper-literal ("wide") consensus n_c = 2s-1 (reading A1) -- `not gpu`.

The paper's M(t) stacks the derivative orders 0..d-1 with d = 2p-1 (L231), so each boundary carries 2s-1 orders and each
x-update is over-determined (L257).  z_0 and z_N are the given end states, which go to order s-1 only (L141, Eq. 2c,
L261): the orders s..2s-2 at the two trajectory ends do not exist (rowmask).  What fixes this mode without an
implementation to compare against:

  * M's rows are the derivatives of the polynomial up to order 2s-2 (numpy's polynomial calculus);
  * with the waypoints held (HARD, PINNED_Z) the limit is THE direct minimum-jerk/snap solution: C^{2s-2} continuity
    plus waypoints plus end states is a square system (2sN equations per dimension), the optimality conditions of L259-264
    -- had the high orders been fixed at the ends (a plausible misreading), the limit would be a different curve;
  * FREE (Alg. 1 verbatim, L264 "we do not constrain the intermediate conditions"), unconstrained: the limit is the single
    rest-to-rest polynomial from p_0 to p_N;
  * FREE with a box corridor and a speed bound: the limit is the optimum of the sampled QCQP with C^{2s-2} junctions,
    found by scipy's SLSQP (which never sees ADMM, slacks or duals);
  * one x-update (Eq. 20a) recomputed as a stacked least-squares problem with numpy.linalg.lstsq (never forms H or its inverse);
  * the four residual norms recomputed from the iterates (Eq. 21-22, readings A7/A8) over the rows that exist;
  * per-iterate invariants: duals of missing rows stay 0, consensus duals antisymmetric on all 2s-1 averaged orders.
"""
import numpy as np
import pytest
import scipy.optimize
from numpy.polynomial import polynomial as Pl

from oracle import direct
from oracle.top_oracle import Oracle, eval_poly
from paper_2507_10290_b200 import workloads as W


def scaled(c, T):
    n = c.shape[-1]
    return c * (np.asarray(T)[:, None, None] ** np.arange(n)[None, None, :])


def relerr(a, b, T):
    return np.abs(scaled(a - b, T)).max() / np.abs(scaled(b, T)).max()


def deriv_rows(n, orders, t):
    M = np.zeros((len(orders), n))
    for r, k in enumerate(orders):
        for a in range(n):
            e = np.zeros(n); e[a] = 1.0
            M[r, a] = Pl.polyval(t, Pl.polyder(e, k)) if k > 0 else Pl.polyval(t, e)
    return M


def wide_M(s, T):
    """M(T) of PAPER.md:L231 taken literally: orders 0..2s-2 at t = 0, then at t = T."""
    return np.vstack([deriv_rows(2 * s, range(2 * s - 1), 0.0), deriv_rows(2 * s, range(2 * s - 1), T)])


def existing_rows(s, N, i):
    """Rows of segment i that take part in the consensus: everything, except the orders >= s at the two trajectory ends."""
    nc = 2 * s - 1
    keep = np.ones(2 * nc, dtype=bool)
    if i == 0:
        keep[s:nc] = False
    if i == N - 1:
        keep[nc + s:] = False
    return keep


@pytest.mark.parametrize("s", [3, 4])
def test_wide_M_rows_and_rowmask(s):
    rng = np.random.default_rng(s)
    N, nc = 4, 2 * s - 1
    T = rng.uniform(0.6, 2.0, size=N)
    o = Oracle(np.cumsum(rng.normal(size=(N + 1, 3)), axis=0), T, s, 1.0, consensus="wide")
    M, mask = o.get("M"), o.get("rowmask")
    assert M.shape == (N, 2 * nc, 2 * s) and o.get("z").shape == (N + 1, nc, 3) and o.get("u").shape == (N, 2 * nc, 3)
    c = rng.normal(size=2 * s)
    P = np.polynomial.Polynomial(c)
    for i in range(N):
        for k in range(nc):
            assert np.isclose(M[i, k] @ c, P.deriv(k)(0.0) if k else P(0.0), rtol=1e-13)
            assert np.isclose(M[i, nc + k] @ c, P.deriv(k)(T[i]) if k else P(T[i]), rtol=1e-13)
        assert np.array_equal(mask[i] > 0, existing_rows(s, N, i))
    # N = 1: both ends are trajectory ends
    o1 = Oracle(np.array([[0.0, 0, 0], [1.0, 2, 3]]), np.array([1.5]), s, 1.0, consensus="wide")
    assert np.array_equal(o1.get("rowmask")[0] > 0, existing_rows(s, 1, 0))


@pytest.mark.parametrize("mode,tol", [("hard", 1e-8), ("pinned_z", 1e-6)])
def test_wide_config1_converges_to_direct_solution(mode, tol):
    w = W.config1()
    o = Oracle(w.waypoints[0], w.durations[0], w.s, w.rho, mode=mode, consensus="wide")
    o.sweep(w.sweeps)
    ref = direct.dense_kkt(w.waypoints[0], w.durations[0], w.s)
    assert relerr(o.get("coeffs"), ref, w.durations[0]) < tol
    r = o.residuals()
    assert r["r_p"] < 1e-5 and r["r_p_gap"] < 1e-5
    # C^{2s-2} at every junction is now IMPOSED (r_p -> 0), not just emergent
    c = o.get("coeffs")
    for k in range(2 * w.s - 1):
        gap = eval_poly(c, w.durations[0], k, [1.0])[:-1, 0] - eval_poly(c, w.durations[0], k, [0.0])[1:, 0]
        assert np.abs(gap).max() < 1e-5
    # the orders >= s at the trajectory ends are NOT zero in the optimum (snap / jerk is free there): fixing them would
    # have produced another curve
    jerk0 = eval_poly(ref, w.durations[0], w.s, [0.0])[0, 0]
    assert np.abs(jerk0).max() > 1e-3


@pytest.mark.parametrize("s,N,sd", [(3, 2, False), (3, 4, True), (4, 3, False), (4, 5, True)])
def test_wide_small_N_brute_force(s, N, sd):
    rng = np.random.default_rng(300 + 10 * N + s)
    wp = np.cumsum(rng.uniform(-2, 2, size=(N + 1, 3)), axis=0)
    T = rng.uniform(0.8, 1.6, size=N)
    sdv, edv = (rng.normal(size=(s - 1, 3)), rng.normal(size=(s - 1, 3))) if sd else (None, None)
    o = Oracle(wp, T, s, rho=10.0, consensus="wide", start_derivs=sdv, end_derivs=edv)
    o.solve(1e-11, 400000, use_rd_norm=True)
    assert relerr(o.get("coeffs"), direct.dense_kkt(wp, T, s, sdv, edv), T) < 1e-8
    # FREE mode, unconstrained: one rest-to-rest polynomial from p_0 to p_N (rest ends only)
    if not sd and s == 3:      # (s = 4 needs 3e6 sweeps: half a minute; the jerk case pins the same code)
        f = Oracle(wp, T, s, rho=10.0, mode="free", consensus="wide")
        f.solve(1e-10, 3000000, use_rd_norm=True)
        one = direct.dense_kkt(np.stack([wp[0], wp[-1]]), np.array([T.sum()]), s)
        tk = np.concatenate([[0.0], np.cumsum(T)])
        got = eval_poly(f.get("coeffs"), T, 0, [0.0])[:, 0]
        want = eval_poly(one, [T.sum()], 0, tk[:-1] / T.sum())[0]
        assert np.abs(got - want).max() < 1e-6


@pytest.mark.parametrize("mode", ["free", "pinned_z"])
def test_wide_x_update_is_the_least_squares_solution(mode):
    """Eq. 20a for one segment is argmin c'Q~c + rho/2 ||M c - z~ + u||^2 over the rows that exist (Eq. 5):
    a stacked least-squares problem [sqrt2 L; sqrt(rho) M] c ~ [0; sqrt(rho)(z~ - u)] with Q = L'L, solved by lstsq."""
    rng = np.random.default_rng(11)
    s, N, rho = 4, 5, 7.0
    nc = 2 * s - 1
    wp = np.cumsum(rng.uniform(-2, 2, size=(N + 1, 3)), axis=0)
    T = rng.uniform(0.7, 1.5, size=N)
    o = Oracle(wp, T, s, rho, mode=mode, consensus="wide")
    o.sweep(3)
    z, u = o.get("z"), o.get("u")
    o.sweep(1)
    C = o.get("C")
    for i in range(N):
        keep = existing_rows(s, N, i)
        M = wide_M(s, T[i])[keep]
        D = np.diag(T[i] ** np.arange(2 * s))
        Q = D @ (direct.Q_unit(s) * T[i] ** (1 - 2 * s)) @ D
        lam, V = np.linalg.eigh(Q)
        L = np.sqrt(np.maximum(lam, 0))[:, None] * V.T
        g = (np.vstack([z[i], z[i + 1]]) - u[i])[keep]
        A = np.vstack([np.sqrt(2.0) * L, np.sqrt(rho) * M])
        b = np.vstack([np.zeros((2 * s, 3)), np.sqrt(rho) * g])
        want, *_ = np.linalg.lstsq(A, b, rcond=None)
        assert np.abs((C[i] - want) * (T[i] ** np.arange(2 * s))[:, None]).max() < 1e-9 * np.abs(want * (T[i] ** np.arange(2 * s))[:, None]).max()


def recompute_residuals(o, z_prev, mutate=None):
    s, N, T, rho = o.s, o.N, o.T, o.rho
    nc = 2 * s - 1
    C, z = o.get("C"), o.get("z")
    rp2 = rd2 = rdn2 = gap2 = 0.0
    for i in range(N):
        keep = existing_rows(s, N, i)
        if mutate == "count_missing_rows":
            keep = np.ones_like(keep)
        M = wide_M(s, T[i])
        B = M @ C[i]
        zt, ztp = np.vstack([z[i], z[i + 1]]), np.vstack([z_prev[i], z_prev[i + 1]])
        res = (B - zt)[keep]
        rp2 += (res ** 2).sum()
        g = rho * (M[keep].T @ (zt - ztp)[keep])
        rd2 += (g ** 2).sum()
        rdn2 += ((g / (T[i] ** np.arange(2 * s))[:, None]) ** 2).sum()
        if i < N - 1:
            Bn = wide_M(s, T[i + 1]) @ C[i + 1]
            gap2 += ((B[nc:] - Bn[:nc]) ** 2).sum()             # Eq. 21 verbatim, all 2s-1 orders of the junction
    return np.sqrt(rp2), np.sqrt(rd2), np.sqrt(rdn2), np.sqrt(gap2)


@pytest.mark.parametrize("case", ["free", "hard_constrained"])
def test_wide_residual_norms_from_iterates(case):
    if case == "free":
        w = W.config1()
        o = Oracle(w.waypoints[0], w.durations[0], w.s, 3.0, mode="free", consensus="wide")
    else:
        w = W.small_constrained(N=9, s=4, acc=True)
        o = Oracle(w.waypoints[0], w.durations[0], w.s, w.rho, samples=w.samples, box_lo=w.box_lo[0], box_hi=w.box_hi[0],
                   vmax=w.vmax, amax=w.amax, consensus="wide")
    for k in range(5):
        z_prev = o.get("z")
        o.sweep(1)
        r = o.residuals()
        rp, rd, rdn, gap = recompute_residuals(o, z_prev)
        for key, val in (("r_p", rp), ("r_d", rd), ("r_d_norm", rdn), ("r_p_gap", gap)):
            assert abs(r[key] - val) <= 1e-12 * abs(val), (case, k, key, r[key], val)
        if case == "free":      # every interior row is an average, the fixed rows are the ends' orders 0..s-1
            s, nc = o.s, 2 * o.s - 1
            C, z = o.get("C"), o.get("z")
            B0 = (wide_M(s, o.T[0]) @ C[0])[:s] - z[0][:s]
            BN = (wide_M(s, o.T[-1]) @ C[-1])[nc:nc + s] - z[-1][:s]
            assert abs(rp ** 2 - (gap ** 2 / 2 + (B0 ** 2).sum() + (BN ** 2).sum())) <= 1e-11 * rp ** 2
        if k == 0:      # counting the rows that do not exist is a different number
            rp_bad, *_ = recompute_residuals(o, z_prev, "count_missing_rows")
            assert abs(rp_bad - r["r_p"]) > 1e-3 * r["r_p"]


def test_wide_per_iterate_invariants():
    w = W.small_constrained(N=17, s=4, acc=True)
    s, nc = w.s, 2 * w.s - 1
    o = Oracle(w.waypoints[0], w.durations[0], w.s, w.rho, w.samples, w.box_lo[0], w.box_hi[0], w.vmax, w.amax, consensus="wide")
    for k in (1, 1, 3, 40):
        o.sweep(k)
        U, z, C = o.get("u"), o.get("z"), o.get("C")
        assert np.all(U[0, s:nc] == 0) and np.all(U[-1, nc + s:] == 0)          # no such rows: no duals
        assert np.all(z[0, s:] == 0) and np.all(z[-1, s:] == 0)                  # never touched
        anti = U[:-1, nc:, :] + U[1:, :nc, :]
        assert np.abs(anti[:, 1:, :]).max() <= 1e-11 * max(1.0, np.abs(U).max())
        for j in range(1, o.N):                                                 # Eq. 20b on every averaged order
            Bl = (wide_M(s, o.T[j - 1]) @ C[j - 1])[nc:]
            Br = (wide_M(s, o.T[j]) @ C[j])[:nc]
            assert np.allclose(z[j][1:], 0.5 * (Bl + Br)[1:], rtol=1e-12, atol=1e-12 * np.abs(Bl).max())


def test_wide_free_constrained_limit_equals_slsqp_optimum():
    """FREE waypoints + C^{2s-2} junctions + box corridor + speed bound: (N-1) m degrees of freedom are left (the interior
    waypoint positions); the converged CADMM iterate must be the optimum of that sampled QCQP."""
    s, N, m, Ms = 3, 3, 3, 8
    n = 2 * s
    WP = np.array([[0, 0, 0], [2, 1, 0], [4, -1, 0.5], [6, 0, 0.0]])
    TT = np.array([1.5, 1.2, 1.6])
    taus = (np.arange(Ms) + 1) / (Ms + 1)
    lo = np.minimum(WP[:-1], WP[1:]) - 0.25
    hi = np.maximum(WP[:-1], WP[1:]) + 0.25
    # unconstrained FREE limit: one polynomial; its peak sample speed sets an active bound
    one = direct.dense_kkt(np.stack([WP[0], WP[-1]]), np.array([TT.sum()]), s)
    vmax = 0.9 * np.sqrt((eval_poly(one, [TT.sum()], 1, np.linspace(0, 1, 200)) ** 2).sum(-1)).max()

    o = Oracle(WP, TT, s, rho=10.0, samples=Ms, box_lo=lo, box_hi=hi, vmax=vmax, mode="free", consensus="wide")
    o.solve(1e-10, 3000000, use_rd_norm=True)
    got = o.get("coeffs")

    D = [np.diag(TT[i] ** np.arange(n)) for i in range(N)]
    Qp = [D[i] @ (direct.Q_unit(s) * TT[i] ** (1 - 2 * s)) @ D[i] for i in range(N)]

    def cost(x):
        c = x.reshape(N, m, n)
        return sum(c[i, d] @ Qp[i] @ c[i, d] for i in range(N) for d in range(m))

    def grad(x):
        c = x.reshape(N, m, n)
        return np.stack([[2 * Qp[i] @ c[i, d] for d in range(m)] for i in range(N)]).ravel()

    def row(i, d, vec):
        r = np.zeros((N, m, n)); r[i, d] = vec
        return r.ravel()

    Aeq, beq = [], []
    for d in range(m):
        Aeq.append(row(0, d, direct.beta(n, 0, 0.0))); beq.append(WP[0, d])
        Aeq.append(row(N - 1, d, direct.beta(n, 0, TT[-1]))); beq.append(WP[-1, d])
        for k in range(1, s):
            Aeq.append(row(0, d, direct.beta(n, k, 0.0))); beq.append(0.0)
            Aeq.append(row(N - 1, d, direct.beta(n, k, TT[-1]))); beq.append(0.0)
        for i in range(N - 1):
            for k in range(2 * s - 1):
                Aeq.append(row(i, d, direct.beta(n, k, TT[i])) - row(i + 1, d, direct.beta(n, k, 0.0))); beq.append(0.0)
    Aeq, beq = np.array(Aeq), np.array(beq)
    Ab, bb = [], []
    for i in range(N):
        for tau in taus:
            b0 = direct.beta(n, 0, tau * TT[i])
            for d in range(m):
                Ab.append(row(i, d, b0)); bb.append(hi[i, d])
                Ab.append(-row(i, d, b0)); bb.append(-lo[i, d])
    Ab, bb = np.array(Ab), np.array(bb)
    B1 = [[direct.beta(n, 1, tau * TT[i]) for tau in taus] for i in range(N)]

    def vel_con(x):
        c = x.reshape(N, m, n)
        return np.array([vmax ** 2 - sum((B1[i][j] @ c[i, d]) ** 2 for d in range(m)) for i in range(N) for j in range(Ms)])

    def vel_jac(x):
        c = x.reshape(N, m, n)
        J = []
        for i in range(N):
            for j in range(Ms):
                r = np.zeros((N, m, n))
                for d in range(m):
                    r[i, d] = -2 * (B1[i][j] @ c[i, d]) * B1[i][j]
                J.append(r.ravel())
        return np.array(J)

    cons = [{"type": "eq", "fun": lambda x: Aeq @ x - beq, "jac": lambda x: Aeq},
            {"type": "ineq", "fun": lambda x: bb - Ab @ x, "jac": lambda x: -Ab},
            {"type": "ineq", "fun": vel_con, "jac": vel_jac}]
    res = scipy.optimize.minimize(cost, got.ravel() * 0 + direct.dense_kkt(WP, TT, s).ravel(), jac=grad, constraints=cons,
                                  method="SLSQP", options={"ftol": 1e-15, "maxiter": 800})
    assert res.status in (0, 8), res.message
    assert np.abs(Aeq @ res.x - beq).max() < 1e-8 and (bb - Ab @ res.x).min() > -1e-8 and vel_con(res.x).min() > -1e-8
    # the constraints really bind, and the two optima agree
    assert (vel_con(res.x) < 1e-6).sum() >= 1
    assert abs(cost(got.ravel()) - res.fun) < 1e-6 * res.fun
    assert relerr(got, res.x.reshape(N, m, n), TT) < 2e-5
