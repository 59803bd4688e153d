"""Pins P8-P10 for the constrained part of the oracle (projections, slacks, duals) -- all `not gpu`.

P8  the converged CADMM iterate equals the optimum of the sampled QCQP found by an independent solver
    (scipy SLSQP, which never sees ADMM, slacks or duals);
P9  the converged iterate carries a KKT certificate (stationarity with multipliers rho*v, rho*w,
    complementarity, outward normals);
P10 every iterate satisfies the exact identities of the projections (Eq. 10, 14 / 20d-20g).
"""
import numpy as np
import pytest
import scipy.optimize

from oracle import direct
from oracle.top_oracle import Oracle, eval_poly
from paper_2507_10290_b200 import workloads as W

S_, N_, M_, MS_ = 3, 3, 3, 8
WP = np.array([[0, 0, 0], [2, 1, 0], [4, -1, 0.5], [6, 0, 0.0]])
TT = np.array([1.5, 1.2, 1.6])
TAUS = (np.arange(MS_) + 1) / (MS_ + 1)


def tiny_instance():
    """N=3 jerk; v_max = 0.97 x unconstrained peak sample speed; box = chord bbox + 0.3 x max excursion."""
    unc = direct.dense_kkt(WP, TT, S_)
    V = eval_poly(unc, TT, 1, TAUS)
    P = eval_poly(unc, TT, 0, TAUS)
    lo0, hi0 = np.minimum(WP[:-1], WP[1:]), np.maximum(WP[:-1], WP[1:])
    exc = np.maximum(P - hi0[:, None, :], lo0[:, None, :] - P).max()
    h = 0.3 * exc
    vmax = 0.97 * np.sqrt((V ** 2).sum(-1)).max()
    return unc, lo0 - h, hi0 + h, vmax


@pytest.fixture(scope="module")
def converged():
    unc, lo, hi, vmax = tiny_instance()
    o = Oracle(WP, TT, S_, 10.0, MS_, lo, hi, vmax, 0.0)
    it = o.solve(1e-10, 3000000, use_rd_norm=True)
    assert it < 3000000
    return o, unc, lo, hi, vmax


def test_P8_constrained_limit_equals_slsqp_optimum(converged):
    o, unc, lo, hi, vmax = converged
    n = 2 * S_
    nv = N_ * M_ * n                                     # x = coeffs [N][m][n] flattened, physical time
    Qs = [direct.Q_unit(S_) * (TT[i] ** (1 - 2 * S_)) for i in range(N_)]
    D = [np.diag(TT[i] ** np.arange(n)) for i in range(N_)]
    Qp = [D[i] @ Qs[i] @ D[i] for i in range(N_)]        # Q(T_i) in physical time

    def cost(x):
        c = x.reshape(N_, M_, n)
        return sum(c[i, d] @ Qp[i] @ c[i, d] for i in range(N_) for d in range(M_))

    def grad(x):
        c = x.reshape(N_, M_, n)
        g = np.zeros_like(c)
        for i in range(N_):
            for d in range(M_):
                g[i, d] = 2 * Qp[i] @ c[i, d]
        return g.ravel()

    def row(i, d, vec):
        r = np.zeros((N_, M_, n)); r[i, d] = vec
        return r.ravel()

    Aeq, beq = [], []
    for d in range(M_):
        for i in range(N_):
            Aeq.append(row(i, d, direct.beta(n, 0, 0.0))); beq.append(WP[i, d])
            Aeq.append(row(i, d, direct.beta(n, 0, TT[i]))); beq.append(WP[i + 1, d])
        for i in range(N_ - 1):
            for k in range(1, S_):
                Aeq.append(row(i, d, direct.beta(n, k, TT[i])) - row(i + 1, d, direct.beta(n, k, 0.0))); beq.append(0.0)
        for k in range(1, S_):
            Aeq.append(row(0, d, direct.beta(n, k, 0.0))); beq.append(0.0)
            Aeq.append(row(N_ - 1, d, direct.beta(n, k, TT[-1]))); beq.append(0.0)
    Aeq, beq = np.array(Aeq), np.array(beq)
    Abox, bbox = [], []                                  # Abox x <= bbox
    for i in range(N_):
        for tau in TAUS:
            b0 = direct.beta(n, 0, tau * TT[i])
            for d in range(M_):
                Abox.append(row(i, d, b0)); bbox.append(hi[i, d])
                Abox.append(-row(i, d, b0)); bbox.append(-lo[i, d])
    Abox, bbox = np.array(Abox), np.array(bbox)
    B1 = [[direct.beta(n, 1, tau * TT[i]) for tau in TAUS] for i in range(N_)]

    def vel_con(x):
        c = x.reshape(N_, M_, n)
        return np.array([vmax ** 2 - sum((B1[i][j] @ c[i, d]) ** 2 for d in range(M_))
                         for i in range(N_) for j in range(MS_)])

    def vel_jac(x):
        c = x.reshape(N_, M_, n)
        J = []
        for i in range(N_):
            for j in range(MS_):
                r = np.zeros((N_, M_, n))
                for d in range(M_):
                    r[i, d] = -2 * (B1[i][j] @ c[i, d]) * B1[i][j]
                J.append(r.ravel())
        return np.array(J)

    cons = [{"type": "eq", "fun": lambda x: Aeq @ x - beq, "jac": lambda x: Aeq},
            {"type": "ineq", "fun": lambda x: bbox - Abox @ x, "jac": lambda x: -Abox},
            {"type": "ineq", "fun": vel_con, "jac": vel_jac}]
    res = scipy.optimize.minimize(cost, unc.ravel(), jac=grad, constraints=cons, method="SLSQP",
                                  options={"ftol": 1e-15, "maxiter": 500})
    # status 8 ("positive directional derivative") is SLSQP's way of saying it cannot improve below ftol;
    # accept it only if the point is feasible to 1e-9
    assert res.status in (0, 8), res.message
    assert np.abs(Aeq @ res.x - beq).max() < 1e-9 and (bbox - Abox @ res.x).min() > -1e-9 and vel_con(res.x).min() > -1e-9
    ref = res.x.reshape(N_, M_, n)
    got = o.get("coeffs")
    assert abs(o.objective() - res.fun) < 1e-7 * res.fun
    assert cost(got.ravel()) == pytest.approx(o.objective(), rel=1e-12)
    sc = TT[:, None, None] ** np.arange(n)[None, None, :]
    assert np.abs((got - ref) * sc).max() / np.abs(ref * sc).max() < 2e-6
    # P11: the constrained optimum costs more than the unconstrained one
    assert res.fun > direct.objective(unc, TT, S_) * 1.01


def test_P9_kkt_certificate_at_convergence(converged):
    o, unc, lo, hi, vmax = converged
    rho, n, s = 10.0, 2 * S_, S_
    C, Q, M = o.get("C"), o.get("Q"), o.get("M")
    E0, E1 = o.get("E0"), o.get("E1")
    U, Vp, Vn, Wv = o.get("u"), o.get("v_pos"), o.get("v_neg"), o.get("w_v")
    Sp, Sn, Phi = o.get("s_pos"), o.get("s_neg"), o.get("phi_v")
    for i in range(N_):
        g = 2 * Q[i] @ C[i] + rho * (M[i].T @ U[i] + E0[i].T @ (Vp[i] - Vn[i]) + E1[i].T @ Wv[i])   # [n][m]
        Ew = np.stack([M[i][0], M[i][s]])                    # beta_0(0), beta_0(T)
        lam, *_ = np.linalg.lstsq(Ew.T, g, rcond=None)       # HARD mode: residual gradient in span(Ew')
        assert np.abs(g - Ew.T @ lam).max() < 1e-6 * max(1.0, np.abs(g).max())
    # multipliers: rho*v >= 0, complementary with the slack; rho*w is an outward normal of the ball
    # (the literal update v += Ac + s - b leaves v at a few ulps instead of exactly 0 when the slack is active)
    ulp = 1e-14 * max(1.0, np.abs(hi).max())
    assert Vp.min() >= -ulp and Vn.min() >= -ulp and Sp.min() >= 0 and Sn.min() >= 0
    assert np.abs(Vp * Sp).max() < 1e-12 and np.abs(Vn * Sn).max() < 1e-12
    P = np.einsum("ijn,ind->ijd", E0, C)
    assert np.abs(P + Sp - hi[:, None, :]).max() < 1e-8 and np.abs(-P + Sn + lo[:, None, :]).max() < 1e-8
    Vel = np.einsum("ijn,ind->ijd", E1, C)
    assert np.abs(Vel - Phi).max() < 1e-8
    speed = np.sqrt((Phi ** 2).sum(-1))
    wn = np.sqrt((Wv ** 2).sum(-1))
    assert speed.max() <= vmax * (1 + 1e-14)
    active = wn > 1e-9
    assert active.sum() >= 1 and (Vp + Vn > 1e-9).sum() >= 1        # both constraint kinds really bind
    assert np.all(speed[active] > vmax * (1 - 1e-9))                # w != 0 only on the boundary
    cosang = (Wv * Phi).sum(-1)[active] / (wn[active] * speed[active])
    assert np.all(cosang > 1 - 1e-12)                               # w parallel to phi (outward normal)


@pytest.mark.parametrize("s,acc", [(4, True), (3, False)])
def test_P10_per_iterate_invariants(s, acc):
    w = W.small_constrained(N=29, s=s, acc=acc)
    o = Oracle(w.waypoints[0], w.durations[0], w.s, w.rho, w.samples, w.box_lo[0], w.box_hi[0], w.vmax, w.amax)
    lo, hi = w.box_lo[0][:, None, :], w.box_hi[0][:, None, :]
    for k in (0, 1, 1, 3, 25, 170):
        prev = {f: o.get(f) for f in ("v_pos", "v_neg", "w_v", "w_a")}
        o.sweep(k)
        C = o.get("C")
        P = np.einsum("ijn,ind->ijd", o.get("E0"), C)
        Sp, Sn, Vp, Vn = o.get("s_pos"), o.get("s_neg"), o.get("v_pos"), o.get("v_neg")
        ulp = 1e-14 * max(1.0, np.abs(hi).max())
        assert Sp.min() >= 0 and Sn.min() >= 0 and Vp.min() >= -ulp and Vn.min() >= -ulp
        assert np.abs(Vp * Sp).max() <= ulp * max(1.0, Sp.max()) and np.abs(Vn * Sn).max() <= ulp * max(1.0, Sn.max())  # Moreau pair
        if k == 1:   # s = max(0, -(Ac - b + v_old)), v = v_old + Ac + s - b  (Eq. 10 / 20d, 20e), independently
            q = hi - P - prev["v_pos"]
            assert np.allclose(Sp, np.maximum(q, 0), atol=1e-13) and np.allclose(Vp, np.maximum(-q, 0), atol=1e-13)
            q = P - lo - prev["v_neg"]
            assert np.allclose(Sn, np.maximum(q, 0), atol=1e-13) and np.allclose(Vn, np.maximum(-q, 0), atol=1e-13)
        for kind, bound, fld in ((1, w.vmax, "v"), (2, w.amax, "a")):
            if bound <= 0:
                continue
            Phi, Wd = o.get("phi_" + fld), o.get("w_" + fld)
            nrm = np.sqrt((Phi ** 2).sum(-1))
            assert nrm.max() <= bound * (1 + 4e-16)
            Y = Phi + Wd
            cross = np.cross(Phi, Wd)
            assert np.abs(cross).max() <= 1e-12 * max(1.0, np.abs(Y).max() ** 2)     # W parallel to Phi
            inside = np.sqrt((Y ** 2).sum(-1)) <= bound
            assert np.abs(Wd[inside]).max(initial=0.0) == 0
            if k == 1:   # Eq. 14: phi = projection of (B c + w_old) onto the ball, independently
                Bc = np.einsum("ijn,ind->ijd", o.get("E%d" % kind), C) + prev["w_" + fld]
                nb = np.sqrt((Bc ** 2).sum(-1, keepdims=True))
                want = np.where(nb > bound, Bc * bound / np.maximum(nb, 1e-300), Bc)
                assert np.allclose(Phi, want, atol=1e-13)
        # consensus duals are antisymmetric on averaged rows; position gap is 0 in HARD mode
        U = o.get("u")
        if k > 0:
            anti = U[:-1, s:, :] + U[1:, :s, :]
            assert np.abs(anti[:, 1:, :]).max() <= 1e-11 * max(1.0, np.abs(U).max())
            B_end = np.einsum("irn,ind->ird", o.get("M")[:, s:s + 1], C)[:-1, 0]
            assert np.abs(B_end - w.waypoints[0][1:-1]).max() < 1e-9 * max(1.0, np.abs(w.waypoints).max())
        # z_0, z_N stay at the given end states (rest)
        z = o.get("z")
        assert np.all(z[0, 1:] == 0) and np.all(z[-1, 1:] == 0)
        assert np.array_equal(z[0, 0], w.waypoints[0][0]) and np.array_equal(z[-1, 0], w.waypoints[0][-1])


def test_nonrest_end_states_reach_direct_solution():
    rng = np.random.default_rng(5)
    N, s = 5, 4
    wp = np.cumsum(rng.uniform(-2, 2, size=(N + 1, 3)), axis=0)
    T = rng.uniform(0.8, 1.6, size=N)
    sd, ed = rng.normal(size=(s - 1, 3)), rng.normal(size=(s - 1, 3))
    o = Oracle(wp, T, s, rho=10.0, start_derivs=sd, end_derivs=ed)
    o.solve(1e-10, 2000000, use_rd_norm=True)
    ref = direct.banded_optimality(wp, T, s, sd, ed)
    sc = T[:, None, None] ** np.arange(2 * s)[None, None, :]
    assert np.abs((o.get("coeffs") - ref) * sc).max() / np.abs(ref * sc).max() < 1e-7
