"""Test infrastructure shared by the oracle's pin P8/P9 (tests/test_oracle_constrained.py) and the GPU test of the
converged constrained iterate (tests/test_gpu_converged.py): the tiny sampled QCQP and its optimum by scipy SLSQP
(an independent solver that never sees ADMM, slacks or duals), and the KKT certificate of a converged iterate."""
import numpy as np
import scipy.optimize

from oracle import direct
from oracle.top_oracle import eval_poly

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



def box_as_planes(lo, hi):
    """The axis-aligned box lo <= p <= hi as 6 half-spaces a'p <= b per segment: [N][6][4]."""
    N = lo.shape[0]
    pl = np.zeros((N, 6, 4))
    for d in range(3):
        pl[:, d, d] = 1.0; pl[:, d, 3] = hi[:, d]
        pl[:, 3 + d, d] = -1.0; pl[:, 3 + d, 3] = -lo[:, d]
    return pl


def slsqp_optimum(unc, lo, hi, vmax, planes=None):
    """Optimum of min sum c'Q c s.t. waypoints, C^(s-1) continuity, rest ends, box (or polytope planes [N][K][4]:
    a'p <= b) and speed bound at the samples."""
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
            if planes is None:
                for d in range(M_):
                    Abox.append(row(i, d, b0)); bbox.append(hi[i, d])
                    Abox.append(-row(i, d, b0)); bbox.append(-lo[i, d])
            else:
                for k in range(planes.shape[1]):
                    Abox.append(sum(planes[i, k, d] * row(i, d, b0) for d in range(M_))); bbox.append(planes[i, k, 3])
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
    return res, cost


def kkt_certificate(C, U, Vp, Vn, Wv, Sp, Sn, Phi, lo, hi, vmax, rho):
    """P9: stationarity 2QC + rho[M'U + E0'(V+ - V-) + E1'W] in span(Ew') (HARD mode), multiplier signs,
    complementarity, outward normals.  C [N][n][m]; U [N][2s][m]; sample fields [N][Ms][m].  Matrices are built here
    from the definition of the polynomial (oracle.direct.beta / Q_unit), not taken from the implementation under test."""
    n, s = 2 * S_, S_
    for i in range(N_):
        D = np.diag(TT[i] ** np.arange(n))
        Q = D @ (direct.Q_unit(S_) * (TT[i] ** (1 - 2 * S_))) @ D
        M = np.array([direct.beta(n, r % s, 0.0 if r < s else TT[i]) for r in range(2 * s)])
        E0 = np.array([direct.beta(n, 0, tau * TT[i]) for tau in TAUS])
        E1 = np.array([direct.beta(n, 1, tau * TT[i]) for tau in TAUS])
        g = 2 * Q @ C[i] + rho * (M.T @ U[i] + E0.T @ (Vp[i] - Vn[i]) + E1.T @ Wv[i])   # [n][m]
        Ew = np.stack([M[0], M[s]])                          # beta_0(0), beta_0(T)
        lam, *_ = np.linalg.lstsq(Ew.T, g, rcond=None)       # HARD mode: residual gradient in span(Ew')
        assert np.abs(g - Ew.T @ lam).max() < 1e-6 * max(1.0, np.abs(g).max())
        P = E0 @ C[i]
        assert np.abs(P + Sp[i] - hi[i][None, :]).max() < 1e-8 and np.abs(-P + Sn[i] + lo[i][None, :]).max() < 1e-8
        assert np.abs(E1 @ C[i] - Phi[i]).max() < 1e-8
    # multipliers: rho*v >= 0, complementary with the slack; rho*w is an outward normal of the ball
    # (the literal update v += Ac + s - b leaves v at a few ulps instead of exactly 0 when the slack is active)
    ulp = 1e-14 * max(1.0, np.abs(hi).max())
    assert Vp.min() >= -ulp and Vn.min() >= -ulp and Sp.min() >= 0 and Sn.min() >= 0
    assert np.abs(Vp * Sp).max() < 1e-12 and np.abs(Vn * Sn).max() < 1e-12
    speed = np.sqrt((Phi ** 2).sum(-1))
    wn = np.sqrt((Wv ** 2).sum(-1))
    assert speed.max() <= vmax * (1 + 1e-14)
    active = wn > 1e-9
    assert active.sum() >= 1 and (Vp + Vn > 1e-9).sum() >= 1        # both constraint kinds really bind
    assert np.all(speed[active] > vmax * (1 - 1e-9))                # w != 0 only on the boundary
    cosang = (Wv * Phi).sum(-1)[active] / (wn[active] * speed[active])
    assert np.all(cosang > 1 - 1e-12)                               # w parallel to phi (outward normal)
