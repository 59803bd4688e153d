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

from tests.qcqp_ref import MS_, M_, N_, S_, TAUS, TT, WP, kkt_certificate, slsqp_optimum, tiny_instance


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
    res, cost = slsqp_optimum(unc, lo, hi, vmax)
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
    # the oracle's own matrices must be the ones the certificate builds from the definition
    n = 2 * S_
    for i in range(N_):
        assert np.allclose(o.get("M")[i], [direct.beta(n, r % S_, 0.0 if r < S_ else TT[i]) for r in range(2 * S_)], rtol=1e-13)
        assert np.allclose(o.get("E1")[i], [direct.beta(n, 1, tau * TT[i]) for tau in TAUS], rtol=1e-13)
    kkt_certificate(o.get("C"), o.get("u"), o.get("v_pos"), o.get("v_neg"), o.get("w_v"), o.get("s_pos"), o.get("s_neg"),
                    o.get("phi_v"), lo, hi, vmax, 10.0)


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
