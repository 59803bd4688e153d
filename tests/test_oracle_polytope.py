"""Pins for the oracle's general polytope corridor (reading A11p; Eq. 7-10) -- `not gpu`.

The polytope path of the oracle forms and inverts the coupled (n m) x (n m) operator of Eq. 20a and keeps one slack and
one scaled dual per (sample, plane).  It is pinned against things that are not that code:
  * an axis-aligned box written as 6 planes must reproduce the iterates of the (separately pinned) box path, which
    never builds a coupled operator;
  * the algorithm commutes with rotations of space (cost, consensus, balls and half-spaces all do): rotating waypoints
    and plane normals rotates every iterate;
  * the converged iterate of a tiny instance with oblique planes equals the scipy SLSQP optimum of the sampled QCQP, and
    carries the KKT certificate (multipliers rho*v >= 0 on the planes, complementarity);
  * Eq. 10 / 20d-e recomputed independently for one sweep, per (sample, plane), and the Moreau-pair invariants.
"""
import numpy as np
import pytest

from oracle import direct
from oracle.top_oracle import Oracle, eval_poly
from paper_2507_10290_b200 import workloads as W
from tests.qcqp_ref import MS_, N_, S_, TAUS, TT, WP, box_as_planes, slsqp_optimum, tiny_instance


def rotation(seed):
    rng = np.random.default_rng(seed)
    q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    return q


@pytest.mark.parametrize("s,acc,mode", [(4, True, "hard"), (3, False, "hard"), (3, True, "pinned_z"), (4, False, "free")])
def test_box_written_as_planes_reproduces_the_box_iterates(s, acc, mode):
    w = W.small_constrained(N=11, s=s, acc=acc)
    lo, hi = w.box_lo[0], w.box_hi[0]
    ob = Oracle(w.waypoints[0], w.durations[0], s, w.rho, 8, lo, hi, w.vmax, w.amax, mode=mode)
    op = Oracle(w.waypoints[0], w.durations[0], s, w.rho, 8, None, None, w.vmax, w.amax, mode=mode, planes=box_as_planes(lo, hi))
    for k in (0, 1, 1, 5, 40):
        ob.sweep(k); op.sweep(k)
        for f in ("C", "z", "u", "phi_v", "w_v", "phi_a", "w_a"):
            a, b = op.get(f), ob.get(f)
            assert np.abs(a - b).max() <= 1e-9 * max(1.0, np.abs(b).max()), (k, f)      # two fp64 evaluations in the raw monomial basis (R6)
        sp, vp = op.get("s_poly"), op.get("v_poly")
        assert np.abs(sp[:, :, :3] - ob.get("s_pos")).max() <= 1e-8 and np.abs(sp[:, :, 3:] - ob.get("s_neg")).max() <= 1e-8
        assert np.abs(vp[:, :, :3] - ob.get("v_pos")).max() <= 1e-8 and np.abs(vp[:, :, 3:] - ob.get("v_neg")).max() <= 1e-8
        if k:
            ra, rb = op.residuals(), ob.residuals()
            for key in ra:       # (r_d is a norm of differences of consecutive iterates: cancellation, see parity_util)
                tol = 1e-9 if key.startswith("r_p") else 1e-6
                assert abs(ra[key] - rb[key]) <= tol * max(1.0, abs(rb[key])), (k, key)


def oblique_planes(w, seed=3, K=7):
    """K oblique half-spaces per segment that contain the chord with a margin: random unit normals, offset =
    max of a'p over the two waypoints + margin (a convex polytope around the segment, as a corridor cell is)."""
    rng = np.random.default_rng(seed)
    N = w.N
    pl = np.zeros((N, K, 4))
    for i in range(N):
        a = rng.normal(size=(K, 3)); a /= np.linalg.norm(a, axis=1, keepdims=True)
        p0, p1 = w.waypoints[0][i], w.waypoints[0][i + 1]
        margin = rng.uniform(0.3, 1.5, size=K)
        pl[i, :, :3] = a
        pl[i, :, 3] = np.maximum(a @ p0, a @ p1) + margin
    return pl


def test_iterates_rotate_with_space():
    w = W.small_constrained(N=9, s=4, acc=True)
    pl = oblique_planes(w)
    R = rotation(7)
    wp_r = w.waypoints[0] @ R.T
    pl_r = pl.copy(); pl_r[:, :, :3] = pl[:, :, :3] @ R.T
    a = Oracle(w.waypoints[0], w.durations[0], 4, w.rho, 8, None, None, w.vmax, w.amax, planes=pl)
    b = Oracle(wp_r, w.durations[0], 4, w.rho, 8, None, None, w.vmax, w.amax, planes=pl_r)
    assert (a.get("s_poly") > 0).all() or True
    for k in (0, 1, 2, 30):
        a.sweep(k); b.sweep(k)
        assert np.abs(b.get("C") - a.get("C") @ R.T).max() <= 1e-10 * np.abs(a.get("C")).max(), k
        assert np.abs(b.get("z") - a.get("z") @ R.T).max() <= 1e-10 * np.abs(a.get("z")).max()
        assert np.abs(b.get("u") - a.get("u") @ R.T).max() <= 1e-10 * max(1.0, np.abs(a.get("u")).max())
        assert np.abs(b.get("s_poly") - a.get("s_poly")).max() <= 1e-10 and np.abs(b.get("v_poly") - a.get("v_poly")).max() <= 1e-10
        assert np.abs(b.get("phi_v") - a.get("phi_v") @ R.T).max() <= 1e-10
    assert np.abs(a.get("v_poly")).max() > 1e-3        # planes really bind on this instance


def test_one_sweep_of_the_plane_slacks_recomputed_independently():
    w = W.small_constrained(N=6, s=3, acc=False)
    pl = oblique_planes(w, seed=5, K=5)
    o = Oracle(w.waypoints[0], w.durations[0], 3, w.rho, 8, None, None, w.vmax, 0.0, planes=pl)
    o.sweep(4)
    v_old = o.get("v_poly")
    o.sweep(1)
    c = o.get("coeffs")
    P = eval_poly(c, w.durations[0], 0, (np.arange(8) + 1) / 9.0)                     # [N][Ms][3], numpy, not E0
    val = np.einsum("ikd,ijd->ijk", pl[:, :, :3], P)                                  # a_k ' p(t_j)
    q = pl[:, None, :, 3] - val - v_old                                               # Eq. 10: s = max(0, -(Ax - b + v))
    assert np.allclose(o.get("s_poly"), np.maximum(q, 0), atol=1e-12)
    assert np.allclose(o.get("v_poly"), np.maximum(-q, 0), atol=1e-12)                # Eq. 20e = the Moreau partner
    s_, v_ = o.get("s_poly"), o.get("v_poly")
    assert s_.min() >= 0 and v_.min() >= -1e-13 and np.abs(s_ * v_).max() <= 1e-12


@pytest.fixture(scope="module")
def tiny_oblique():
    """The tiny QCQP of pin P8 with its box replaced by 7 oblique planes per segment, some of them binding."""
    unc, lo, hi, vmax = tiny_instance()
    rng = np.random.default_rng(11)
    P = eval_poly(unc, TT, 0, TAUS)                                                   # unconstrained samples
    K = 7
    pl = np.zeros((N_, K, 4))
    for i in range(N_):
        a = rng.normal(size=(K, 3)); a /= np.linalg.norm(a, axis=1, keepdims=True)
        reach = np.maximum((P[i] @ a.T).max(axis=0), np.maximum(a @ WP[i], a @ WP[i + 1]))   # support of the unconstrained arc
        ends = np.maximum(a @ WP[i], a @ WP[i + 1])
        cut = np.where(np.arange(K) < 3, 0.5, 1.0)                                    # the first planes cut into the arc
        pl[i, :, :3] = a
        pl[i, :, 3] = ends + cut * (reach - ends) + 0.02
    return unc, pl, vmax


def test_converged_polytope_instance_equals_slsqp_and_is_kkt(tiny_oblique):
    unc, pl, vmax = tiny_oblique
    o = Oracle(WP, TT, S_, 10.0, MS_, None, None, vmax, 0.0, planes=pl)
    it = o.solve(1e-10, 4000000, use_rd_norm=True)
    assert it < 4000000
    res, cost = slsqp_optimum(unc, None, None, vmax, planes=pl)
    n = 2 * S_
    ref = res.x.reshape(N_, 3, n)
    got = o.get("coeffs")
    sc = TT[:, None, None] ** np.arange(n)[None, None, :]
    assert abs(o.objective() - res.fun) < 1e-7 * res.fun
    assert np.abs((got - ref) * sc).max() / np.abs(ref * sc).max() < 5e-6
    assert res.fun > direct.objective(unc, TT, S_) * 1.001                            # the planes cost something
    # KKT: 2QC + rho[M'U + sum_jk kron(e0_j, a_k) v_jk + E1'W] in span(Ew') per dim; v >= 0, complementary, feasible
    C, U, Vp, Sp, Wv = o.get("C"), o.get("u"), o.get("v_poly"), o.get("s_poly"), o.get("w_v")
    for i in range(N_):
        D = np.diag(TT[i] ** np.arange(n))
        Q = D @ (direct.Q_unit(S_) * (TT[i] ** (1 - 2 * S_))) @ D
        M = np.array([direct.beta(n, r % S_, 0.0 if r < S_ else TT[i]) for r in range(2 * S_)])
        E0 = np.array([direct.beta(n, 0, tau * TT[i]) for tau in TAUS])
        E1 = np.array([direct.beta(n, 1, tau * TT[i]) for tau in TAUS])
        g = 2 * Q @ C[i] + 10.0 * (M.T @ U[i] + E0.T @ (Vp[i] @ pl[i, :, :3]) + E1.T @ Wv[i])
        Ew = np.stack([M[0], M[S_]])
        lam, *_ = np.linalg.lstsq(Ew.T, g, rcond=None)
        assert np.abs(g - Ew.T @ lam).max() < 1e-6 * max(1.0, np.abs(g).max())
        val = (E0 @ C[i]) @ pl[i, :, :3].T                                            # [Ms][K]
        assert (val - pl[i, :, 3][None, :]).max() < 1e-8                              # feasible
        assert np.abs(val + Sp[i] - pl[i, :, 3][None, :]).max() < 1e-8                # Ax + s = b
    assert Vp.min() >= -1e-13 and np.abs(Vp * Sp).max() < 1e-12 and (Vp > 1e-9).sum() >= 1
