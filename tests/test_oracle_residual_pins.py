"""Pins for the oracle's residual norms r_p, r_d, r_d_norm, r_p_gap (oracle/top_oracle.c, sweep_once) -- `not gpu`.

These four numbers decide every top_solve stop, every Eq. 24 step and every time-to-eps figure, and the CUDA path is
matched to them; "they go to zero" does not pin them (a dropped rho, M instead of M', a wrong power of T or a miscounted
row still goes to zero).  Here each norm is recomputed for single sweeps from the oracle's own ITERATES only
(coefficients and consensus variables before / after the sweep), with the evaluation matrices rebuilt from the
definition of the polynomial (numpy.polynomial derivatives, not oracle.get("M")), written from the paper:

  Eq. 21   r_p_gap = || stack_j ( sigma~_j(T_j) - sigma~_{j+1}(0) ) ||   over the N-1 junctions
  reading A7                   r_p     = || stack_i ( M(T_i) c_i - z~_i^{k+1} ) ||            over all 2s rows of all segments
  Eq. 22, A8  r_d  = rho || stack_i M(T_i)' ( z~_i^{k+1} - z~_i^k ) ||   (monomial, physical time)
  normalised variant           component a of segment i divided by T_i^a
and the identity  r_p^2 = r_p_gap^2 / 2 + (fixed-row terms)  that ties A7 to Eq. 21 on averaged rows.
Plausible mistakes are shown to FAIL the pin (sensitivity block at the end of the test).
"""
import numpy as np
import pytest
from numpy.polynomial import polynomial as Pl

from oracle.top_oracle import Oracle
from paper_2507_10290_b200 import workloads as W


def deriv_rows(n, orders, t):
    """Row k: coefficients-to-value map of the k-th derivative at time t, from numpy's polynomial calculus."""
    M = np.zeros((len(orders), n))
    for r, k in enumerate(orders):
        for a in range(n):
            e = np.zeros(n); e[a] = 1.0
            M[r, a] = Pl.polyval(t, Pl.polyder(e, k)) if k > 0 else Pl.polyval(t, e)
    return M


def consensus_matrix(s, T):
    """M(T) of PAPER.md:L231: derivative orders 0..s-1 at t = 0, then at t = T (reading A1: n_c = s)."""
    n = 2 * s
    return np.vstack([deriv_rows(n, range(s), 0.0), deriv_rows(n, range(s), T)])


def stacked_z(z, i):
    """z~_i = (z_{i-1}; z_i) as a [2s, m] block (Eq. 4)."""
    return np.vstack([z[i], z[i + 1]])


def recompute(o, z_prev, mutate=None):
    """The four norms of the sweep that took z_prev to o's current z, from iterates only."""
    s, N, T, rho = o.s, o.N, o.T, o.rho
    C, z = o.get("C"), o.get("z")                     # [N][n][m], [N+1][s][m]
    rp2 = rd2 = rdn2 = gap2 = 0.0
    fixed2 = 0.0
    for i in range(N):
        M = consensus_matrix(s, T[i])
        B = M @ C[i]                                  # boundary derivatives of segment i, [2s][m]
        res = B - stacked_z(z, i)
        rp2 += (res ** 2).sum()
        dz = stacked_z(z, i) - stacked_z(z_prev, i)
        Mt = M.T if mutate != "no_transpose" else M
        g = (rho if mutate != "no_rho" else 1.0) * (Mt @ dz)          # [n][m]
        rd2 += (g ** 2).sum()
        pw = T[i] ** np.arange(2 * s) if mutate != "wrong_power" else T[i] ** (np.arange(2 * s) + 1)
        rdn2 += ((g / pw[:, None]) ** 2).sum()
        if i < N - 1:
            Bn = consensus_matrix(s, T[i + 1]) @ C[i + 1]
            gap = B[s:] - Bn[:s]                       # Eq. 21 verbatim: end of segment i against start of i+1
            gap2 += (gap ** 2).sum()
        # rows whose z is not an average of two segments: the two trajectory ends (all orders)
        if i == 0:
            fixed2 += (res[:s] ** 2).sum()
        if i == N - 1:
            fixed2 += (res[s:] ** 2).sum()
    return np.sqrt(rp2), np.sqrt(rd2), np.sqrt(rdn2), np.sqrt(gap2), fixed2


def cases():
    w1 = W.config1()
    yield "cfg1 unconstrained jerk", Oracle(w1.waypoints[0], w1.durations[0], w1.s, 3.0, mode="free"), 6
    yield "cfg1 hard", Oracle(w1.waypoints[0], w1.durations[0], w1.s, 2.5), 5      # rho != 1: a dropped rho must show
    w2 = W.small_constrained(N=9, s=4, acc=True)
    yield "small constrained snap", Oracle(w2.waypoints[0], w2.durations[0], w2.s, w2.rho, samples=w2.samples,
                                           box_lo=w2.box_lo[0], box_hi=w2.box_hi[0], vmax=w2.vmax, amax=w2.amax), 5
    rng = np.random.default_rng(5)
    sd, ed = rng.normal(size=(2, 3)), rng.normal(size=(2, 3))
    w3 = W.small_constrained(N=6, s=3, acc=False)
    yield "non-rest ends, pinned_z", Oracle(w3.waypoints[0], w3.durations[0], 3, 7.0, samples=8, box_lo=w3.box_lo[0],
                                            box_hi=w3.box_hi[0], vmax=w3.vmax, start_derivs=sd, end_derivs=ed,
                                            mode="pinned_z"), 4


@pytest.mark.parametrize("name,o,sweeps", list(cases()), ids=lambda v: v if isinstance(v, str) else "")
def test_residual_norms_from_iterates(name, o, sweeps):
    for k in range(sweeps):
        z_prev = o.get("z")
        o.sweep(1)
        r = o.residuals()
        rp, rd, rdn, gap, fixed2 = recompute(o, z_prev)
        for key, val in (("r_p", rp), ("r_d", rd), ("r_d_norm", rdn), ("r_p_gap", gap)):
            assert abs(r[key] - val) <= 1e-12 * max(abs(val), 1e-300), (name, k, key, r[key], val)
        # reading A7 against Eq. 21: on a junction both segments are at distance gap/2 from their average
        if "unconstrained jerk" in name:            # FREE mode: every interior row is an average, only the ends are fixed
            assert abs(rp ** 2 - (gap ** 2 / 2.0 + fixed2)) <= 1e-11 * rp ** 2, (name, k)
        # ---- sensitivity: each plausible mistake moves the recomputed value well outside the pin's tolerance
        if k == 0:
            _, rd_norho, _, _, _ = recompute(o, z_prev, "no_rho")
            _, rd_notr, rdn_notr, _, _ = recompute(o, z_prev, "no_transpose")
            _, _, rdn_pw, _, _ = recompute(o, z_prev, "wrong_power")
            assert abs(rd_norho - r["r_d"]) > 1e-3 * r["r_d"], name
            assert abs(rd_notr - r["r_d"]) > 1e-3 * r["r_d"], name
            assert abs(rdn_pw - r["r_d_norm"]) > 1e-3 * r["r_d_norm"], name
            # counting only the junction gaps (Eq. 21 verbatim) instead of all rows is a different number
            assert abs(r["r_p_gap"] - r["r_p"]) > 1e-3 * r["r_p"], name


def test_gap_identity_with_pinned_and_hard_rows():
    """HARD / PINNED_Z: the position rows are not averages either (they stay at the waypoints), so
    r_p^2 = (gap^2 over the averaged rows)/2 + all non-averaged rows."""
    w = W.small_constrained(N=7, s=4, acc=False)
    for mode in ("hard", "pinned_z"):
        o = Oracle(w.waypoints[0], w.durations[0], w.s, w.rho, samples=8, box_lo=w.box_lo[0], box_hi=w.box_hi[0],
                   vmax=w.vmax, mode=mode)
        o.sweep(3)
        s, N, T = o.s, o.N, o.T
        C, z = o.get("C"), o.get("z")
        avg2 = other2 = 0.0
        for i in range(N):
            B = consensus_matrix(s, T[i]) @ C[i]
            res = B - stacked_z(z, i)
            for r in range(2 * s):
                junction = i + (r >= s)
                averaged = 0 < junction < N and not (r % s == 0)      # orders 1..s-1 at interior junctions
                if averaged and r >= s:
                    Bn = consensus_matrix(s, T[i + 1]) @ C[i + 1]
                    avg2 += ((B[r] - Bn[r - s]) ** 2).sum() / 2.0
                elif not averaged:
                    other2 += (res[r] ** 2).sum()
        rp = o.residuals()["r_p"]
        assert abs(rp ** 2 - (avg2 + other2)) <= 1e-10 * rp ** 2, mode
