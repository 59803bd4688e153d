"""`-m gpu`: the NumericSolve branch (TOP_XUPDATE_NUMERIC; Eq. 15-17, Alg. 1 lines 6-7; reading A20) on
the CUDA path against the oracle's numeric branch (pinned by tests/test_oracle_numeric.py).

Tolerance.  The x-update is an inner ITERATION stopped when the L-BFGS step falls below 1e-10 of the coefficients (or the
line search reaches the rounding floor): two correct implementations agree on c^{k+1} to about that tolerance, not to
rounding, and the difference is carried from sweep to sweep (ADMM is non-expansive: at most additively).
derives the bar used here: 1e-6 norm-relative on every field over the first few hundred sweeps (measured: 1e-14 after one
sweep, <= 4e-7 after 300)."""
import numpy as np
import pytest

from paper_2507_10290_b200 import build as top_build
from paper_2507_10290_b200 import top
from paper_2507_10290_b200 import workloads as W
from tests import qcqp_ref as Q
from tests.parity_util import make_oracle, scaled

pytestmark = pytest.mark.gpu
TOL = 1e-6


@pytest.fixture(scope="module", autouse=True)
def built():
    top_build.build()


def compare(sol, oracles, w, where, tol=TOL):
    worst = {}
    coeffs, z, u = sol.coeffs(), sol.state("z"), sol.state("u")
    st = {f: sol.state(f) for f in ("s_pos", "s_neg", "v_pos", "v_neg", "y_v", "y_a")}
    res = sol.residuals()
    for b, o in enumerate(oracles):
        T = w.durations[b]
        ref = scaled(o.get("coeffs"), T)
        worst["coeffs"] = max(worst.get("coeffs", 0), np.abs(scaled(coeffs[b], T) - ref).max() / np.abs(ref).max())
        zr = o.get("z")
        worst["z"] = max(worst.get("z", 0), np.abs(z[b] - zr).max() / np.abs(zr).max())
        worst["u"] = max(worst.get("u", 0), np.abs(u[b] - o.get("u")).max() / np.abs(zr).max())
        for f in st:
            r = o.get(f)
            floor = max(np.abs(o.get("s_pos")).max(), 1e-3) if f[0] in "sv" else max(np.abs(r).max(), 1e-6)
            worst[f] = max(worst.get(f, 0), np.abs(st[f][b] - r).max() / floor)
        ro = o.residuals()
        if o.iter > 0:
            worst["r_p"] = max(worst.get("r_p", 0), abs(res["r_p"][b] - ro["r_p"]) / max(ro["r_p"], 1e-3 * np.abs(zr).max()))
    for k, v in worst.items():
        assert v < tol, (where, k, v, worst)
    return worst


def run(w, checkpoints, mode="hard", **kw):
    oracles = [make_oracle(w, b, mode=mode, numeric=True) for b in range(w.batch)]
    sol = top.from_workload(w, dtype="f64", mode=mode, numeric=True, **kw)
    compare(sol, oracles, w, "iterate 0")
    done = 0
    for cp in checkpoints:
        sol.iterate(cp - done)
        for o in oracles:
            o.sweep(cp - done)
        done = cp
        compare(sol, oracles, w, "sweep %d" % cp)
    return sol, oracles


def tiny(vscale=1.0, amax=0.0):
    unc, lo, hi, vmax = Q.tiny_instance()
    return W.Workload("tiny_qcqp", 1, 3, 3, 3, "f64", Q.WP[None].astype(float), Q.TT[None], rho=10.0, samples=8,
                      box_lo=lo[None], box_hi=hi[None], vmax=vmax * vscale, amax=amax)


@pytest.mark.parametrize("mode", ["hard", "pinned_z", "free"])
def test_numeric_tiny_instance(mode):
    sol, (o,) = run(tiny(0.9, 2.5), [1, 2, 3, 5, 10, 30, 100, 300], mode=mode)
    if mode != "free":
        assert o.get("y_v").max() > 0                                  # the multipliers are in play
    gi, oi = sol.inner_iterations(), o.inner_iters
    assert 0.5 * oi - 10 <= gi <= 1.5 * oi + 10, (gi, oi)               # comparable inner work (the stop decisions are taken at a
                                                                        # tolerance near the rounding floor: the counts differ)


@pytest.mark.parametrize("s,acc", [(3, False), (4, False), (4, True)])
def test_numeric_small_constrained(s, acc):
    w = W.small_constrained(N=37, s=s, acc=acc)
    run(w, [1, 2, 5, 20, 60])


def test_numeric_batch_and_dims():
    run(W.small_constrained(N=21, s=3, acc=False, batch=4), [1, 3, 20])
    for dims in (1, 2):
        run(W.small_constrained(N=13, s=4, acc=True, dims=dims, seed=9), [1, 3, 20])


def test_numeric_without_violation_is_the_closed_form_branch():
    """No ball violated: one L-BFGS step with the exact inverse Hessian lands on the closed-form x-update."""
    w = W.small_constrained(N=29, s=4, acc=False)
    w.vmax = 1e3
    num = top.from_workload(w, dtype="f64", numeric=True)
    wc = W.small_constrained(N=29, s=4, acc=False)
    wc.vmax = 0.0
    cf = top.from_workload(wc, dtype="f64")
    for k in (1, 5, 50):
        num.iterate(k - num.iteration); cf.iterate(k - cf.iteration)
        for f in ("z", "u", "s_pos", "v_neg"):
            a, b = num.state(f), cf.state(f)
            assert np.abs(a - b).max() <= 1e-10 * max(1.0, np.abs(b).max()), (k, f)
    assert num.state("y_v").max() == 0
    assert num.inner_iterations() <= 2 * 50 * w.N


def test_numeric_solve_and_full_size_sampled():
    """N = 10 000 (config 4's shape): 3 sweeps against the oracle on every field, then top_solve's host loop runs."""
    w = W.config4(N=10000)
    sol, _ = run(w, [1, 3])
    w2 = tiny(0.97)
    s2 = top.from_workload(w2, dtype="f64", numeric=True, check_every=10, max_iter=3000, eps_n_scaled=True)
    ok, it = s2.solve(0.05)
    assert ok and it[0] % 10 == 0 and it[0] < 3000
    r = s2.residuals()
    assert r["r_p"][0] < 0.15 and r["r_d"][0] < 0.15


def test_numeric_set_rho_and_adaptive_rho():
    """Eq. 24 / top_set_rho in the numeric branch: the multipliers of Eq. 17 are scaled duals too (times rho_old / rho_new),
    the initial inverse Hessian is rebuilt for the new rho."""
    w = tiny(0.9, 2.5)
    o = make_oracle(w, 0, numeric=True)
    sol = top.from_workload(w, dtype="f64", numeric=True)
    sol.iterate(15); o.sweep(15)
    sol.set_rho(3.5); o.set_rho(3.5)
    sol.iterate(25); o.sweep(25)
    compare(sol, [o], w, "after set_rho")
    # Alg. 1 line 14 every sweep, the paper's parameters, N-scaled tolerance
    o2 = make_oracle(w, 0, numeric=True)
    s2 = top.from_workload(w, dtype="f64", numeric=True, adaptive_rho=True, check_every=1, max_iter=120, eps_n_scaled=True)
    it_o = o2.solve_adaptive(0.05 * w.N, 120)
    ok, it = s2.solve(0.05)
    assert it[0] == it_o and abs(s2.rho - o2.rho) <= 1e-12 * o2.rho, (it, it_o, s2.rho, o2.rho)
    compare(s2, [o2], w, "after adaptive solve")


def test_numeric_unsupported():
    w = W.small_constrained(N=9, s=4, acc=False)
    for kw in ({"dtype": "f32"}, {"dtype": "f64", "consensus": "wide"}):
        with pytest.raises(top.TopError) as e:
            top.from_workload(w, numeric=True, **kw)
        assert e.value.status == top.TOP_E_UNSUPPORTED
    with pytest.raises(top.TopError):
        top.from_workload(w, dtype="f64", numeric=True).snapshot()
    with pytest.raises(top.TopError):
        top.from_workload(w, dtype="f64").inner_iterations()


def test_numeric_random_option_sweep():
    """Seeded random draws over the NumericSolve options (N incl. 1 and sizes that span several CTAs, s, box / ball subsets, waypoint
    mode, rho, batch) against the oracle's numeric branch, at the derived 1e-6 bar, over the first sweeps."""
    rng = np.random.default_rng(29)
    for case in range(12):
        N = int(rng.choice([1, 2, 5, 17, 64, 129, 300])); s = int(rng.choice([3, 4])); acc = bool(rng.integers(2))
        batch = int(rng.choice([1, 1, 2]))
        w = W.small_constrained(N=N, s=s, acc=acc, batch=batch, seed=int(rng.integers(1 << 30)))
        if rng.integers(4) == 0:
            w.box_lo, w.box_hi = None, None
        w.rho = float(rng.choice([1.0, 10.0, 80.0]))
        mode = str(rng.choice(["hard", "hard", "pinned_z", "free"]))
        cps = sorted(set(int(k) for k in rng.integers(1, 25, size=3)))
        run(w, cps, mode=mode)[0].close()
