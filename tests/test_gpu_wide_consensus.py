"""`-m gpu`: the paper-literal consensus n_c = 2s-1 (TOP_CONSENSUS_WIDE; reading A1) on the
CUDA path against the oracle's wide mode (pinned by tests/test_oracle_wide_consensus.py), iterate by iterate, every field
1e-9 norm-relative; converged results against the direct solution; the in-kernel stop rule, set_rho, snapshot, reset."""
import numpy as np
import pytest

from oracle import direct
from paper_2507_10290_b200 import build as top_build
from paper_2507_10290_b200 import top
from paper_2507_10290_b200 import workloads as W
from tests.parity_util import field_errors, make_oracle, scaled

pytestmark = pytest.mark.gpu

TOL_ITER, TOL_RES, TOL_RES_SELF = 1e-9, 1e-9, 1e-6


@pytest.fixture(scope="module", autouse=True)
def built():
    top_build.build()


def check_fields(errs, where):
    for k, v in errs.items():
        tol = TOL_RES_SELF if k.startswith("resself_") else (TOL_RES if k.startswith("res_") else TOL_ITER)
        assert v < tol, (where, k, v, errs)


def run_wide(w, checkpoints, mode="hard", b_list=None, long_double=False, **kw):
    b_list = list(range(w.batch)) if b_list is None else b_list
    oracles = [make_oracle(w, b, mode=mode, long_double=long_double, consensus="wide") for b in b_list]
    sol = top.from_workload(w, mode=mode, dtype="f64", consensus="wide", **kw)
    assert sol.state("z").shape[2] == 2 * w.s - 1 and sol.state("u").shape[2] == 2 * (2 * w.s - 1)
    check_fields(field_errors(sol, oracles, w, b_list), "iterate 0")
    done = 0
    for cp in checkpoints:
        sol.iterate(cp - done)
        for o in oracles:
            o.sweep(cp - done)
        done = cp
        check_fields(field_errors(sol, oracles, w, b_list), "sweep %d" % cp)
    return sol, oracles


@pytest.mark.parametrize("mode", ["hard", "pinned_z", "free"])
def test_wide_config1_iterates_and_limit(mode):
    w = W.config1()
    sol, (o,) = run_wide(w, list(range(1, 21)) + [50, 100, 300], mode=mode)
    if mode != "free":
        T = w.durations[0]
        ref = direct.banded_optimality(w.waypoints[0], T, w.s)
        assert np.abs(scaled(sol.coeffs()[0] - ref, T)).max() / np.abs(scaled(ref, T)).max() < 1e-6


@pytest.mark.parametrize("s,acc", [(3, False), (3, True), (4, False), (4, True)])
@pytest.mark.parametrize("sync", ["grid", "neighbour", "pairwise"])
def test_wide_small_constrained_ragged(s, acc, sync):
    """N=37, 8 segments per CTA: 5 CTAs (the second row block crosses CTA edges through the mailbox), the last one ragged."""
    w = W.small_constrained(N=37, s=s, acc=acc)
    run_wide(w, [1, 2, 3, 4, 5, 10, 50, 200], sync=sync, segs_per_cta=8)


@pytest.mark.parametrize("mode", ["free", "pinned_z"])
def test_wide_paper_literal_free_waypoints_constrained(mode):
    """Alg. 1 verbatim (waypoints averaged like every other row) with the wide consensus and all sets."""
    w = W.small_constrained(N=37, s=4, acc=True)
    run_wide(w, [1, 2, 3, 10, 100, 400], mode=mode, segs_per_cta=8)


def test_wide_single_segment_and_two_segments():
    for N in (1, 2, 3):
        w = W.small_constrained(N=N, s=4, acc=True)
        run_wide(w, [1, 2, 5, 30])


def test_wide_batch_and_dims2():
    w = W.small_constrained(N=21, s=3, acc=False, batch=5)
    run_wide(w, [1, 3, 20, 100], segs_per_cta=12)
    for dims in (1, 2):
        run_wide(W.small_constrained(N=13, s=4, acc=True, dims=dims, seed=9), [1, 3, 20])


def test_wide_config2_iterates():
    w = W.config2()
    run_wide(w, [1, 10, 100, 1000])


def test_wide_long_chain_many_ctas():
    """N = 4000 snap with all constraint sets: 148 CTAs, every CTA edge exchanges both row blocks."""
    w = W.config4(N=4000)
    run_wide(w, [1, 2, 10, 100], long_double=True)


def test_wide_unconstrained_converges_to_direct_solution_many_ctas():
    w = W.config3(N=200)
    w.rho = 10.0
    sol = top.from_workload(w, dtype="f64", consensus="wide", segs_per_cta=8, check_every=8, max_iter=200000, rd_normalised=True)
    ok, it = sol.solve(1e-7)        # (the high-order rows slow the iteration down: ~1.3e4 sweeps here, 1e3 with n_c = s)
    assert ok
    T = w.durations[0]
    ref = direct.banded_optimality(w.waypoints[0], T, w.s)
    assert np.abs(scaled(sol.coeffs()[0] - ref, T)).max() / np.abs(scaled(ref, T)).max() < 1e-6
    r = sol.residuals()
    assert r["r_p"][0] < 1e-7 and r["r_p_gap"][0] < 1e-7


@pytest.mark.parametrize("ce", [1, 8])
def test_wide_in_kernel_solve_matches_oracle_count(ce):
    # (unconstrained: with the waypoints held, C^(2s-2) junctions leave no freedom for inequality sets to bind -- the
    # constrained HARD + wide problem is generically infeasible and never meets a tolerance)
    w = W.config3(N=37)
    w.rho = 10.0
    o = make_oracle(w, 0, consensus="wide")
    sol = top.from_workload(w, dtype="f64", consensus="wide", segs_per_cta=8, check_every=ce, max_iter=20000)
    eps = 1.0
    it_o = 0
    while it_o < 20000:
        o.sweep(ce); it_o += ce
        r = o.residuals()
        if r["r_p"] < eps and r["r_d"] < eps:
            break
    ok, it = sol.solve(eps)
    assert ok and it[0] == it_o, (it, it_o)
    check_fields(field_errors(sol, [o], w, [0]), "after solve")


def test_wide_adaptive_solve_matches_oracle():
    w = W.small_constrained(N=23, s=4, acc=True)
    o = make_oracle(w, 0, consensus="wide")
    sol = top.from_workload(w, dtype="f64", consensus="wide", segs_per_cta=8, check_every=1, max_iter=400, adaptive_rho=True,
                            eps_n_scaled=True)
    it_o = o.solve_adaptive(0.05 * w.N, 400)
    ok, it = sol.solve(0.05)
    assert it[0] == it_o and abs(sol.rho - o.rho) <= 1e-12 * o.rho, (it, it_o, sol.rho, o.rho)
    check_fields(field_errors(sol, [o], w, [0]), "after adaptive solve")


def test_wide_set_rho_snapshot_reset():
    w = W.small_constrained(N=29, s=4, acc=True)
    o = make_oracle(w, 0, consensus="wide")
    sol = top.from_workload(w, dtype="f64", consensus="wide", segs_per_cta=8)
    sol.iterate(7); o.sweep(7)
    sol.set_rho(3.5); o.set_rho(3.5)
    sol.iterate(5); o.sweep(5)
    w.rho = 3.5
    check_fields(field_errors(sol, [o], w, [0]), "after set_rho")
    snap = sol.snapshot()
    sol.iterate(9)
    a = {f: sol.state(f) for f in ("z", "u", "w_v")}
    sol.restore(snap)
    sol.iterate(9)
    for f, v in a.items():
        assert np.array_equal(sol.state(f), v), f
    # a snapshot of a wide solver does not restore into a default one
    other = top.from_workload(w, dtype="f64", segs_per_cta=8)
    with pytest.raises(top.TopError):
        other.restore(snap)
    # reset: a new problem on the live handle
    w2 = W.small_constrained(N=29, s=4, acc=True, seed=77)
    o2 = make_oracle(w2, 0, consensus="wide")
    sol.reset(w2.waypoints[0], w2.durations[0], w2.rho, box_lo=w2.box_lo[0], box_hi=w2.box_hi[0], vmax=w2.vmax, amax=w2.amax)
    sol.iterate(11); o2.sweep(11)
    check_fields(field_errors(sol, [o2], w2, [0]), "after reset")


def test_wide_unsupported_combinations():
    w = W.small_constrained(N=9, s=4, acc=False)
    for kw in ({"dtype": "f32"}, {"dtype": "f64", "lanes": 8}, {"dtype": "f64", "no_mma": True, "lanes": 4}):
        with pytest.raises(top.TopError) as e:
            top.from_workload(w, consensus="wide", **kw)
        assert e.value.status == top.TOP_E_UNSUPPORTED
    big = W.config4(N=10000)
    with pytest.raises(top.TopError) as e:
        top.from_workload(big, consensus="wide", dtype="f64")
    assert e.value.status == top.TOP_E_UNSUPPORTED
