"""`-m gpu`: general polytope corridors on the CUDA path (Eq. 7-10) against the
oracle, which forms the coupled (n m) x (n m) operator directly while the CUDA path works per segment in the eigen-frame of
sum_k a_k a_k' (three decoupled operators): iterate-by-iterate parity of every field incl. the per-(sample, plane) slack and
dual, the box written as six planes against the box solver, reset / set_rho / snapshot on a polytope solver."""
import numpy as np
import pytest

from oracle.top_oracle import Oracle
from paper_2507_10290_b200 import build as top_build
from paper_2507_10290_b200 import top
from paper_2507_10290_b200 import workloads as W
from tests.parity_util import scaled
from tests.qcqp_ref import box_as_planes

pytestmark = pytest.mark.gpu
TOL = 1e-9


@pytest.fixture(scope="module", autouse=True)
def built():
    top_build.build()


def poly_oracle(w, b=0, mode="hard", **kw):
    return Oracle(w.waypoints[b], w.durations[b], w.s, w.rho, w.samples, None, None, w.vmax, w.amax, mode=mode,
                  planes=w.planes[b], **kw)


def compare(sol, oracles, w, where):
    c = sol.coeffs()
    st = {f: sol.state(f) for f in ("z", "u", "s_poly", "v_poly", "phi_v", "w_v", "phi_a", "w_a")}
    res = sol.residuals()
    for b, o in enumerate(oracles):
        T = w.durations[b]
        cref = scaled(o.get("coeffs"), T)
        assert np.abs(scaled(c[b], T) - cref).max() / np.abs(cref).max() < TOL, where
        zref = o.get("z")
        assert np.abs(st["z"][b] - zref).max() / np.abs(zref).max() < TOL, where
        assert np.abs(st["u"][b] - o.get("u")).max() / max(np.abs(zref).max(), np.abs(o.get("u")).max()) < TOL, where
        sscale = max(np.abs(o.get("s_poly")).max(), 1e-3)
        for f in ("s_poly", "v_poly"):
            assert np.abs(st[f][b] - o.get(f)).max() / sscale < TOL, (where, f)
        for f, bound in (("phi_v", w.vmax), ("w_v", w.vmax), ("phi_a", w.amax), ("w_a", w.amax)):
            if bound > 0:
                assert np.abs(st[f][b] - o.get(f)).max() / bound < TOL, (where, f)
        if o.iter > 0:
            r = o.residuals()
            assert abs(res["r_p"][b] - r["r_p"]) < TOL * max(r["r_p"], 1e-3 * np.abs(zref).max()), where
            assert abs(res["r_d"][b] - r["r_d"]) < 1e-6 * max(r["r_d"], 1e-3 * w.rho * np.abs(o.get("M")).max() * np.abs(zref).max()), where


@pytest.mark.parametrize("s,acc,K,segs,mode", [(4, True, 7, 8, "hard"), (3, False, 5, 0, "hard"), (4, False, 16, 16, "pinned_z"),
                                               (3, True, 1, 4, "free")])
def test_polytope_iterates_match_oracle(s, acc, K, segs, mode):
    w = W.polytope_corridor(W.small_constrained(N=45, s=s, acc=acc, seed=21), K=K, seed=5)
    sol = top.from_workload(w, segs_per_cta=segs, mode=mode)
    o = poly_oracle(w, mode=mode, long_double=True)
    compare(sol, [o], w, "iterate 0")
    done = 0
    for cp in (1, 2, 3, 10, 50, 200):
        sol.iterate(cp - done); o.sweep(cp - done, 1); done = cp
        compare(sol, [o], w, "sweep %d" % cp)
    assert np.abs(sol.state("v_poly")).max() > 1e-3          # planes really bind
    sol.close()


def test_polytope_batch_and_dims2():
    w = W.polytope_corridor(W.small_constrained(N=30, s=4, acc=True, batch=3, dims=2, seed=4), K=6, seed=9)
    sol = top.from_workload(w, segs_per_cta=8)
    oracles = [poly_oracle(w, b) for b in range(3)]
    for k in (1, 20, 60):
        sol.iterate(k)
        for o in oracles:
            o.sweep(k, 1)
        compare(sol, oracles, w, "batch sweep %d" % k)
    sol.close()


def test_box_as_six_planes_equals_the_box_solver():
    w = W.small_constrained(N=40, s=4, acc=True, seed=8)
    box = top.from_workload(w, segs_per_cta=8)
    wp = W.small_constrained(N=40, s=4, acc=True, seed=8)
    wp.planes, wp.box_lo, wp.box_hi = box_as_planes(w.box_lo[0], w.box_hi[0])[None], None, None
    pol = top.from_workload(wp, segs_per_cta=8)
    for k in (1, 10, 100):
        box.iterate(k); pol.iterate(k)
        T = w.durations[0]
        a, b = scaled(pol.coeffs()[0], T), scaled(box.coeffs()[0], T)
        assert np.abs(a - b).max() / np.abs(b).max() < 1e-10
        assert np.abs(pol.state("z") - box.state("z")).max() / np.abs(box.state("z")).max() < 1e-10
        sp = pol.state("s_poly")[0]
        # plane order of box_as_planes: +x +y +z -x -y -z; the eigen-frame of 2 I is any rotation: slacks are frame-free
        assert np.abs(sp[:, :, :3] - box.state("s_pos")[0]).max() < 1e-9 and np.abs(sp[:, :, 3:] - box.state("s_neg")[0]).max() < 1e-9
    box.close(); pol.close()


def test_polytope_set_rho_reset_snapshot_and_solve():
    w = W.polytope_corridor(W.small_constrained(N=33, s=4, acc=True, seed=2), K=8, seed=1)
    sol = top.from_workload(w, segs_per_cta=8, check_every=1, max_iter=4000)
    o = poly_oracle(w)
    sol.iterate(15); o.sweep(15, 1)
    sol.set_rho(3.0); o.set_rho(3.0)
    sol.iterate(10); o.sweep(10, 1)
    w.rho = 3.0
    compare(sol, [o], w, "after set_rho")
    snap = sol.snapshot()
    sol.iterate(7)
    ref = sol.state("v_poly").copy(); cref = sol.coeffs().copy()
    sol.restore(snap)
    sol.iterate(7)
    assert np.array_equal(sol.state("v_poly"), ref) and np.array_equal(sol.coeffs(), cref)
    # a new problem of the same shape, then the stop rule (host loop) with the oracle's sweep count
    w2 = W.polytope_corridor(W.small_constrained(N=33, s=4, acc=True, seed=3), K=8, seed=6)
    sol.reset(w2.waypoints, w2.durations, w2.rho, vmax=w2.vmax, amax=w2.amax, planes=w2.planes)
    o2 = poly_oracle(w2)
    ito = o2.solve(300.0, 4000)            # (r_d of Eq. 22 is large on these durations: a loose tolerance, hundreds of sweeps)
    assert 5 < ito < 4000, ito
    ok, it = sol.solve(300.0)
    assert ok and int(it[0]) == ito, (it, ito)
    compare(sol, [o2], w2, "after reset + solve")
    sol.close()


def test_polytope_unsupported_combinations():
    w = W.polytope_corridor(W.small_constrained(N=12, s=4, acc=False), K=4)
    for kw in (dict(dtype="f32"), dict(lanes=8), dict(no_mma=True)):
        with pytest.raises(top.TopError) as e:
            top.from_workload(w, **kw)
        assert e.value.status == top.TOP_E_UNSUPPORTED, kw
    w17 = W.polytope_corridor(W.small_constrained(N=12, s=4, acc=False), K=17)
    with pytest.raises(top.TopError) as e:
        top.from_workload(w17)
    assert e.value.status == top.TOP_E_UNSUPPORTED


@pytest.mark.parametrize("s,acc,K,segs,mode", [(4, True, 7, 8, "free"), (3, False, 5, 0, "hard"), (4, True, 12, 16, "pinned_z")])
def test_polytope_with_paper_literal_consensus(s, acc, K, segs, mode):
    """The paper's literal configuration: polytope corridor cells (L222) + 2s-1 consensus orders (L231) + free waypoints
    (Alg. 1 verbatim): the POLY + WIDE instantiation against the oracle's coupled operator with its wide consensus."""
    w = W.polytope_corridor(W.small_constrained(N=45, s=s, acc=acc, seed=23), K=K, seed=6)
    sol = top.from_workload(w, segs_per_cta=segs, mode=mode, consensus="wide")
    o = poly_oracle(w, mode=mode, long_double=True, consensus="wide")
    assert sol.state("z").shape[2] == 2 * s - 1
    compare(sol, [o], w, "iterate 0")
    done = 0
    for cp in (1, 2, 3, 10, 50, 200):
        sol.iterate(cp - done); o.sweep(cp - done); done = cp
        compare(sol, [o], w, "sweep %d" % cp)


def test_polytope_wide_set_rho_and_adaptive_solve():
    """top_set_rho and Eq. 24 on the paper's literal configuration (polytope corridor + n_c = 2s-1): every scaled dual is
    rescaled by rho_old / rho_new -- also the second consensus block (orders s..2s-2) -- so the multipliers rho * u are
    unchanged (reading A16) and the iterates stay on the oracle's (coupled operator, wide consensus)."""
    w = W.polytope_corridor(W.small_constrained(N=33, s=4, acc=True, seed=12), K=6, seed=4)
    sol = top.from_workload(w, segs_per_cta=8, mode="free", consensus="wide")
    o = poly_oracle(w, mode="free", long_double=True, consensus="wide")
    sol.iterate(12); o.sweep(12, 1)
    u_before = sol.state("u").copy()
    assert np.abs(u_before[0, 1:-1, 4:7]).max() > 0 and np.abs(u_before[0, 1:-1, 11:14]).max() > 0     # the second block is live
    sol.set_rho(2.5); o.set_rho(2.5)
    assert np.allclose(sol.state("u") * 2.5, u_before * w.rho, rtol=1e-14, atol=0)       # rho * u unchanged, every row
    w.rho = 2.5
    compare(sol, [o], w, "right after set_rho")
    sol.iterate(9); o.sweep(9, 1)
    compare(sol, [o], w, "9 sweeps after set_rho")
    sol.close()
    # Eq. 24 through top_solve (host loop on polytope solvers: every change of rho goes through top_set_rho)
    w2 = W.polytope_corridor(W.small_constrained(N=33, s=4, acc=True, seed=12), K=6, seed=4)
    o2 = poly_oracle(w2, mode="free", long_double=True, consensus="wide")
    n_ref = o2.solve_adaptive(1e-300, 60, every=2)         # never converges: 60 sweeps with a test (and Eq. 24) every 2nd
    assert n_ref == 60 and o2.rho != w2.rho
    sol2 = top.from_workload(w2, segs_per_cta=8, mode="free", consensus="wide", adaptive_rho=True, check_every=2, max_iter=60)
    ok, it = sol2.solve(1e-300)
    assert not ok and sol2.iteration == 60
    assert sol2.rho == pytest.approx(o2.rho, rel=1e-12)
    w2.rho = o2.rho
    compare(sol2, [o2], w2, "adaptive, 60 sweeps")
    sol2.close()


@pytest.mark.parametrize("Np,kw,segs", [(5920, {}, 40), (4736, {"consensus": "wide", "mode": "free"}, 32)])
def test_polytope_full_size_on_the_plan_bench_times(Np, kw, segs):
    """The two polytope workloads bench.py quotes (config-4 shape, K = 8 planes per segment; N = 5920, and the paper's literal
    configuration with n_c = 2s-1 and free waypoints at N = 4736) on the planner's own launch: 148 CTAs over the L2 mailbox,
    5 / 4 octet warps per CTA -- not the <= 16-CTA cluster plan the small cases above run on.  Every field incl. the
    per-(sample, plane) slack and dual against the long-double oracle's coupled operator, 1e-9."""
    w = W.polytope_corridor(W.config4(seed=1004, N=Np), K=8, seed=3)
    sol = top.from_workload(w, **kw)
    li = sol.launch_info()
    assert li["waves"] == 1 and li["ctas"] > 16 and li["segs_per_cta"] == segs, li
    o = poly_oracle(w, long_double=True, **kw)
    compare(sol, [o], w, "iterate 0")
    done = 0
    for cp in (1, 2, 10, 100):
        sol.iterate(cp - done); o.sweep(cp - done, 0); done = cp
        compare(sol, [o], w, "N=%d sweep %d" % (Np, cp))
    sol.close()


@pytest.mark.parametrize("sync", ["pairwise", "neighbour", "grid"])
@pytest.mark.parametrize("kw", [{}, {"consensus": "wide", "mode": "free"}])
def test_polytope_explicit_sync_modes(sync, kw):
    """POLY / POLY+WIDE over the L2 mailbox with each inter-CTA synchronisation (the explicit modes never use the cluster)."""
    w = W.polytope_corridor(W.small_constrained(N=301, s=4, acc=True, seed=31), K=7, seed=9)
    sol = top.from_workload(w, sync=sync, segs_per_cta=8, **kw)
    assert sol.launch_info()["ctas"] == 38
    o = poly_oracle(w, long_double=True, **kw)
    done = 0
    for cp in (1, 2, 3, 25, 120):
        sol.iterate(cp - done); o.sweep(cp - done, 1); done = cp
        compare(sol, [o], w, "%s sweep %d" % (sync, cp))
    sol.close()


def test_polytope_random_option_sweep():
    """Seeded random sweep over the polytope options (sizes incl. ragged CTAs, s, K, acc, waypoint mode, consensus width, sync mode,
    segments per CTA, rho, launch chunking, a change of rho in between) against the long-double oracle."""
    rng = np.random.default_rng(11)
    for case in range(30):
        N = int(rng.choice([1, 2, 5, 9, 17, 33, 64, 129, 300]))
        s = int(rng.choice([3, 4])); acc = bool(rng.integers(2)); K = int(rng.choice([1, 3, 6, 8, 13, 16]))
        w = W.polytope_corridor(W.small_constrained(N=N, s=s, acc=acc, seed=int(rng.integers(1 << 30))), K=K, seed=int(rng.integers(1 << 30)))
        if rng.integers(3) == 0:
            w.vmax = 0.0
        w.rho = float(rng.choice([0.3, 1.0, 10.0, 80.0]))
        mode = str(rng.choice(["hard", "hard", "pinned_z", "free"]))
        kw = {"consensus": "wide"} if rng.integers(3) == 0 else {}
        sync = str(rng.choice(["auto", "pairwise", "neighbour", "grid"]))
        segs = int(rng.choice([0, 4, 8, 16]))
        sol = top.from_workload(w, mode=mode, sync=sync, segs_per_cta=segs, **kw)
        o = poly_oracle(w, mode=mode, long_double=True, **kw)
        ks = [int(k) for k in rng.integers(1, 40, size=3)]
        for j, k in enumerate(ks):
            sol.iterate(k); o.sweep(k, 1)
            compare(sol, [o], w, (case, N, s, acc, K, w.rho, mode, kw, sync, segs, ks, j))
            if j == 0 and case % 3 == 0:
                w.rho = w.rho * 1.7
                sol.set_rho(w.rho); o.set_rho(w.rho)
        sol.close()
