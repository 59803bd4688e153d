"""`-m gpu` parity tests: the CUDA path (through the C ABI / ctypes binding) against the CPU oracle on the same
seeded inputs, iterate by iterate.  Tolerances are north_star's: fp64 1e-9 norm-relative per field at every
compared sweep, 1e-6 on coefficients at the end; fp32 (mixed) 1e-3 m on sampled positions."""
import numpy as np
import pytest

from oracle import direct
from paper_2507_10290_b200 import build as top_build
from paper_2507_10290_b200 import top
from paper_2507_10290_b200 import workloads as W
from tests.parity_util import field_errors, make_oracle, sampled_positions, scaled

pytestmark = pytest.mark.gpu

TOL_ITER = 1e-9      # north_star: "GPU fp64 must match the oracle iterate-by-iterate to 1e-9 relative"
TOL_RES = 1e-9       # residual norms: r_p against itself, r_d against its natural scale (parity_util.field_errors)
TOL_RES_SELF = 1e-6  # r_d against itself (a norm of differences of consecutive iterates: DESIGN.md "Residual parity")


@pytest.fixture(scope="module", autouse=True)
def built():
    top_build.build()


def check_fields(errs, where):
    for k, v in errs.items():
        tol = TOL_RES_SELF if k.startswith("resself_") else (TOL_RES if k.startswith("res_") else TOL_ITER)
        assert v < tol, (where, k, v, errs)


def run_parity(w, checkpoints, mode="hard", sync="auto", segs_per_cta=0, b_list=None, long_double=False, threads=1, lanes=0):
    b_list = list(range(w.batch)) if b_list is None else b_list
    oracles = [make_oracle(w, b, mode=mode, long_double=long_double) for b in b_list]
    sol = top.from_workload(w, mode=mode, sync=sync, segs_per_cta=segs_per_cta, dtype="f64", lanes=lanes)
    errs0 = field_errors(sol, oracles, w, b_list)       # iterate 0 (Init, reading A9)
    check_fields(errs0, "iterate 0")
    done = 0
    worst = {}
    for cp in checkpoints:
        sol.iterate(cp - done)
        for o in oracles:
            o.sweep(cp - done, threads)
        done = cp
        assert sol.iteration == done
        errs = field_errors(sol, oracles, w, b_list)
        check_fields(errs, "sweep %d" % cp)
        for k, v in errs.items():
            worst[k] = max(worst.get(k, 0), v)
    return sol, oracles, worst


CHECK_DENSE = list(range(1, 21)) + [50, 100, 200, 300]


def test_config1_iterates_and_direct_solution():
    w = W.config1()
    sol, (o,), worst = run_parity(w, CHECK_DENSE)
    c = sol.coeffs()[0]
    T = w.durations[0]
    ref = direct.banded_optimality(w.waypoints[0], T, w.s)
    assert np.abs(scaled(c - ref, T)).max() / np.abs(scaled(ref, T)).max() < 1e-6
    assert np.abs(scaled(c - o.get("coeffs"), T)).max() / np.abs(scaled(ref, T)).max() < 1e-6


@pytest.mark.parametrize("mode", ["pinned_z", "free"])
def test_config1_other_waypoint_modes(mode):
    run_parity(W.config1(), [1, 2, 3, 10, 100], mode=mode)


@pytest.mark.parametrize("s,acc", [(3, False), (3, True), (4, False), (4, True)])
@pytest.mark.parametrize("sync", ["grid", "neighbour", "pairwise"])
def test_small_constrained_ragged(s, acc, sync):
    """N=37: several CTAs (segs_per_cta=8 -> 5 CTAs, last one ragged with 5 of 8 segments)."""
    w = W.small_constrained(N=37, s=s, acc=acc)
    run_parity(w, [1, 2, 3, 4, 5, 10, 50, 200], sync=sync, segs_per_cta=8)


@pytest.mark.parametrize("segs", [0, 4, 12, 64])
def test_cta_split_does_not_change_results(segs):
    w = W.small_constrained(N=61, s=4, acc=True, seed=21)
    run_parity(w, [1, 7, 64], segs_per_cta=segs)


def test_single_segment_and_two_segments():
    for N in (1, 2, 3):
        w = W.small_constrained(N=N, s=4, acc=True, seed=5)
        run_parity(w, [1, 2, 10, 100])
        w = W.small_constrained(N=N, s=3, acc=False, seed=6)
        w.samples, w.box_lo, w.box_hi, w.vmax = 0, None, None, 0.0
        run_parity(w, [1, 2, 10, 100])


def test_config2_iterates():
    w = W.config2()
    sol, (o,), worst = run_parity(w, [1, 2, 3, 10, 100, 1000, 10000])
    # per-iterate invariants on the GPU state (P10)
    sp, vp = sol.state("s_pos"), sol.state("v_pos")
    assert sp.min() >= 0 and vp.min() >= 0 and np.abs(sp * vp).max() == 0
    phi = sol.state("phi_v")
    assert np.sqrt((phi ** 2).sum(-1)).max() <= w.vmax * (1 + 4e-16)


def test_config3_fp64_iterates_and_converged_rho10():
    w = W.config3()
    run_parity(w, [1, 2, 3, 10, 100, 1000])
    w10 = W.config3(rho=10.0)
    sol = top.from_workload(w10)
    sol.iterate(1000)
    T = w10.durations[0]
    ref = direct.banded_optimality(w10.waypoints[0], T, w10.s)
    assert np.abs(scaled(sol.coeffs()[0] - ref, T)).max() / np.abs(scaled(ref, T)).max() < 1e-6


def test_config3_fp32_positions():
    w = W.config3(dtype="f32")
    o = make_oracle(w)
    o.sweep(1000)
    sol = top.from_workload(w, dtype="f32")
    sol.iterate(1000)
    T = w.durations[0]
    got = sampled_positions(sol.coeffs()[0], T)
    ref = sampled_positions(o.get("coeffs"), T)
    assert np.abs(got - ref).max() < 1e-3


def test_batch_of_trajectories_fp64():
    w = W.small_constrained(N=19, s=4, acc=True, batch=5, seed=3)
    run_parity(w, [1, 2, 3, 20, 100], segs_per_cta=8)


def test_nonrest_end_states():
    w = W.config1()
    sd = np.array([[[1.0, -0.5, 0.2], [0.1, 0.0, -0.3]]])
    ed = np.array([[[-0.7, 0.4, 0.0], [0.0, 0.2, 0.1]]])
    from oracle.top_oracle import Oracle
    o = Oracle(w.waypoints[0], w.durations[0], w.s, w.rho, start_derivs=sd[0], end_derivs=ed[0])
    sol = top.TopSolver(w.waypoints, w.durations, w.s, w.rho, start_derivs=sd, end_derivs=ed)
    for _ in range(5):
        sol.iterate(20); o.sweep(20)
        check_fields(field_errors(sol, [o], w), "end states")


def test_solve_iteration_count_matches_oracle():
    w = W.config1()
    o = make_oracle(w)
    n_ref = o.solve(1e-3, 100000)
    sol = top.from_workload(w, check_every=1, max_iter=100000)
    ok, iters = sol.solve(1e-3)
    assert ok
    if iters[0] != n_ref:      # +-1 only when a residual sits within 1e-9 of eps at that sweep
        assert abs(int(iters[0]) - n_ref) == 1
        r = sol.residuals()
        assert min(abs(r["r_p"][0] - 1e-3), abs(r["r_d"][0] - 1e-3)) < 1e-9 * 1e-3
    ok2, it2 = top.from_workload(w, check_every=32, max_iter=64).solve(1e-12)
    assert not ok2 and it2[0] == 64


def test_dims_1_and_2():
    for dims in (1, 2):
        w = W.small_constrained(N=9, s=4, acc=True, dims=dims, seed=9)
        run_parity(w, [1, 5, 50])


def test_capacity_is_reported():
    assert top.capacity(4, "f64", True) >= 10000
    assert top.capacity(3, "f32", False) >= 14000


@pytest.mark.parametrize("lanes", [8, 4])
def test_streaming_long_chain_matches_oracle(lanes):
    """A chain longer than the on-chip capacity is streamed in pieces with halos (temporal blocking).  Forced here
    with a small segs_per_cta (capacity = #SMs x 4 segments); N = 2000 -> several pieces, halo 64, so 150 sweeps
    cross two halo refreshes.  Results must be those of the resident kernel: iterate parity with the oracle."""
    w = W.small_constrained(N=2000, s=4, acc=True, seed=77)
    # (long-double oracle: at this size the fp64 oracle's own rounding error is the size of the 1e-9 bar, see
    # test_config4_full_size_iterates)
    sol, (o,), worst = run_parity(w, [1, 2, 63, 64, 65, 150], segs_per_cta=4, lanes=lanes, threads=0, long_double=True)
    assert sol.launch_info()["waves"] >= 3
    # bitwise equal to the resident run (same per-segment arithmetic, same order)
    ref = top.from_workload(w, segs_per_cta=16, lanes=lanes)
    assert ref.launch_info()["waves"] == 1
    ref.iterate(150)
    for f in ("z", "u", "s_pos", "v_neg", "phi_v", "w_a"):
        assert np.array_equal(sol.state(f), ref.state(f)), f
    assert np.array_equal(sol.coeffs(), ref.coeffs())


def test_streaming_beyond_capacity_unconstrained():
    cap = top.capacity(3, "f64", False)
    w = W.config3(N=cap + 1000, rho=10.0)
    sol = top.from_workload(w)
    assert sol.launch_info()["waves"] >= 2
    sol.iterate(300)
    T = w.durations[0]
    ref = direct.banded_optimality(w.waypoints[0], T, w.s)
    assert np.abs(scaled(sol.coeffs()[0] - ref, T)).max() / np.abs(scaled(ref, T)).max() < 1e-6


# ------------------------------------------------------------------ BASELINE.json's full sizes, bench.py's launch plan

def test_config4_full_size_iterates():
    """N=10,000 (148 CTAs x 68 segments, the configuration bench.py times): every field, element by element."""
    # The fp64 oracle works in the paper's raw monomial basis (cond(H) up to 1e13, reading A12): at this size its
    # own rounding error against the same oracle in long double is 1e-10..5e-10 norm-relative (measured in
    # test_fp64_oracle_rounding_error_at_full_size), i.e. it would consume the 1e-9 budget.  The CUDA path is
    # therefore held to 1e-9 against the oracle run in long double (same algorithm, same order, more digits).
    w = W.config4()
    sol, (o,), worst = run_parity(w, [1, 2, 10, 100, 300], long_double=True, threads=0)
    info = sol.launch_info()
    assert info["ctas"] >= 140 and info["waves"] == 1
    # per-iterate invariants on the GPU state (P10)
    for side in ("pos", "neg"):
        sp, vp = sol.state("s_" + side), sol.state("v_" + side)
        assert sp.min() >= 0 and vp.min() >= 0 and np.abs(sp * vp).max() == 0
    assert np.sqrt((sol.state("phi_v") ** 2).sum(-1)).max() <= w.vmax * (1 + 1e-15)
    assert np.sqrt((sol.state("phi_a") ** 2).sum(-1)).max() <= w.amax * (1 + 1e-15)
    z = sol.state("z")
    assert np.abs(z[0, :, 0, :] - w.waypoints[0]).max() < 1e-9          # HARD mode: position rows are the waypoints


def test_config4_launch_chunking_is_invisible():
    """top_iterate(k1) then top_iterate(k2) is iterate k1+k2, bit for bit, in both inter-CTA sync modes."""
    w = W.config4(N=1500)
    a = top.from_workload(w, sync="neighbour"); a.iterate(37)
    b = top.from_workload(w, sync="neighbour"); b.iterate(20); b.iterate(1); b.iterate(16)
    c = top.from_workload(w, sync="grid"); c.iterate(37)
    e = top.from_workload(w, sync="pairwise"); e.iterate(30); e.iterate(7)
    assert np.array_equal(a.coeffs(), e.coeffs()) and np.array_equal(a.state("u"), e.state("u"))
    for f in ("z", "u", "s_pos", "v_neg", "phi_v", "w_a"):
        assert np.array_equal(a.state(f), b.state(f)), f
        assert np.array_equal(a.state(f), c.state(f)), f
    assert np.array_equal(a.coeffs(), b.coeffs()) and np.array_equal(a.coeffs(), c.coeffs())
    ra, rb = a.residuals(), b.residuals()
    assert ra["r_p"][0] == rb["r_p"][0] and ra["r_d"][0] == rb["r_d"][0]


def test_config5_batch_fp32_positions():
    """256 x 512 segments, fp32 (mixed), 500 sweeps, 7 waves of whole trajectories: sampled positions of 24
    trajectories spread over the batch (every wave) against the fp64 oracle, 1e-3 m (north_star)."""
    w = W.config5()
    sol = top.from_workload(w)
    assert sol.launch_info()["waves"] > 1
    sol.iterate(500)
    c = sol.coeffs()
    worst = 0.0
    for b in list(range(0, 256, 11)):
        o = make_oracle(w, b)
        o.sweep(500)
        T = w.durations[b]
        err = np.abs(sampled_positions(c[b], T) - sampled_positions(o.get("coeffs"), T)).max()
        worst = max(worst, err)
    assert worst < 1e-3, worst
    r = sol.residuals()
    assert np.all(np.isfinite(r["r_p"])) and r["r_p"].shape == (256,)


def test_config5_batch_fp64_waves_match_oracle():
    """The same batch in fp64 (more waves): wave boundaries and trajectory ends inside CTAs do not leak."""
    w = W.config5(batch=40)
    sol = top.from_workload(w, dtype="f64")
    sol.iterate(60)
    bl = [0, 1, 18, 19, 20, 38, 39]
    oracles = [make_oracle(w, b) for b in bl]
    for o in oracles:
        o.sweep(60)
    check_fields(field_errors(sol, oracles, w, bl), "cfg5 fp64 batch=40")


def test_fp64_oracle_rounding_error_at_full_size():
    """Context for the test above: fp64 oracle vs long-double oracle on config 4, and the CUDA path vs both."""
    w = W.config4()
    o, ol = make_oracle(w), make_oracle(w, long_double=True)
    sol = top.from_workload(w)
    o.sweep(100, 0); ol.sweep(100, 0); sol.iterate(100)
    T = w.durations[0]
    ref = scaled(ol.get("coeffs"), T)
    e_oracle = np.abs(scaled(o.get("coeffs"), T) - ref).max() / np.abs(ref).max()
    e_gpu = np.abs(scaled(sol.coeffs()[0], T) - ref).max() / np.abs(ref).max()
    assert e_gpu < 1e-9
    assert e_oracle < 2e-9            # the fp64 oracle itself stays close to the bar ...
    assert np.abs(scaled(sol.coeffs()[0], T) - scaled(o.get("coeffs"), T)).max() / np.abs(ref).max() < 1e-9 + e_oracle


# ------------------------------------------------------------------ adaptive rho (Eq. 24)

def test_set_rho_matches_oracle_iterates():
    w = W.small_constrained(N=37, s=4, acc=True)
    o = make_oracle(w)
    sol = top.from_workload(w, segs_per_cta=8)
    for rho, k in [(10.0, 20), (3.0, 15), (47.0, 30), (10.0, 10)]:
        sol.set_rho(rho); o.set_rho(rho)
        assert sol.rho == rho
        sol.iterate(k); o.sweep(k)
        check_fields(field_errors(sol, [o], w), "after rho=%g" % rho)


@pytest.mark.parametrize("every", [1, 8])
def test_adaptive_solve_matches_oracle(every):
    w = W.config2(N=40)
    o = make_oracle(w)
    n_ref = o.solve_adaptive(1e-3, 3000, every=every)
    sol = top.from_workload(w, adaptive_rho=True, check_every=every, max_iter=3000)
    ok, iters = sol.solve(1e-3)
    assert sol.rho == pytest.approx(o.rho, rel=1e-12)        # the same sequence of Eq. 24 decisions
    assert int(iters[0]) == n_ref and sol.iteration == o.iter
    check_fields(field_errors(sol, [o], w), "adaptive, every=%d" % every)


def test_adaptive_rho_config1_reaches_direct_solution():
    w = W.config1()
    sol = top.from_workload(w, adaptive_rho=True, check_every=1, max_iter=200000)
    ok, iters = sol.solve(1e-6)
    assert ok and sol.rho != 1.0
    T = w.durations[0]
    ref = direct.banded_optimality(w.waypoints[0], T, w.s)
    assert np.abs(scaled(sol.coeffs()[0] - ref, T)).max() / np.abs(scaled(ref, T)).max() < 1e-6


# ------------------------------------------------------------------ the 4-lanes-per-segment kernel (cadmm_sweeps_kernel4)

@pytest.mark.parametrize("s,acc,segs", [(3, False, 12), (3, True, 8), (4, False, 8), (4, True, 20)])
@pytest.mark.parametrize("sync", ["grid", "pairwise"])
def test_four_lane_kernel_small_ragged(s, acc, segs, sync):
    w = W.small_constrained(N=37, s=s, acc=acc)
    run_parity(w, [1, 2, 3, 10, 50, 200], sync=sync, segs_per_cta=segs, lanes=4)


def test_four_lane_kernel_configs():
    run_parity(W.config1(), [1, 10, 300], lanes=4)
    run_parity(W.config1(), [1, 10, 100], lanes=4, mode="free")
    run_parity(W.config2(), [1, 100, 1000], lanes=4)
    run_parity(W.config3(), [1, 100], lanes=4)
    run_parity(W.config4(), [1, 20, 100], lanes=4, long_double=True, threads=0)
    w = W.small_constrained(N=19, s=4, acc=True, batch=5, seed=3)
    run_parity(w, [1, 20, 100], segs_per_cta=8, lanes=4)


# ------------------------------------------------------------------ device-side stop rule (in-kernel top_solve)

def test_in_kernel_solve_many_ctas_matches_oracle_count():
    """N=1000 -> 125 CTAs of 64 threads: every CTA all-gathers the 125 residual partial sums and stops at the same
    sweep as the oracle (check every sweep)."""
    w = W.config3(rho=10.0)
    o = make_oracle(w)
    n_ref = o.solve(1e-3, 5000)
    sol = top.from_workload(w, check_every=1, max_iter=5000)
    ok, iters = sol.solve(1e-3)
    assert ok and int(iters[0]) == n_ref and sol.iteration == n_ref
    check_fields(field_errors(sol, [o], w), "in-kernel solve, 125 CTAs")
    r, ro = sol.residuals(), o.residuals()
    assert r["r_p"][0] < 1e-3 and abs(r["r_p"][0] - ro["r_p"]) < 1e-9 * max(1.0, ro["r_p"])


def test_in_kernel_solve_equals_host_loop():
    """batch = 1 uses the in-kernel stop rule, batch = 2 (two copies) the host loop: same count, same iterate."""
    w1 = W.config2(N=40)
    a = top.from_workload(w1, check_every=8, max_iter=40000, rd_normalised=True)
    ok_a, it_a = a.solve(1.0)
    w2 = W.config2(N=40)
    w2.batch = 2
    for name in ("waypoints", "durations", "box_lo", "box_hi"):
        setattr(w2, name, np.concatenate([getattr(w1, name)] * 2, axis=0))
    b = top.from_workload(w2, check_every=8, max_iter=40000, rd_normalised=True)
    ok_b, it_b = b.solve(1.0)
    assert ok_a and ok_b and int(it_a[0]) == int(it_b[0]) == int(it_b[1])
    assert np.array_equal(a.coeffs()[0], b.coeffs()[0]) and np.array_equal(a.coeffs()[0], b.coeffs()[1])
    # cap reached: both report the cap and stay usable
    c = top.from_workload(w1, check_every=8, max_iter=24)
    ok_c, it_c = c.solve(1e-12)
    assert not ok_c and int(it_c[0]) == 24 and c.iteration == 24
    c.iterate(8)
    assert c.iteration == 32


# ------------------------------------------------------------------ API surface

def test_device_output_and_user_stream():
    """top_get_coeffs into a device buffer, everything enqueued on a caller-provided (non-default) stream."""
    import torch
    w = W.small_constrained(N=37, s=4, acc=True)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        sol = top.from_workload(w, stream=st.cuda_stream, segs_per_cta=8)
        sol.iterate(25)
        out = torch.zeros((1, w.N, 3, 8), dtype=torch.float64, device="cuda")
        sol.coeffs_to_device(out.data_ptr())
        st.synchronize()
    host = sol.coeffs()
    assert np.array_equal(out.cpu().numpy(), host)
    o = make_oracle(w)
    o.sweep(25)
    T = w.durations[0]
    assert np.abs(scaled(host[0] - o.get("coeffs"), T)).max() / np.abs(scaled(o.get("coeffs"), T)).max() < 1e-9
    # fp32 solver writes fp32 coefficients
    s32 = top.from_workload(w, dtype="f32")
    s32.iterate(5)
    assert s32.coeffs().dtype == np.float32


def test_state_accessor_errors_and_iterate_zero():
    import ctypes
    w = W.small_constrained(N=5, s=3, acc=False)
    sol = top.from_workload(w)
    assert np.all(np.isnan(sol.residuals()["r_p"]))            # NaN before the first sweep
    sol.iterate(0)
    assert sol.iteration == 0
    with pytest.raises(top.TopError) as e:
        sol.state("no_such_field")
    assert e.value.status == top.TOP_E_INVALID
    buf = np.zeros(7)
    st = sol._L.top_get_state(sol._h, b"z", buf.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), buf.size)
    assert st == top.TOP_E_INVALID
    assert np.all(sol.state("phi_a") == 0)                     # a constraint set that is off reads as zeros
    with pytest.raises(top.TopError):
        sol.iterate(-1)
    with pytest.raises(top.TopError):
        sol.set_rho(-2.0)
    z0 = sol.state("z")
    assert np.array_equal(z0[0, :, 0, :], w.waypoints[0])      # iterate 0: z positions are the waypoints (A9)


def test_streaming_batch_fp32_and_solve():
    """Streamed pieces may span trajectory ends (batch of chains longer than the forced capacity); fp32 state in the
    ping-pong buffers; top_set_rho and top_solve (host loop) on a streamed solver."""
    w = W.small_constrained(N=700, s=4, acc=False, batch=3, seed=31)
    sol = top.from_workload(w, segs_per_cta=4, dtype="f64")
    assert sol.launch_info()["waves"] >= 3
    oracles = [make_oracle(w, b) for b in range(3)]
    sol.iterate(70)
    for o in oracles:
        o.sweep(70, 0)
    check_fields(field_errors(sol, oracles, w), "streamed batch, 70 sweeps")
    sol.set_rho(4.0)
    for o in oracles:
        o.set_rho(4.0)
    sol.iterate(70)
    for o in oracles:
        o.sweep(70, 0)
    check_fields(field_errors(sol, oracles, w), "streamed batch after set_rho")
    # fp32 (mixed) on the same streamed plan: positions against the fp64 oracle
    s32 = top.from_workload(w, segs_per_cta=4, dtype="f32")
    s32.set_rho(4.0)          # before any sweep: duals are zero, only the operator changes
    ofresh = make_oracle(w, 1)
    ofresh.set_rho(4.0)
    s32.iterate(130); ofresh.sweep(130, 0)
    T = w.durations[1]
    assert np.abs(sampled_positions(s32.coeffs()[1], T) - sampled_positions(ofresh.get("coeffs"), T)).max() < 1e-3
    # host-loop solve on a streamed solver: stops at a multiple of check_every, reports per-trajectory counts
    s3 = top.from_workload(w, segs_per_cta=4, check_every=16, max_iter=64, rd_normalised=True)
    ok, iters = s3.solve(1e-9)
    assert not ok and np.all(iters == 64) and s3.iteration == 64


def test_snapshot_restore_resumes_bit_for_bit():
    """Checkpoint / resume: save at sweep 40 (after a rho change), restore into a fresh solver, sweep on: identical to
    the uninterrupted run; a snapshot of another problem is refused."""
    w = W.small_constrained(N=150, s=4, acc=True, batch=2, seed=41)
    a = top.from_workload(w, segs_per_cta=8)
    a.iterate(25); a.set_rho(3.0); a.iterate(15)
    snap = a.snapshot()
    a.iterate(33)
    b = top.from_workload(w, segs_per_cta=8)
    b.restore(snap)
    assert b.iteration == 40 and b.rho == 3.0
    assert np.all(np.isfinite(b.residuals()["r_p"]))            # the residuals of sweep 40 travel with the snapshot
    b.iterate(33)
    for f in ("z", "u", "s_pos", "v_neg", "phi_v", "w_a"):
        assert np.array_equal(a.state(f), b.state(f)), f
    assert np.array_equal(a.coeffs(), b.coeffs())
    assert np.array_equal(a.residuals()["r_d"], b.residuals()["r_d"]) and b.iteration == a.iteration == 73
    other = top.from_workload(W.small_constrained(N=150, s=3, acc=True, batch=2, seed=41), segs_per_cta=8)
    with pytest.raises(top.TopError) as e:
        other.restore(snap)
    assert e.value.status == top.TOP_E_INVALID


def test_reset_reuses_the_handle_for_a_new_problem():
    """top_reset: a new problem of the same shape on an existing handle (re-planning): iterates equal those of a fresh
    solver bit for bit, the constraint selection is checked, an adaptive solve after a reset works."""
    w1 = W.small_constrained(N=53, s=4, acc=True, seed=11)
    w2 = W.small_constrained(N=53, s=4, acc=True, seed=12)
    sol = top.from_workload(w1, segs_per_cta=8)
    sol.iterate(40)
    sol.reset(w2.waypoints, w2.durations, 7.0, box_lo=w2.box_lo, box_hi=w2.box_hi, vmax=2.5, amax=4.0)
    assert sol.iteration == 0 and sol.rho == 7.0
    w2.rho, w2.vmax, w2.amax = 7.0, 2.5, 4.0
    fresh = top.from_workload(w2, segs_per_cta=8)
    o = make_oracle(w2)
    for k in (0, 1, 30):
        sol.iterate(k); fresh.iterate(k); o.sweep(k, 1)
        for f in ("z", "u", "s_pos", "v_neg", "phi_v", "w_a"):
            assert np.array_equal(sol.state(f), fresh.state(f)), (k, f)
        assert np.array_equal(sol.coeffs(), fresh.coeffs())
        check_fields(field_errors(sol, [o], w2), "after reset, sweep %d" % k)
    with pytest.raises(top.TopError) as e:      # another constraint selection needs another solver
        sol.reset(w2.waypoints, w2.durations, 7.0, box_lo=w2.box_lo, box_hi=w2.box_hi, vmax=2.5, amax=0.0)
    assert e.value.status == top.TOP_E_INVALID
    # rho changes after a reset go through the (lazily built) spectral form of the NEW problem
    sol.set_rho(3.0); o.set_rho(3.0)
    sol.iterate(5); o.sweep(5, 1)
    check_fields(field_errors(sol, [o], w2), "after reset and set_rho")
    sol.close(); fresh.close()
