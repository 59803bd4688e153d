"""`-m gpu`: short chains run as ONE thread-block cluster (<= 16 CTAs; boundary rows through distributed shared memory,
DESIGN.md 5.8).  The exchange path must not change a single bit: the same plan over the L2 mailbox (explicit
sync="pairwise") gives identical state; the default plan of top_create matches the oracle iterate by iterate."""
import numpy as np
import pytest

from paper_2507_10290_b200 import build as top_build
from paper_2507_10290_b200 import top
from paper_2507_10290_b200 import workloads as W
from tests.parity_util import field_errors, make_oracle

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def built():
    top_build.build()


def check(errs, where):
    for k, v in errs.items():
        tol = 1e-6 if k.startswith("resself_") else 1e-9
        assert v < tol, (where, k, v)


@pytest.mark.parametrize("maker,kw", [
    (lambda: W.config2(), {}),
    (lambda: W.config3(N=1000), {}),
    (lambda: W.small_constrained(N=301, s=4, acc=True), {}),
    (lambda: W.small_constrained(N=77, s=3, acc=False), {"mode": "free"}),
    (lambda: W.small_constrained(N=60, s=4, acc=True, batch=3), {}),
    (lambda: W.small_constrained(N=120, s=4, acc=True), {"consensus": "wide", "mode": "free"}),
])
def test_default_plan_is_a_cluster_and_matches_oracle(maker, kw):
    w = maker()
    sol = top.from_workload(w, dtype="f64", **kw)
    li = sol.launch_info()
    assert 2 <= li["ctas"] <= 16 and li["waves"] == 1, li
    oracles = [make_oracle(w, b, **kw) for b in range(w.batch)]
    done = 0
    for cp in (1, 2, 3, 10, 100, 500):
        sol.iterate(cp - done)
        for o in oracles:
            o.sweep(cp - done)
        done = cp
        check(field_errors(sol, oracles, w), "sweep %d" % cp)
    # the same plan over the L2 mailbox: bit-identical
    ref = top.from_workload(w, dtype="f64", lanes=4, segs_per_cta=li["segs_per_cta"], sync="pairwise", **kw)
    assert ref.launch_info()["ctas"] == li["ctas"]
    ref.iterate(done)
    for f in ("z", "u") + (("s_pos", "w_v") if w.samples else ()):
        assert np.array_equal(sol.state(f), ref.state(f)), f
    assert np.array_equal(sol.coeffs(), ref.coeffs())


def test_cluster_in_kernel_solve_and_many_launches():
    w = W.config2()
    o = make_oracle(w, 0)
    sol = top.from_workload(w, dtype="f64", check_every=1, max_iter=30000, eps_n_scaled=True)
    assert 2 <= sol.launch_info()["ctas"] <= 16
    it_o = o.solve(0.05 * w.N, 30000)
    ok, it = sol.solve(0.05)
    assert ok and it[0] == it_o, (it, it_o)
    check(field_errors(sol, [o], w, [0]), "after solve")
    for _ in range(50):          # many short launches: mailbox sequence numbers keep growing, the mailbox is re-cleared
        sol.iterate(3); o.sweep(3)
    check(field_errors(sol, [o], w, [0]), "after 50 short launches")


@pytest.mark.parametrize("sync", ["auto", "pairwise", "neighbour"])
def test_mailbox_sequence_numbers_across_the_32_bit_wrap(sync, monkeypatch):
    """The slots of the inter-CTA mailboxes carry the low 32 bits of a sweep counter, and a cleared slot carries 0: a
    launch must never issue 0 (a reader would take a cleared slot for its neighbour's row) nor re-issue a number that a
    slot still holds.  Solvers whose counter starts just below 2^32 (test hook TOP_TEST_SEQ_START) must give bit for bit
    the state of a solver that starts at 0: cluster plan (slots in distributed shared memory) and L2-mailbox plans,
    plain sweeps in launches of several lengths and the in-kernel stop rule (whose launch reserves max_iter numbers but
    must consume only the sweeps it ran)."""
    w = W.small_constrained(N=301, s=4, acc=True) if sync == "auto" else W.small_constrained(N=1200, s=4, acc=True)
    kw = dict(dtype="f64", sync=sync, check_every=4, max_iter=1 << 30)
    ref = top.from_workload(w, **kw)
    ctas = ref.launch_info()["ctas"]
    assert (2 <= ctas <= 16) if sync == "auto" else ctas > 16, ctas
    for start in ((1 << 32) - 40, (1 << 32) - 1, (3 << 32) - 7):
        monkeypatch.setenv("TOP_TEST_SEQ_START", str(start))
        sol = top.from_workload(w, **kw)
        monkeypatch.delenv("TOP_TEST_SEQ_START")
        ref.reset(w.waypoints, w.durations, w.rho, box_lo=w.box_lo, box_hi=w.box_hi, vmax=w.vmax, amax=w.amax)
        for k in (1, 5, 30, 2, 64):          # unguarded, the wrap would fall inside a launch, at a launch boundary, or on the first sweep
            sol.iterate(k); ref.iterate(k)
            for f in ("z", "u", "s_pos", "v_neg", "phi_v", "w_a"):
                assert np.array_equal(sol.state(f), ref.state(f)), (sync, start, k, f)
        assert np.array_equal(sol.coeffs(), ref.coeffs())
        a, b = sol.residuals(), ref.residuals()
        assert all(np.array_equal(a[k], b[k]) for k in a)
        # the in-kernel stop rule reserves max_iter = 2^30 numbers per launch but must consume only the sweeps it ran: six
        # solves that stop at their first test (four such launches used to walk through the whole 32-bit space)
        for _ in range(6):
            oka, ita = sol.solve(1e30); okb, itb = ref.solve(1e30)
            assert oka and okb and ita[0] == itb[0] == 4 and sol.iteration == ref.iteration, (ita, itb)
        assert np.array_equal(sol.state("u"), ref.state("u")) and np.array_equal(sol.coeffs(), ref.coeffs())
        sol.iterate(9); ref.iterate(9)
        assert np.array_equal(sol.state("z"), ref.state("z")) and np.array_equal(sol.state("w_v"), ref.state("w_v"))
        sol.close()
    ref.close()
