"""`-m gpu`: race evidence for the synchronisation the fp64 tensor-core kernel builds by hand (warp-pair named barriers with
per-pair thread counts, split octets on three warps, the LL mailbox in L2, the cluster mailbox and residual all-gather in
distributed shared memory).  compute-sanitizer is not available on the test runner, so the evidence is
behavioural: a few hundred seeded random cases in which the planner's own launch (cluster and / or split, pairwise
barriers) and the same problem with one CTA-wide barrier per sweep over the L2 mailbox (sync="neighbour": no split, no
cluster, no named barriers) must agree BIT FOR BIT -- state, coefficients, residual sums, sweep counts and rho sequence of
the in-kernel stop rule.  A missed wait or a barrier with a wrong thread count shows as a differing bit in some case."""
import numpy as np
import pytest

from paper_2507_10290_b200 import build as top_build
from paper_2507_10290_b200 import top
from paper_2507_10290_b200 import workloads as W

pytestmark = pytest.mark.gpu

STATE = ("z", "u", "s_pos", "s_neg", "v_pos", "v_neg", "phi_v", "w_v", "phi_a", "w_a")


def same_bits(a, b, w, where):
    for f in STATE:
        if (f.endswith("_a") and not w.amax) or (f.endswith("_v") and not w.vmax) or (f[0] in "sv" and w.box_lo is None):
            continue
        assert np.array_equal(a.state(f), b.state(f)), (where, f)
    assert np.array_equal(a.coeffs(), b.coeffs()), where
    ra, rb = a.residuals(), b.residuals()
    for k in ra:
        assert np.array_equal(ra[k], rb[k]), (where, k, ra[k], rb[k])


@pytest.mark.parametrize("seed", [101, 102, 103, 104, 105])
def test_planner_launch_equals_cta_barrier_launch_bit_for_bit(seed):
    top_build.build()
    rng = np.random.default_rng(seed)
    plans = set()
    for case in range(100):
        s = int(rng.choice([3, 4])); acc = bool(rng.integers(2))
        segs = int(rng.choice([0, 0, 4, 8, 12, 16, 20, 24, 36, 40, 68, 72]))
        if segs == 0:
            N = int(rng.choice([int(rng.integers(9, 400)), int(rng.integers(400, 3000))]))
        else:
            N = int(rng.integers(segs + 1, min(148 * segs, 40 * segs) + 1))      # 2..40 CTAs of that size
        w = W.small_constrained(N=N, s=s, acc=acc, seed=int(rng.integers(1 << 30)))
        if rng.integers(5) == 0:      # (the split instantiation needs box + velocity; other selections run unsplit)
            w.vmax = 0.0
        w.rho = float(rng.choice([1.0, 10.0, 80.0]))
        mode = str(rng.choice(["hard", "hard", "pinned_z", "free"]))
        ce = int(rng.choice([1, 2, 3, 4, 8, 32])); adaptive = bool(rng.integers(2))
        kw = dict(dtype="f64", lanes=4, mode=mode, check_every=ce, max_iter=int(rng.integers(20, 200)), adaptive_rho=adaptive)
        a = top.from_workload(w, segs_per_cta=segs, **kw)                       # the planner's launch (sync auto)
        li = a.launch_info()
        b = top.from_workload(w, segs_per_cta=li["segs_per_cta"], sync="neighbour", **kw)
        lb = b.launch_info()
        assert lb["ctas"] == li["ctas"] and lb["threads"] == 32 * ((li["segs_per_cta"] + 7) // 8), (li, lb)
        plans.add((li["ctas"] <= 16, li["threads"] != lb["threads"]))
        where = (seed, case, N, s, acc, segs, w.vmax, w.rho, mode, ce, adaptive, li)
        for k in rng.integers(1, 50, size=3):
            a.iterate(int(k)); b.iterate(int(k))
            same_bits(a, b, w, where)
        # the stop rule (in the kernel for these single-trajectory solvers) and Eq. 24: same decisions on both launches
        eps = float(rng.choice([1e-30, 0.5, 0.9])) * float(a.residuals()["r_p"][0])
        oka, ita = a.solve(eps); okb, itb = b.solve(eps)
        assert oka == okb and ita[0] == itb[0] and a.rho == b.rho and a.iteration == b.iteration, (where, ita, itb, a.rho, b.rho)
        same_bits(a, b, w, where)
        a.iterate(7); b.iterate(7)
        same_bits(a, b, w, where)
        a.close(); b.close()
    # the draw reached cluster and L2 plans, split and unsplit launches
    assert {p[0] for p in plans} == {True, False} and {p[1] for p in plans} == {True, False}, plans
