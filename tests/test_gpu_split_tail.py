"""`-m gpu`: the split tail of the fp64 tensor-core kernel: CTAs holding 4k+1 octets (5 or 9 warps of 8
segments) run their LAST octet on three warps, one flat dimension each.  The arithmetic of a (row, dim) is that of the
unsplit lane, so the results must be bit-identical to a launch that does not split (sync="neighbour" keeps the CTA barrier
and therefore the unsplit kernel) -- state, coefficients and residual sums -- and match the oracle iterate by iterate."""
import numpy as np
import pytest

from paper_2507_10290_b200 import build as top_build
from paper_2507_10290_b200 import top
from paper_2507_10290_b200 import workloads as W
from tests.parity_util import field_errors, make_oracle

pytestmark = pytest.mark.gpu

STATE = ("z", "u", "s_pos", "s_neg", "v_pos", "v_neg", "phi_v", "w_v", "phi_a", "w_a")


@pytest.fixture(scope="module", autouse=True)
def built():
    top_build.build()


def check(errs, where):
    for k, v in errs.items():
        tol = 1e-6 if k.startswith("resself_") else 1e-9
        assert v < tol, (where, k, v)


def pair(w, segs, **kw):
    split = top.from_workload(w, dtype="f64", lanes=4, segs_per_cta=segs, sync="pairwise", **kw)
    plain = top.from_workload(w, dtype="f64", lanes=4, segs_per_cta=segs, sync="neighbour", **kw)
    octets = (segs + 7) // 8
    ls, lp = split.launch_info(), plain.launch_info()
    assert ls["ctas"] == lp["ctas"] >= 2
    assert lp["threads"] == 32 * octets and ls["threads"] == 32 * (octets + 2), (ls, lp)      # last octet on three warps
    return split, plain


def same_bits(a, b, w, where):
    for f in STATE:
        if f.endswith("_a") and not w.amax:
            continue
        assert np.array_equal(a.state(f), b.state(f)), (where, f)
    assert np.array_equal(a.coeffs(), b.coeffs()), where
    ra, rb = a.residuals(), b.residuals()
    for k in ra:
        assert np.array_equal(ra[k], rb[k]), (where, k, ra[k], rb[k])


@pytest.mark.parametrize("s,acc", [(4, True), (4, False), (3, True), (3, False)])
@pytest.mark.parametrize("N,segs", [
    (150, 68),      # 9 octets, tail half full; the last CTA holds 14 segments: its tail octet is empty
    (133, 68),      # the last CTA holds 65 segments: its tail octet has ONE segment, the trajectory's last
    (216, 72),      # full tail octets, three full CTAs
    (100, 36),      # 5 octets
])
def test_split_tail_bit_identical_and_matches_oracle(N, segs, s, acc):
    w = W.small_constrained(N=N, s=s, acc=acc)
    split, plain = pair(w, segs)
    o = make_oracle(w, 0)
    done = 0
    for cp in (1, 2, 3, 10, 60):
        split.iterate(cp - done); plain.iterate(cp - done); o.sweep(cp - done)
        done = cp
        same_bits(split, plain, w, "sweep %d" % cp)
        check(field_errors(split, [o], w, [0]), "sweep %d" % cp)


@pytest.mark.parametrize("mode", ["pinned_z", "free"])
def test_split_tail_waypoint_modes_and_batch(mode):
    w = W.small_constrained(N=70, s=4, acc=True, batch=3)      # 3 trajectories of 70 segments in one chain of CTAs of 68
    split, plain = pair(w, 68, mode=mode)
    oracles = [make_oracle(w, b, mode=mode) for b in range(w.batch)]
    split.iterate(25); plain.iterate(25)
    for o in oracles:
        o.sweep(25)
    same_bits(split, plain, w, mode)
    check(field_errors(split, oracles, w), mode)


def test_split_tail_default_plan_config4_and_many_launches():
    """config 4 (N = 10 000: 148 CTAs x 68 segments) takes the split launch by default; chunked launches are bit-identical."""
    w = W.config4()
    a = top.from_workload(w, dtype="f64")
    li = a.launch_info()
    assert li["ctas"] == 148 and li["segs_per_cta"] == 68 and li["threads"] == 352, li
    b = top.from_workload(w, dtype="f64", sync="neighbour")
    assert b.launch_info()["threads"] == 288
    a.iterate(40)
    for k in (1, 2, 3, 4, 30):
        b.iterate(k)
    same_bits(a, b, w, "config 4, 40 sweeps")
    # set_rho between launches (operator rows re-read by the tail warps), then on
    a.set_rho(4.0); b.set_rho(4.0)
    a.iterate(7); b.iterate(7)
    same_bits(a, b, w, "after set_rho")
    # the in-kernel stop rule runs the unsplit SOLVE instantiation from the state the split launches left
    a2 = top.from_workload(W.small_constrained(N=150, s=4, acc=True), dtype="f64", lanes=4, segs_per_cta=68, sync="pairwise", check_every=4, max_iter=40)
    b2 = top.from_workload(W.small_constrained(N=150, s=4, acc=True), dtype="f64", lanes=4, segs_per_cta=68, sync="neighbour", check_every=4, max_iter=40)
    a2.iterate(9); b2.iterate(9)
    a2.solve(1e-12); b2.solve(1e-12)
    same_bits(a2, b2, W.small_constrained(N=150, s=4, acc=True), "iterate then solve")


# ---- short chains as one cluster: EVERY octet of a CTA on three warps (<= 3 octets per CTA), sweeps and in-kernel solve

@pytest.mark.parametrize("N,s,acc,threads", [
    (100, 4, False, 96),      # config 2's shape: 13 CTAs of one octet
    (77, 3, True, 96),
    (200, 4, True, 192),      # two octets per CTA
    (301, 4, True, 288),      # three; the last CTA is ragged
    (500, 4, True, 128),      # four octets per CTA: not split
])
def test_all_octets_split_in_a_cluster_bit_identical(N, s, acc, threads):
    w = W.small_constrained(N=N, s=s, acc=acc)
    a = top.from_workload(w, dtype="f64")
    li = a.launch_info()
    assert 2 <= li["ctas"] <= 16 and li["threads"] == threads, li
    b = top.from_workload(w, dtype="f64", lanes=4, segs_per_cta=li["segs_per_cta"], sync="neighbour")      # L2 mailbox, unsplit
    assert b.launch_info()["threads"] == 32 * ((li["segs_per_cta"] + 7) // 8)
    o = make_oracle(w, 0)
    done = 0
    for cp in (1, 2, 3, 10, 100, 400):
        a.iterate(cp - done); b.iterate(cp - done); o.sweep(cp - done)
        done = cp
        same_bits(a, b, w, "sweep %d" % cp)
        check(field_errors(a, [o], w, [0]), "sweep %d" % cp)


@pytest.mark.parametrize("adaptive", [False, True])
@pytest.mark.parametrize("N,ce", [(100, 1), (100, 3), (200, 4), (301, 1)])
def test_all_octets_split_in_kernel_solve(N, ce, adaptive):
    """The SPLIT + SOLVE instantiation: same decisions, same sweep count, same rho sequence as the oracle and as the unsplit
    solve kernel; state bit-identical to the latter."""
    w = W.small_constrained(N=N, s=4, acc=True)
    kw = dict(check_every=ce, max_iter=600, adaptive_rho=adaptive, eps_n_scaled=True)
    a = top.from_workload(w, dtype="f64", **kw)
    li = a.launch_info()
    assert li["threads"] == 96 * ((li["segs_per_cta"] + 7) // 8), li
    b = top.from_workload(w, dtype="f64", lanes=4, segs_per_cta=li["segs_per_cta"], sync="neighbour", **kw)
    o = make_oracle(w, 0)
    eps = 0.05
    if adaptive and ce == 1:
        it_o = o.solve_adaptive(eps * w.N, 600)
    else:
        it_o = None
    oka, ita = a.solve(eps)
    okb, itb = b.solve(eps)
    assert oka == okb and ita[0] == itb[0] and a.rho == b.rho, (ita, itb, a.rho, b.rho)
    same_bits(a, b, w, "after solve")
    if it_o is not None:
        assert ita[0] == it_o and abs(a.rho - o.rho) <= 1e-12 * o.rho, (ita, it_o, a.rho, o.rho)
        check(field_errors(a, [o], w, [0]), "after adaptive solve")
    elif not adaptive:
        o.sweep(int(ita[0]))
        check(field_errors(a, [o], w, [0]), "after solve")
    # and on from there with plain sweeps (split launch continues from the solve kernel's state)
    a.iterate(5); b.iterate(5)
    same_bits(a, b, w, "solve then iterate")
