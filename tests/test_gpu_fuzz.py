"""`-m gpu`: seeded random sweep over the options of the CUDA path (sizes 1..300 incl. ragged CTAs, s, constraint subsets,
dims, batch, rho, waypoint mode, lanes per segment (or the planner's own choice), inter-CTA sync mode ("auto": one
thread-block cluster when the launch is <= 16 CTAs), segments per CTA, launch chunking, consensus width) against the
oracle run in long double; every state field of every compared iterate within 1e-9 norm-relative."""
import numpy as np
import pytest

from paper_2507_10290_b200 import build as top_build
from paper_2507_10290_b200 import top
from paper_2507_10290_b200 import workloads as W
from tests.parity_util import field_errors, make_oracle, sampled_positions

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("seed", [2, 3, 4])
def test_random_option_sweep(seed):
    top_build.build()
    rng = np.random.default_rng(seed)
    for case in range(40):
        N = int(rng.choice([1, 2, 3, 5, 8, 17, 33, 64, 129, 300]))
        s = int(rng.choice([3, 4])); acc = bool(rng.integers(2))
        batch = int(rng.choice([1, 1, 2, 4])); dims = int(rng.choice([3, 3, 2, 1]))
        w = W.small_constrained(N=N, s=s, acc=acc, batch=batch, dims=dims, seed=int(rng.integers(1 << 30)))
        cons = int(rng.integers(4))
        if cons == 0:
            w.samples, w.box_lo, w.box_hi, w.vmax, w.amax = 0, None, None, 0.0, 0.0
        elif cons == 1:
            w.box_lo, w.box_hi = None, None
        elif cons == 2:
            w.vmax = 0.0
        w.rho = float(rng.choice([0.3, 1.0, 10.0, 80.0]))
        mode = str(rng.choice(["hard", "hard", "pinned_z", "free"]))
        lanes = int(rng.choice([8, 4])); sync = str(rng.choice(["pairwise", "neighbour", "grid"]))
        segs = int(rng.choice([0, 4, 8, 16]))
        extra = {}
        if seed >= 4:      # the later additions: planner's own lane choice, cluster exchange, paper-literal consensus
            lanes = int(rng.choice([0, 4])); sync = str(rng.choice(["auto", "auto", "pairwise"]))
            if rng.integers(3) == 0:
                lanes = int(rng.choice([0, 4])); extra = {"consensus": "wide"}
        ks = [int(k) for k in rng.integers(1, 40, size=3)]
        sol = top.from_workload(w, mode=mode, lanes=lanes, sync=sync, segs_per_cta=segs, dtype="f64", **extra)
        oracles = [make_oracle(w, b, mode=mode, long_double=True, **extra) for b in range(batch)]
        for k in ks:
            sol.iterate(k)
            for o in oracles:
                o.sweep(k, 1)
            for name, v in field_errors(sol, oracles, w).items():
                tol = 1e-6 if name.startswith("resself_") else 1e-9
                assert v < tol, (case, name, v, N, s, acc, batch, dims, cons, w.rho, mode, lanes, sync, segs, ks, extra)
        sol.close()
        if case % 4 == 0 and w.samples and not extra:      # the fp32 (mixed) variant on the same case: sampled positions, 1e-3 m
            sol = top.from_workload(w, mode=mode, lanes=lanes, sync=sync, segs_per_cta=segs, dtype="f32")
            sol.iterate(sum(ks))
            for b, o in enumerate(oracles):
                T = w.durations[b]
                d = np.abs(sampled_positions(sol.coeffs()[b].astype(np.float64), T) - sampled_positions(o.get("coeffs"), T)).max()
                assert d < 1e-3, (case, "fp32", d, N, s, acc, batch, dims, cons, w.rho, mode, lanes, sync, segs, ks)
            sol.close()
