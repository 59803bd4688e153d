"""Shared helpers of the GPU parity tests: run the oracle and the CUDA path on the same seeded workload and
compare every state field of an iterate (SURVEY.md section 8(c) "Parity protocol")."""
import numpy as np

from oracle.top_oracle import Oracle, eval_poly

FIELDS_SAMPLE = ["s_pos", "s_neg", "v_pos", "v_neg", "phi_v", "w_v", "phi_a", "w_a"]


def make_oracle(w, b=0, mode="hard", **kw):
    return Oracle(w.waypoints[b], w.durations[b], w.s, w.rho, samples=w.samples,
                  box_lo=None if w.box_lo is None else w.box_lo[b],
                  box_hi=None if w.box_hi is None else w.box_hi[b], vmax=w.vmax, amax=w.amax, mode=mode, **kw)


def scaled(c, T):
    """c^_k = c_k T^k (metres): the norm in which coefficients are compared (reading A12)."""
    n = c.shape[-1]
    return c * (np.asarray(T)[:, None, None] ** np.arange(n)[None, None, :])


def field_errors(solver, oracles, w, b_list=None):
    """Norm-relative error max|gpu - cpu| / scale per field, over the trajectories in b_list."""
    b_list = list(range(len(oracles))) if b_list is None else b_list
    errs = {}

    def upd(name, got, ref, floor):
        scale = max(np.abs(ref).max(), floor)
        errs[name] = max(errs.get(name, 0.0), float(np.abs(got - ref).max() / scale))

    coeffs = solver.coeffs().astype(np.float64)
    z, u = solver.state("z"), solver.state("u")
    samp = {f: solver.state(f) for f in FIELDS_SAMPLE} if w.samples else {}
    res = solver.residuals()
    for k, b in enumerate(b_list):
        o = oracles[k]
        T = w.durations[b]
        cref = scaled(o.get("coeffs"), T)
        upd("coeffs", scaled(coeffs[b], T), cref, 1e-300)
        zref = o.get("z")
        upd("z", z[b], zref, 1e-300)
        upd("u", u[b], o.get("u"), np.abs(zref).max())
        if w.samples:
            sscale = max(np.abs(o.get("s_pos")).max(), np.abs(o.get("s_neg")).max(), 1e-3)
            for f in FIELDS_SAMPLE:
                floor = sscale if f[0] in "sv" else (w.vmax if f.endswith("_v") else w.amax)
                if floor > 0:
                    upd(f, samp[f][b], o.get(f), floor)
        r = o.residuals()
        if o.iter > 0:
            # residual norms: relative to the norm itself, or -- once the iteration has converged to the rounding
            # floor -- to 1e-3 x the scale of the quantities whose difference is normed (with the 1e-6 gate this
            # is the same 1e-9-of-scale bar as for the state fields)
            zmax = np.abs(zref).max()
            Mo = o.get("M")
            Mhat = Mo / (np.asarray(T)[:, None, None] ** np.arange(Mo.shape[-1])[None, None, :])
            floors = {"r_p": 1e-3 * zmax, "r_p_gap": 1e-3 * zmax, "r_d": 1e-3 * w.rho * np.abs(Mo).max() * zmax,
                      "r_d_norm": 1e-3 * w.rho * np.abs(Mhat).max() * zmax}
            for key in ("r_p", "r_d", "r_d_norm", "r_p_gap"):
                ref = r[key]
                errs["res_" + key] = max(errs.get("res_" + key, 0.0), abs(res[key][b] - ref) / max(abs(ref), floors[key]))
    return errs


def sampled_positions(coeffs, T, per_segment=16):
    """Positions at per_segment uniform samples per segment, ends included (fp32 parity metric)."""
    return eval_poly(coeffs, T, 0, np.linspace(0.0, 1.0, per_segment))
