"""Seeded synthetic inputs for the five BASELINE.json configs.

This module holds NONE of the method's arithmetic: it only draws waypoints,
durations and constraint-set parameters.  It is the single piece of code that
both the CPU oracle's tests and the CUDA path's tests / bench share
(task rule: "only the seeded input generators serve both").

The paper's own workloads are RRT* paths inside FIRI corridors (PAPER.md:L301,
L222) and N+1 points sampled from a curve; neither the maps
nor the curve are available, so seeded random walks with the same shape
(tens .. thousands of segments, 0.5-5 m long) stand in for them
(DESIGN.md "Input recipe").

Every generator returns a `Workload` with host float64 numpy arrays:
  waypoints  [batch, N+1, dims]   metres
  durations  [batch, N]           seconds
  box_lo/hi  [batch, N, dims] or None
  vmax, amax                      <=0 means "constraint off"
Start and end are at rest (derivatives 1..s-1 zero) in all configs.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np


@dataclass
class Workload:
    name: str
    batch: int
    N: int
    s: int                     # 3 = minimum jerk, 4 = minimum snap
    dims: int
    dtype: str                 # "f64" or "f32": arithmetic type of the GPU run
    waypoints: np.ndarray      # [batch, N+1, dims]
    durations: np.ndarray      # [batch, N]
    rho: float
    samples: int = 0           # Ms; 0 => no inequality constraints
    box_lo: Optional[np.ndarray] = None   # [batch, N, dims]
    box_hi: Optional[np.ndarray] = None
    vmax: float = 0.0
    amax: float = 0.0
    planes: Optional[np.ndarray] = None   # general polytope corridor [batch, N, K, dims+1]: a_k'p <= b_k (replaces the box)
    sweeps: int = 0            # fixed sweep count of the config (0 = run to eps)
    eps: float = 0.0           # tolerance of the config (0 = fixed sweeps)
    notes: dict = field(default_factory=dict)

    @property
    def constrained(self) -> bool:
        return self.samples > 0


def _random_directions(rng: np.random.Generator, count: int, dims: int) -> np.ndarray:
    """Uniform random unit vectors: normalised standard normals."""
    g = rng.standard_normal((count, dims))
    nrm = np.sqrt((g * g).sum(axis=1, keepdims=True))
    nrm[nrm == 0.0] = 1.0
    return g / nrm


def _random_walk(rng: np.random.Generator, N: int, dims: int, step_lo: float, step_hi: float):
    """Walk from the origin: N steps, length U[step_lo, step_hi], uniform direction."""
    steps = rng.uniform(step_lo, step_hi, size=N)
    dirs = _random_directions(rng, N, dims)
    pts = np.zeros((N + 1, dims))
    pts[1:] = np.cumsum(dirs * steps[:, None], axis=0)
    return pts, steps


def _chord_box(pts: np.ndarray, half_width) -> tuple[np.ndarray, np.ndarray]:
    """Axis-aligned corridor: per-axis [min(p_{i-1},p_i)-h, max(p_{i-1},p_i)+h]."""
    a, b = pts[:-1], pts[1:]
    h = np.asarray(half_width, dtype=np.float64)
    if h.ndim == 1:
        h = h[:, None]
    return np.minimum(a, b) - h, np.maximum(a, b) + h


def config1(seed: int = 1001) -> Workload:
    """N=4, 3D, minimum jerk, fp64, no constraints, rho=1, 300 sweeps."""
    rng = np.random.default_rng(seed)
    N, dims = 4, 3
    pts = rng.uniform(-10.0, 10.0, size=(N + 1, dims))
    chord = np.sqrt(((pts[1:] - pts[:-1]) ** 2).sum(axis=1))
    T = np.maximum(0.5, chord / 2.0)
    return Workload("cfg1_N4_jerk_f64", 1, N, 3, dims, "f64", pts[None], T[None], rho=1.0, sweeps=300)


def config2(seed: int = 1002, N: int = 100) -> Workload:
    """N=100, 3D, minimum snap, fp64, box corridor h=1.5 m, ||v||<=3 at 8 samples, rho=10."""
    rng = np.random.default_rng(seed)
    dims = 3
    pts, steps = _random_walk(rng, N, dims, 1.0, 5.0)
    T = steps / 2.0
    lo, hi = _chord_box(pts, 1.5)
    return Workload("cfg2_N%d_snap_f64_box_vel" % N, 1, N, 4, dims, "f64", pts[None], T[None], rho=10.0,
                    samples=8, box_lo=lo[None], box_hi=hi[None], vmax=3.0, eps=1e-6)


def config3(seed: int = 1003, N: int = 1000, dtype: str = "f64", rho: float = 1.0) -> Workload:
    """N=1000, 3D, minimum jerk, uniform T=1 s, no constraints, 1000 sweeps (fp64 and fp32)."""
    rng = np.random.default_rng(seed)
    dims = 3
    pts, _ = _random_walk(rng, N, dims, 0.5, 2.0)
    T = np.ones(N)
    return Workload("cfg3_N%d_jerk_%s_uniformT" % (N, dtype), 1, N, 3, dims, dtype, pts[None], T[None],
                    rho=rho, sweeps=1000)


def config4(seed: int = 1004, N: int = 10000, time_stretch: float = 1.0) -> Workload:
    """N=10000, 3D, minimum snap, fp64, T=step/U[1,3], box h~U[0.5,2], ||v||<=3, ||a||<=5, rho=10.

    time_stretch (kappa) > 1 gives the flagged feasible variant "4f"
    (the literal config is infeasible for generic seeds).
    """
    rng = np.random.default_rng(seed)
    dims = 3
    pts, steps = _random_walk(rng, N, dims, 1.0, 5.0)
    speed = rng.uniform(1.0, 3.0, size=N)
    T = steps / speed * float(time_stretch)
    h = rng.uniform(0.5, 2.0, size=N)
    lo, hi = _chord_box(pts, h)
    name = "cfg4_N%d_snap_f64_box_vel_acc" % N
    if time_stretch != 1.0:
        name += "_kappa%g" % time_stretch
    return Workload(name, 1, N, 4, dims, "f64", pts[None], T[None], rho=10.0,
                    samples=8, box_lo=lo[None], box_hi=hi[None], vmax=3.0, amax=5.0, eps=1e-4,
                    notes={"time_stretch": time_stretch})


def config5(seed0: int = 5000, batch: int = 256, N: int = 512, dtype: str = "f32") -> Workload:
    """256 independent trajectories x N=512, minimum snap, fp32, box h=1.5 + ||v||<=3, 500 sweeps."""
    dims = 3
    P = np.zeros((batch, N + 1, dims))
    T = np.zeros((batch, N))
    LO = np.zeros((batch, N, dims))
    HI = np.zeros((batch, N, dims))
    for b in range(batch):
        rng = np.random.default_rng(seed0 + b)
        pts, steps = _random_walk(rng, N, dims, 1.0, 5.0)
        P[b], T[b] = pts, steps / 2.0
        LO[b], HI[b] = _chord_box(pts, 1.5)
    return Workload("cfg5_B%d_N%d_snap_%s_box_vel" % (batch, N, dtype), batch, N, 4, dims, dtype, P, T,
                    rho=10.0, samples=8, box_lo=LO, box_hi=HI, vmax=3.0, sweeps=500)


def small_constrained(seed: int = 7, N: int = 37, s: int = 4, acc: bool = True, batch: int = 1,
                      dims: int = 3) -> Workload:
    """A ragged-size constrained case for parity tests (not one of the five configs)."""
    P = np.zeros((batch, N + 1, dims))
    T = np.zeros((batch, N))
    LO = np.zeros((batch, N, dims))
    HI = np.zeros((batch, N, dims))
    for b in range(batch):
        rng = np.random.default_rng(seed + 1000 * b)
        pts, steps = _random_walk(rng, N, dims, 1.0, 5.0)
        speed = rng.uniform(1.0, 3.0, size=N)
        h = rng.uniform(0.5, 2.0, size=N)
        P[b], T[b] = pts, steps / speed
        LO[b], HI[b] = _chord_box(pts, h)
    return Workload("small_N%d_s%d" % (N, s), batch, N, s, dims, "f64", P, T, rho=10.0, samples=8,
                    box_lo=LO, box_hi=HI, vmax=3.0, amax=5.0 if acc else 0.0)


def polytope_corridor(w: Workload, K: int = 8, seed: int = 3, margin=(0.3, 1.5)) -> Workload:
    """Replace the box corridor of `w` by K oblique half-spaces per segment (a convex cell around the chord, as the cells
    of a FIRI flight corridor are): random unit normals, offset = the larger of a'p over the segment's two
    waypoints + a margin.  Holds no method arithmetic: only draws the sets."""
    rng = np.random.default_rng(seed)
    pl = np.zeros((w.batch, w.N, K, w.dims + 1))
    for b in range(w.batch):
        for i in range(w.N):
            a = rng.standard_normal((K, w.dims))
            a /= np.sqrt((a * a).sum(axis=1, keepdims=True))
            p0, p1 = w.waypoints[b, i], w.waypoints[b, i + 1]
            pl[b, i, :, :w.dims] = a
            pl[b, i, :, w.dims] = np.maximum(a @ p0, a @ p1) + rng.uniform(margin[0], margin[1], size=K)
    w.planes, w.box_lo, w.box_hi = pl, None, None
    w.name += "_poly%d" % K
    return w


def fig5_curve(theta: np.ndarray) -> np.ndarray:
    """The reference curve of the Fig. 5 stand-in: a closed-form 3-D Lissajous figure (metres), theta in [0, 2 pi].
    The paper does not name its curve; any smooth parameterised curve has the workload's shape."""
    theta = np.asarray(theta, dtype=np.float64)
    return np.stack([10.0 * np.sin(2.0 * theta), 8.0 * np.sin(3.0 * theta + 0.5), 3.0 * np.cos(5.0 * theta)], axis=-1)


def fig5(N: int = 1024, s: int = 3, rho: float = 10.0, speed: float = 2.0) -> Workload:
    """PAPER.md:L355-361 (Fig. 5): N+1 points sampled uniformly in the parameter of a curve, the trajectory is forced
    through them (HARD waypoints), no inequality constraints; durations = chord length / `speed`."""
    theta = np.linspace(0.0, 2.0 * np.pi, N + 1)
    pts = fig5_curve(theta)
    chord = np.sqrt(((pts[1:] - pts[:-1]) ** 2).sum(axis=1))
    T = np.maximum(chord / speed, 1e-3)
    return Workload("fig5_N%d_s%d" % (N, s), 1, N, s, 3, "f64", pts[None], T[None], rho=rho,
                    notes={"theta": theta})


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}
