"""ctypes wrapper around oracle/top_oracle.c (the CPU oracle; TEST INFRASTRUCTURE ONLY).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
import this.  It never imports the product package.  The shared library is (re)built with gcc
on first use when missing or older than its source.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "top_oracle.c")
MODES = {"hard": 0, "pinned_z": 1, "free": 2}


def build(force: bool = False) -> None:
    """Compile libtop_oracle.so (fp64 sweep) and libtop_oracle_ld.so (long-double sweep)."""
    for lib, flags in (("libtop_oracle.so", []), ("libtop_oracle_ld.so", ["-DORACLE_LONG_DOUBLE"])):
        out = os.path.join(_HERE, lib)
        if not force and os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(_SRC):
            continue
        tmp = out + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fPIC", "-shared", "-fopenmp", *flags, "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, out)


_libs: dict = {}


def _lib(long_double: bool):
    key = bool(long_double)
    if key not in _libs:
        build()
        L = ctypes.CDLL(os.path.join(_HERE, "libtop_oracle_ld.so" if key else "libtop_oracle.so"))
        dp = ctypes.POINTER(ctypes.c_double)
        L.oracle_create.restype = ctypes.c_void_p
        L.oracle_create.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp, dp, dp, ctypes.c_int,
                                    dp, dp, ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_int]
        L.oracle_create_poly.restype = ctypes.c_void_p
        L.oracle_create_poly.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp, dp, dp, ctypes.c_int, ctypes.c_int, dp,
                                         ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_int]
        L.oracle_create_ex.restype = ctypes.c_void_p
        L.oracle_create_ex.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp, dp, dp, ctypes.c_int, dp, dp, ctypes.c_int, dp,
                                       ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_int]
        L.oracle_set_numeric.restype = ctypes.c_int
        L.oracle_set_numeric.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_double]
        L.oracle_inner_iters.restype = ctypes.c_int64
        L.oracle_inner_iters.argtypes = [ctypes.c_void_p]
        L.oracle_numeric_eval.restype = ctypes.c_double
        L.oracle_numeric_eval.argtypes = [ctypes.c_void_p, ctypes.c_int, dp, dp]
        L.oracle_destroy.argtypes = [ctypes.c_void_p]
        L.oracle_sweep.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_int]
        L.oracle_solve.restype = ctypes.c_int64
        L.oracle_solve.argtypes = [ctypes.c_void_p, ctypes.c_double, ctypes.c_int64, ctypes.c_int, ctypes.c_int]
        L.oracle_set_rho.restype = ctypes.c_int
        L.oracle_set_rho.argtypes = [ctypes.c_void_p, ctypes.c_double]
        L.oracle_rho.restype = ctypes.c_double
        L.oracle_rho.argtypes = [ctypes.c_void_p]
        L.oracle_solve_adaptive.restype = ctypes.c_int64
        L.oracle_solve_adaptive.argtypes = [ctypes.c_void_p, ctypes.c_double, ctypes.c_int64, ctypes.c_int, ctypes.c_double,
                                            ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_int]
        L.oracle_residuals.argtypes = [ctypes.c_void_p, dp]
        L.oracle_objective.restype = ctypes.c_double
        L.oracle_objective.argtypes = [ctypes.c_void_p]
        L.oracle_iter.restype = ctypes.c_int64
        L.oracle_iter.argtypes = [ctypes.c_void_p]
        L.oracle_get.restype = ctypes.c_int64
        L.oracle_get.argtypes = [ctypes.c_void_p, ctypes.c_char_p, dp]
        L.oracle_threads.restype = ctypes.c_int
        _libs[key] = L
    return _libs[key]


def _dptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


class Oracle:
    """One trajectory (the oracle has no batch dimension; loop over it)."""

    def __init__(self, waypoints, durations, s, rho, samples=0, box_lo=None, box_hi=None, vmax=0.0, amax=0.0,
                 start_derivs=None, end_derivs=None, mode="hard", long_double=False, planes=None, consensus="s",
                 numeric=False, lbfgs_memory=6, max_inner=50, inner_tol=1e-10):
        """consensus: "s" = derivative orders 0..s-1 at every boundary (default, reading A1); "wide" = the paper-literal
        orders 0..2s-2, the orders >= s left out at the two trajectory ends."""
        wp = np.ascontiguousarray(waypoints, dtype=np.float64)
        T = np.ascontiguousarray(durations, dtype=np.float64)
        assert wp.ndim == 2 and T.ndim == 1 and wp.shape[0] == T.shape[0] + 1
        self.N, self.m, self.s, self.n, self.Ms = T.shape[0], wp.shape[1], int(s), 2 * int(s), int(samples)
        self.nc = {"s": int(s), "wide": 2 * int(s) - 1}[consensus]
        self.T = T
        keep = [wp, T]
        def opt(a, shape):
            if a is None:
                return None
            a = np.ascontiguousarray(a, dtype=np.float64)
            assert a.shape == shape, (a.shape, shape)
            keep.append(a)
            return a
        lo = opt(box_lo, (self.N, self.m)); hi = opt(box_hi, (self.N, self.m))
        sd = opt(start_derivs, (self.s - 1, self.m)); ed = opt(end_derivs, (self.s - 1, self.m))
        self._L = _lib(long_double)
        self.K = 0
        pl = None
        if planes is not None:            # general polytope corridor: [N][K][m+1] = (normal, offset), normal'p <= offset
            pl = np.ascontiguousarray(planes, dtype=np.float64)
            assert pl.ndim == 3 and pl.shape[0] == self.N and pl.shape[2] == self.m + 1 and lo is None and hi is None
            keep.append(pl)
            self.K = pl.shape[1]
        self._h = self._L.oracle_create_ex(self.N, self.s, self.m, _dptr(wp), _dptr(T), _dptr(sd), _dptr(ed), self.Ms,
                                           _dptr(lo), _dptr(hi), self.K, _dptr(pl), float(vmax), float(amax), float(rho),
                                           MODES[mode], self.nc)
        if not self._h:
            raise ValueError("oracle_create rejected the inputs")
        if numeric:       # NumericSolve branch (reading A20): L-BFGS x-update for the ball sets
            if self._L.oracle_set_numeric(self._h, int(lbfgs_memory), int(max_inner), float(inner_tol)) != 0:
                raise ValueError("oracle_set_numeric rejected the inputs")

    def __del__(self):
        if getattr(self, "_h", None):
            self._L.oracle_destroy(self._h)
            self._h = None

    def sweep(self, k=1, threads=1):
        self._L.oracle_sweep(self._h, int(k), int(threads))

    def solve(self, eps, max_iter, use_rd_norm=False, threads=1):
        return int(self._L.oracle_solve(self._h, float(eps), int(max_iter), int(use_rd_norm), int(threads)))

    def set_rho(self, rho):
        if self._L.oracle_set_rho(self._h, float(rho)) != 0:
            raise ValueError("oracle_set_rho failed")

    @property
    def rho(self):
        return float(self._L.oracle_rho(self._h))

    def solve_adaptive(self, eps, max_iter, mu=10.0, tau_incr=1.1, tau_decr=1.1, every=1, use_rd_norm=False, threads=1):
        return int(self._L.oracle_solve_adaptive(self._h, float(eps), int(max_iter), int(use_rd_norm), float(mu),
                                                 float(tau_incr), float(tau_decr), int(every), int(threads)))

    @property
    def inner_iters(self):
        return int(self._L.oracle_inner_iters(self._h))

    def numeric_eval(self, i, c, want_grad=True):
        """F (A20) and its gradient for segment i at coefficients c [n][m], with the solver's current z, u, s, v, w."""
        c = np.ascontiguousarray(c, dtype=np.float64)
        g = np.zeros_like(c) if want_grad else None
        F = float(self._L.oracle_numeric_eval(self._h, int(i), _dptr(c), _dptr(g)))
        return (F, g) if want_grad else F

    def residuals(self):
        out = np.zeros(4)
        self._L.oracle_residuals(self._h, _dptr(out))
        return {"r_p": out[0], "r_d": out[1], "r_d_norm": out[2], "r_p_gap": out[3]}

    def objective(self):
        return float(self._L.oracle_objective(self._h))

    @property
    def iter(self):
        return int(self._L.oracle_iter(self._h))

    def max_threads(self):
        return int(self._L.oracle_threads())

    _SHAPES = {
        "coeffs": lambda o: (o.N, o.m, o.n), "C": lambda o: (o.N, o.n, o.m), "z": lambda o: (o.N + 1, o.nc, o.m),
        "u": lambda o: (o.N, 2 * o.nc, o.m), "rowmask": lambda o: (o.N, 2 * o.nc), "Pm": lambda o: (o.N, o.n, o.n), "c0": lambda o: (o.N, o.n, o.m),
        "Q": lambda o: (o.N, o.n, o.n), "M": lambda o: (o.N, 2 * o.nc, o.n),
        "E0": lambda o: (o.N, o.Ms, o.n), "E1": lambda o: (o.N, o.Ms, o.n), "E2": lambda o: (o.N, o.Ms, o.n),
        "y_v": lambda o: (o.N, o.Ms), "y_a": lambda o: (o.N, o.Ms), "s_poly": lambda o: (o.N, o.Ms, o.K), "v_poly": lambda o: (o.N, o.Ms, o.K),
    }

    def get(self, name):
        shape = self._SHAPES.get(name, lambda o: (o.N, o.Ms, o.m))(self)
        out = np.zeros(shape)
        cnt = self._L.oracle_get(self._h, name.encode(), _dptr(out))
        if cnt != out.size:
            raise KeyError(name)
        return out


def eval_poly(coeffs, T, order, taus):
    """Evaluate derivative `order` of every segment at normalised times taus in [0,1].

    coeffs [N][m][n] in the paper's basis (Eq. 18: ascending powers of t - t_{i-1}, seconds).
    Returns [N][len(taus)][m].  Plain definition; used by tests on both oracle and GPU output.
    """
    coeffs = np.asarray(coeffs, dtype=np.float64)
    N, m, n = coeffs.shape
    taus = np.asarray(taus, dtype=np.float64)
    out = np.zeros((N, taus.size, m))
    for j in range(order, n):
        f = 1.0
        for q in range(order):
            f *= (j - q)
        t = taus[None, :] * np.asarray(T)[:, None]
        out += f * (t ** (j - order))[:, :, None] * coeffs[:, None, :, j]
    return out
