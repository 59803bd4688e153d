"""Thin ctypes binding over the C ABI of include/top.h (argument marshalling only).

Every step of the CADMM sweep runs inside libtop.so's CUDA kernels; this module holds none of the method's
arithmetic and never imports oracle/.  It fails loudly when the library is missing (there is no CPU path).
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtop.so")

TOP_OK, TOP_NOT_CONVERGED = 0, 1
TOP_E_INVALID, TOP_E_NOMEM, TOP_E_CUDA, TOP_E_UNSUPPORTED, TOP_E_NONFINITE = -1, -2, -3, -4, -5
TOP_F64, TOP_F32 = 0, 1
WAYPOINT = {"hard": 0, "pinned_z": 1, "free": 2}
TOP_RD_NORMALISED = 4
TOP_EPS_N_SCALED = 8
TOP_RHO_ADAPTIVE = 64
TOP_KERNEL_NO_MMA = 128
TOP_CONSENSUS_WIDE = 256
TOP_XUPDATE_NUMERIC = 512
SYNC = {"auto": 0, "grid": 16, "neighbour": 32, "pairwise": 48}

EXPORTS = ["top_create", "top_reset", "top_iterate", "top_solve", "top_get_residuals", "top_get_coeffs", "top_get_state",
           "top_snapshot_bytes", "top_snapshot_save", "top_snapshot_restore", "top_iteration", "top_numeric_info", "top_set_rho", "top_get_rho", "top_launch_info", "top_memory_info", "top_capacity", "top_fma_peak", "top_precompute_operator",
           "top_operator_rows_static",
           "top_destroy", "top_last_error"]


class TopError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__("top status %d: %s" % (status, message))
        self.status = status


class _Constraints(ctypes.Structure):
    _fields_ = [("samples", ctypes.c_int32), ("box_lo", ctypes.POINTER(ctypes.c_double)),
                ("box_hi", ctypes.POINTER(ctypes.c_double)), ("vmax", ctypes.c_double), ("amax", ctypes.c_double),
                ("num_planes", ctypes.c_int32), ("planes", ctypes.POINTER(ctypes.c_double))]


class _Options(ctypes.Structure):
    _fields_ = [("struct_size", ctypes.c_uint32), ("flags", ctypes.c_uint32), ("check_every", ctypes.c_int32),
                ("device", ctypes.c_int32), ("max_iter", ctypes.c_int64), ("cuda_stream", ctypes.c_void_p),
                ("segs_per_cta", ctypes.c_int32), ("lanes_per_segment", ctypes.c_int32), ("adapt_mu", ctypes.c_double),
                ("adapt_tau_incr", ctypes.c_double), ("adapt_tau_decr", ctypes.c_double)]


_lib = None


def lib():
    """Load libtop.so (built by `python -m paper_2507_10290_b200.build`).  No fallback of any kind."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("libtop.so is missing: run `python -m paper_2507_10290_b200.build` "
                          "(the CADMM sweep has no CPU path)")
    L = ctypes.CDLL(LIB_PATH)
    dp = ctypes.POINTER(ctypes.c_double)
    vp = ctypes.c_void_p
    i32p = ctypes.POINTER(ctypes.c_int32)
    L.top_create.restype = ctypes.c_int
    L.top_create.argtypes = [ctypes.POINTER(vp), ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32,
                             ctypes.c_int, dp, dp, dp, dp, ctypes.POINTER(_Constraints), ctypes.c_double,
                             ctypes.POINTER(_Options)]
    L.top_reset.restype = ctypes.c_int
    L.top_reset.argtypes = [vp, dp, dp, dp, dp, ctypes.POINTER(_Constraints), ctypes.c_double]
    L.top_iterate.restype = ctypes.c_int
    L.top_iterate.argtypes = [vp, ctypes.c_int64]
    L.top_solve.restype = ctypes.c_int
    L.top_solve.argtypes = [vp, ctypes.c_double, ctypes.POINTER(ctypes.c_int64)]
    L.top_get_residuals.restype = ctypes.c_int
    L.top_get_residuals.argtypes = [vp, dp, dp, dp, dp]
    L.top_get_coeffs.restype = ctypes.c_int
    L.top_get_coeffs.argtypes = [vp, vp, ctypes.c_int32]
    L.top_get_state.restype = ctypes.c_int
    L.top_get_state.argtypes = [vp, ctypes.c_char_p, dp, ctypes.c_size_t]
    L.top_set_rho.restype = ctypes.c_int
    L.top_set_rho.argtypes = [vp, ctypes.c_double]
    L.top_get_rho.restype = ctypes.c_double
    L.top_get_rho.argtypes = [vp]
    L.top_snapshot_bytes.restype = ctypes.c_size_t
    L.top_snapshot_bytes.argtypes = [vp]
    L.top_snapshot_save.restype = ctypes.c_int
    L.top_snapshot_save.argtypes = [vp, vp, ctypes.c_size_t]
    L.top_snapshot_restore.restype = ctypes.c_int
    L.top_snapshot_restore.argtypes = [vp, vp, ctypes.c_size_t]
    L.top_numeric_info.restype = ctypes.c_int
    L.top_numeric_info.argtypes = [vp, ctypes.POINTER(ctypes.c_int64)]
    L.top_iteration.restype = ctypes.c_int64
    L.top_iteration.argtypes = [vp]
    L.top_launch_info.restype = ctypes.c_int
    L.top_launch_info.argtypes = [vp, i32p, i32p, i32p, i32p, i32p, ctypes.POINTER(ctypes.c_int64)]
    L.top_memory_info.restype = ctypes.c_int
    L.top_memory_info.argtypes = [vp, ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_int64)]
    L.top_capacity.restype = ctypes.c_int64
    L.top_capacity.argtypes = [ctypes.c_int32, ctypes.c_int32, ctypes.c_int, ctypes.c_int32]
    L.top_fma_peak.restype = ctypes.c_double
    L.top_fma_peak.argtypes = [ctypes.c_int32, ctypes.c_int, ctypes.c_int32, vp]
    L.top_precompute_operator.restype = ctypes.c_int
    L.top_precompute_operator.argtypes = [ctypes.c_int32, ctypes.c_double, ctypes.c_double, ctypes.c_int32,
                                          ctypes.c_int32, ctypes.c_int32, ctypes.c_uint32, dp, dp, dp, dp]
    L.top_operator_rows_static.restype = ctypes.c_int
    L.top_operator_rows_static.argtypes = [ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, dp, ctypes.c_double, ctypes.c_int32,
                                           ctypes.c_int32, ctypes.c_int32, ctypes.c_uint32, vp, vp]
    L.top_destroy.restype = ctypes.c_int
    L.top_destroy.argtypes = [vp]
    L.top_last_error.restype = ctypes.c_char_p
    L.top_last_error.argtypes = [vp]
    _lib = L
    return L


def _dptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _f64(a, shape=None):
    if a is None:
        return None
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None and a.shape != shape:
        raise ValueError("expected shape %s, got %s" % (shape, a.shape))
    return a


def precompute_operator(s, T, rho, p0, p1, box=False, vel=False, acc=False, mode="hard"):
    """top_precompute_operator: (Pm_hat [8,8], c0_hat [8,3]) of one segment; host only, launches nothing."""
    L = lib()
    Pm, c0 = np.zeros((8, 8)), np.zeros((8, 3))
    a, b = _f64(p0, (3,)), _f64(p1, (3,))
    st = L.top_precompute_operator(int(s), float(T), float(rho), int(box), int(vel), int(acc), WAYPOINT[mode],
                                   _dptr(a), _dptr(b), _dptr(Pm), _dptr(c0))
    if st != TOP_OK:
        raise TopError(st, L.top_last_error(None).decode())
    return Pm, c0


STATIC_MAX_SEGMENTS = 16384


def operator_rows_static(durations, s, rho, rows_out_ptr: int, box=False, vel=False, acc=False, mode="hard", device=-1,
                         stream=0):
    """top_operator_rows_static: rho * Pm_hat of every segment, written by the GPU into a device buffer the caller already
    owns, for callers that must not allocate device memory (a plug-in in a process that reserved the whole heap, a
    fixed-rate re-planning loop, a thread beside a CUDA-graph capture).  The kernel's scratch is a static array inside the
    library, so at most STATIC_MAX_SEGMENTS segments per call; calls on one device are serialised and the call waits
    for the stream.  Make the first call on a device at start-up, outside any stream capture.

    durations: host array [nseg]; rows_out_ptr: raw device pointer to 64 * nseg doubles, laid out [8 (b)][nseg][8 (a)]
    (e.g. torch.empty((8, nseg, 8), dtype=torch.float64, device="cuda").data_ptr()).  Nothing is returned: the result is
    in the caller's buffer."""
    L = lib()
    T = _f64(np.asarray(durations).reshape(-1))
    st = L.top_operator_rows_static(int(device), int(T.size), int(s), _dptr(T), float(rho), int(box), int(vel), int(acc),
                                    WAYPOINT[mode], ctypes.c_void_p(rows_out_ptr), ctypes.c_void_p(stream))
    if st != TOP_OK:
        raise TopError(st, L.top_last_error(None).decode())


def capacity(s, dtype="f64", constrained=True, device=-1):
    return int(lib().top_capacity(int(device), int(s), TOP_F64 if dtype == "f64" else TOP_F32, int(constrained)))


def fma_peak(dtype="f64", reps=5, device=-1, stream=0):
    """Measured plain-ALU FMA peak in FLOP/s (top_fma_peak)."""
    v = float(lib().top_fma_peak(int(device), TOP_F64 if dtype == "f64" else TOP_F32, int(reps), ctypes.c_void_p(stream)))
    if v < 0:
        raise TopError(TOP_E_CUDA, "top_fma_peak failed")
    return v


class TopSolver:
    """top_create / top_iterate / top_solve / top_get_* for a batch of trajectories.

    waypoints [batch, N+1, dims] (or [N+1, dims]), durations [batch, N] (or [N]); constraint arrays as in
    include/top.h.  `stream` is a raw cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream).
    """

    def __init__(self, waypoints, durations, s, rho, dtype="f64", samples=0, box_lo=None, box_hi=None, vmax=0.0,
                 amax=0.0, start_derivs=None, end_derivs=None, mode="hard", rd_normalised=False, eps_n_scaled=False,
                 sync="auto", check_every=0, max_iter=0, device=-1, stream=0, segs_per_cta=0, lanes=0, adaptive_rho=False,
                 adapt_mu=0.0, adapt_tau_incr=0.0, adapt_tau_decr=0.0, no_mma=False, planes=None, consensus="s", numeric=False):
        L = lib()
        wp = np.asarray(waypoints, dtype=np.float64)
        T = np.asarray(durations, dtype=np.float64)
        if wp.ndim == 2:
            wp, T = wp[None], T[None]
            box_lo = None if box_lo is None else np.asarray(box_lo)[None]
            box_hi = None if box_hi is None else np.asarray(box_hi)[None]
            start_derivs = None if start_derivs is None else np.asarray(start_derivs)[None]
            end_derivs = None if end_derivs is None else np.asarray(end_derivs)[None]
            planes = None if planes is None else np.asarray(planes)[None]
        if wp.ndim != 3 or T.ndim != 2 or wp.shape[0] != T.shape[0] or wp.shape[1] != T.shape[1] + 1:
            raise ValueError("waypoints [batch,N+1,dims] and durations [batch,N] do not match")
        wp, T = _f64(wp), _f64(T)
        self.batch, self.N, self.dims = T.shape[0], T.shape[1], wp.shape[2]
        self.s, self.n, self.dtype = int(s), 2 * int(s), dtype
        self.Ms = int(samples)
        self.nc = {"s": self.s, "wide": 2 * self.s - 1}[consensus]     # consensus derivative orders per boundary
        self.durations = T
        lo = _f64(box_lo, (self.batch, self.N, self.dims))
        hi = _f64(box_hi, (self.batch, self.N, self.dims))
        sd = _f64(start_derivs, (self.batch, self.s - 1, self.dims))
        ed = _f64(end_derivs, (self.batch, self.s - 1, self.dims))
        cons = None
        pl = None if planes is None else _f64(planes)
        if pl is not None and (pl.ndim != 4 or pl.shape[:2] != (self.batch, self.N) or pl.shape[3] != self.dims + 1):
            raise ValueError("planes must be [batch, N, K, dims+1]")
        self.K = 0 if pl is None else pl.shape[2]
        if samples:
            cons = _Constraints(int(samples), _dptr(lo), _dptr(hi), float(vmax), float(amax), self.K, _dptr(pl))
        flags = WAYPOINT[mode] | (TOP_RD_NORMALISED if rd_normalised else 0) | \
            (TOP_EPS_N_SCALED if eps_n_scaled else 0) | SYNC[sync] | (TOP_RHO_ADAPTIVE if adaptive_rho else 0) | \
            (TOP_KERNEL_NO_MMA if no_mma else 0) | (TOP_CONSENSUS_WIDE if consensus == "wide" else 0) | \
            (TOP_XUPDATE_NUMERIC if numeric else 0)
        opt = _Options(ctypes.sizeof(_Options), flags, int(check_every), int(device), int(max_iter),
                       ctypes.c_void_p(stream), int(segs_per_cta), int(lanes), float(adapt_mu), float(adapt_tau_incr),
                       float(adapt_tau_decr))
        self._L = L
        self._h = ctypes.c_void_p()
        st = L.top_create(ctypes.byref(self._h), self.batch, self.N, self.s, self.dims,
                          TOP_F64 if dtype == "f64" else TOP_F32, _dptr(wp), _dptr(T), _dptr(sd), _dptr(ed),
                          ctypes.byref(cons) if cons is not None else None, float(rho), ctypes.byref(opt))
        if st != TOP_OK:
            self._h = ctypes.c_void_p()
            raise TopError(st, L.top_last_error(None).decode())

    def _check(self, st, ok=(TOP_OK,)):
        if st not in ok:
            raise TopError(st, self._L.top_last_error(self._h).decode())
        return st

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._L.top_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def reset(self, waypoints, durations, rho, box_lo=None, box_hi=None, vmax=0.0, amax=0.0, start_derivs=None,
              end_derivs=None, planes=None):
        """top_reset: a new problem of the same shape on this handle (no allocation)."""
        wp = np.asarray(waypoints, dtype=np.float64)
        T = np.asarray(durations, dtype=np.float64)
        if wp.ndim == 2:
            wp, T = wp[None], T[None]
            box_lo = None if box_lo is None else np.asarray(box_lo)[None]
            box_hi = None if box_hi is None else np.asarray(box_hi)[None]
            start_derivs = None if start_derivs is None else np.asarray(start_derivs)[None]
            end_derivs = None if end_derivs is None else np.asarray(end_derivs)[None]
            planes = None if planes is None else np.asarray(planes)[None]
        pl = _f64(planes, (self.batch, self.N, self.K, self.dims + 1)) if planes is not None else None
        wp, T = _f64(wp, (self.batch, self.N + 1, self.dims)), _f64(T, (self.batch, self.N))
        lo = _f64(box_lo, (self.batch, self.N, self.dims)); hi = _f64(box_hi, (self.batch, self.N, self.dims))
        sd = _f64(start_derivs, (self.batch, self.s - 1, self.dims)); ed = _f64(end_derivs, (self.batch, self.s - 1, self.dims))
        cons = _Constraints(self.Ms, _dptr(lo), _dptr(hi), float(vmax), float(amax), 0 if pl is None else self.K, _dptr(pl)) if self.Ms else None
        self._check(self._L.top_reset(self._h, _dptr(wp), _dptr(T), _dptr(sd), _dptr(ed),
                                      ctypes.byref(cons) if cons is not None else None, float(rho)))
        self.durations = T

    def iterate(self, k: int):
        self._check(self._L.top_iterate(self._h, int(k)))

    def solve(self, eps: float):
        """Returns (converged: bool, iters[batch])."""
        it = np.zeros(self.batch, dtype=np.int64)
        st = self._check(self._L.top_solve(self._h, float(eps), it.ctypes.data_as(ctypes.POINTER(ctypes.c_int64))),
                         ok=(TOP_OK, TOP_NOT_CONVERGED))
        return st == TOP_OK, it

    def set_rho(self, rho: float):
        self._check(self._L.top_set_rho(self._h, float(rho)))

    @property
    def rho(self) -> float:
        return float(self._L.top_get_rho(self._h))

    def snapshot(self) -> np.ndarray:
        """Complete iterate as an opaque byte array (top_snapshot_save)."""
        buf = np.zeros(int(self._L.top_snapshot_bytes(self._h)), dtype=np.uint8)
        self._check(self._L.top_snapshot_save(self._h, buf.ctypes.data_as(ctypes.c_void_p), buf.size))
        return buf

    def restore(self, snap: np.ndarray):
        snap = np.ascontiguousarray(snap, dtype=np.uint8)
        self._check(self._L.top_snapshot_restore(self._h, snap.ctypes.data_as(ctypes.c_void_p), snap.size))

    def residuals(self):
        r = [np.zeros(self.batch) for _ in range(4)]
        self._check(self._L.top_get_residuals(self._h, *[_dptr(a) for a in r]))
        return {"r_p": r[0], "r_d": r[1], "r_d_norm": r[2], "r_p_gap": r[3]}

    def coeffs(self):
        """[batch, N, dims, 2s] in the paper's basis (Eq. 18), numpy array of the solver dtype."""
        out = np.zeros((self.batch, self.N, self.dims, self.n), dtype=np.float64 if self.dtype == "f64" else np.float32)
        self._check(self._L.top_get_coeffs(self._h, out.ctypes.data_as(ctypes.c_void_p), 0))
        return out

    def coeffs_to_device(self, device_ptr: int):
        """top_get_coeffs into a device buffer (no host synchronisation)."""
        self._check(self._L.top_get_coeffs(self._h, ctypes.c_void_p(device_ptr), 1))

    _STATE_SHAPES = {"z": lambda o: (o.batch, o.N + 1, o.nc, o.dims), "u": lambda o: (o.batch, o.N, 2 * o.nc, o.dims)}

    def state(self, field: str):
        if field in ("s_poly", "v_poly"):
            shape = (self.batch, self.N, 8, self.K)
        elif field in ("y_v", "y_a"):
            shape = (self.batch, self.N, 8)
        else:
            shape = self._STATE_SHAPES.get(field, lambda o: (o.batch, o.N, 8, o.dims))(self)
        out = np.zeros(shape)
        self._check(self._L.top_get_state(self._h, field.encode(), _dptr(out), out.size))
        return out

    def inner_iterations(self) -> int:
        """top_numeric_info: L-BFGS iterations so far (NumericSolve branch)."""
        v = ctypes.c_int64()
        self._check(self._L.top_numeric_info(self._h, ctypes.byref(v)))
        return v.value

    @property
    def iteration(self) -> int:
        return int(self._L.top_iteration(self._h))

    def launch_info(self):
        v = [ctypes.c_int32() for _ in range(5)]
        n = ctypes.c_int64()
        self._check(self._L.top_launch_info(self._h, *[ctypes.byref(x) for x in v], ctypes.byref(n)))
        keys = ["ctas", "threads", "segs_per_cta", "smem_bytes", "waves"]
        d = {k: x.value for k, x in zip(keys, v)}
        d["launches"] = n.value
        return d

    def memory_info(self):
        a, b = ctypes.c_int64(), ctypes.c_int64()
        self._check(self._L.top_memory_info(self._h, ctypes.byref(a), ctypes.byref(b)))
        return {"device_bytes": a.value, "h2d_bytes_per_problem": b.value}


def from_workload(w, b0: int = 0, b1: Optional[int] = None, **kw) -> TopSolver:
    """Build a solver for trajectories [b0, b1) of a workloads.Workload."""
    b1 = w.batch if b1 is None else b1
    sl = slice(b0, b1)
    return TopSolver(w.waypoints[sl], w.durations[sl], w.s, w.rho, dtype=kw.pop("dtype", w.dtype), samples=w.samples,
                     box_lo=None if w.box_lo is None else w.box_lo[sl],
                     box_hi=None if w.box_hi is None else w.box_hi[sl], vmax=w.vmax, amax=w.amax,
                     planes=None if getattr(w, "planes", None) is None else w.planes[sl], **kw)
