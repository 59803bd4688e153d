"""top_operator_rows_static: the one entry point of the library that allocates nothing on the device.

Some users of this library cannot call cudaMalloc: a planner loaded as a plug-in into a process that reserved the whole
device heap at start-up, a re-planning loop with a hard period (the allocator may synchronise the device and has no
latency bound), a thread that runs beside another thread's CUDA-graph capture, a container with a fixed memory budget.
They own their buffers and nothing else, so they cannot create a solver (top_create takes one arena per solver).  For
them the operator kernel of top_create is reachable through top_operator_rows_static, whose working memory (Gram tables,
the device copy of the durations, a status word) is a static array inside libtop.so: at most
top.STATIC_MAX_SEGMENTS = 16384 segments per call.

The array is shared by every call and keeps the last call's contents, so the GPU test makes two calls in a row with
different sizes and inputs (and one after a call that failed on the device) and checks each against the existing path for
this quantity, top_precompute_operator -- the host twin of the same precompute, segment by segment, at the 1e-10 bar that
tests/test_host_logic.py uses for the operator.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the parity
tests.  It needs nothing from the tests before it and passes alone in a fresh process as well."""
import numpy as np
import pytest

from paper_2507_10290_b200 import top


def _twin_rows(T, s, rho, box, vel, acc, mode):
    """rho * Pm_hat [8, 8] from the host entry point top_precompute_operator (the existing path)."""
    Pm, _ = top.precompute_operator(s, float(T), rho, np.zeros(3), np.ones(3), box=box, vel=vel, acc=acc, mode=mode)
    return rho * Pm


def _check_against_twin(rows, T, s, rho, box, vel, acc, mode, segments):
    """rows [8 (b), nseg, 8 (a)] from the device; compares the listed segments, scaled as tests/test_host_logic.py does."""
    n = 2 * s
    lo = 1 if mode == "hard" else 0       # HARD: row / column 0 is zero (c^_0 is fixed)
    worst = 0.0
    for g in segments:
        got = rows[:, g, :].T             # [a][b]
        ref = _twin_rows(T[g], s, rho, box, vel, acc, mode)
        assert np.all(got[n:] == 0) and np.all(got[:, n:] == 0), g            # zero padding written, no NaN left
        assert np.abs(got - got.T).max() <= 1e-15 * np.abs(got).max(), g        # the kernel symmetrises
        if lo:
            assert np.abs(got[0]).max() <= 1e-12 * np.abs(ref).max() and np.abs(got[:, 0]).max() <= 1e-12 * np.abs(ref).max(), g
        sc = np.sqrt(np.abs(np.diag(ref)))[lo:n]
        err = np.abs((got[lo:n, lo:n] - ref[lo:n, lo:n]) / (sc[:, None] * sc[None, :])).max()
        worst = max(worst, err)
        assert err < 1e-10, (g, T[g], err)
    return worst


def test_static_entry_rejects_sizes_beyond_its_scratch():
    """More segments than the static array holds: a clear TOP_E_UNSUPPORTED, decided before any device work."""
    T = np.ones(top.STATIC_MAX_SEGMENTS + 1)
    with pytest.raises(top.TopError) as ei:
        top.operator_rows_static(T, 4, 10.0, rows_out_ptr=8)      # the pointer is never looked at
    assert ei.value.status == top.TOP_E_UNSUPPORTED
    assert "TOP_STATIC_MAX_SEGMENTS" in str(ei.value) and str(top.STATIC_MAX_SEGMENTS) in str(ei.value)
    for bad in (dict(s=5), dict(rho=0.0), dict(rho=float("nan"))):
        kw = dict(s=4, rho=1.0)
        kw.update(bad)
        with pytest.raises(top.TopError) as ei:
            top.operator_rows_static(np.ones(3), kw["s"], kw["rho"], rows_out_ptr=8)
        assert ei.value.status == top.TOP_E_INVALID
    with pytest.raises(top.TopError) as ei:
        top.operator_rows_static(np.array([1.0, -2.0]), 3, 1.0, rows_out_ptr=8)
    assert ei.value.status == top.TOP_E_INVALID


@pytest.mark.gpu
def test_static_entry_matches_existing_path_on_two_calls_in_a_row():
    import torch
    rng = np.random.default_rng(20250710)
    stream = torch.cuda.current_stream().cuda_stream

    def run(nseg, s, rho, box, vel, acc, mode, segments=None):
        T = rng.uniform(0.3, 4.0, size=nseg)
        out = torch.full((8, nseg, 8), float("nan"), dtype=torch.float64, device="cuda")   # the caller's buffer
        top.operator_rows_static(T, s, rho, out.data_ptr(), box=box, vel=vel, acc=acc, mode=mode, stream=stream)
        rows = out.cpu().numpy()
        assert np.isfinite(rows).all()
        return _check_against_twin(rows, T, s, rho, box, vel, acc, mode, range(nseg) if segments is None else segments)

    # two calls in a row: the second is shorter and has other durations, order, constraint blocks and mode, so anything
    # the first call left in the shared array (durations, tables of the other order, status) would show
    run(300, 4, 10.0, True, True, True, "hard")
    run(77, 3, 0.5, False, True, False, "pinned_z")
    run(1, 4, 300.0, True, False, False, "free")

    # a call that fails ON THE DEVICE (durations so small that the operator overflows) sets the status word;
    # the next call must start from a cleared one
    out = torch.zeros((8, 4, 8), dtype=torch.float64, device="cuda")
    with pytest.raises(top.TopError) as ei:
        top.operator_rows_static(np.full(4, 1e-60), 4, 1.0, out.data_ptr(), stream=stream)
    assert ei.value.status == top.TOP_E_INVALID and "positive definite" in str(ei.value)
    run(50, 4, 1.0, True, True, False, "hard")

    # the largest size the array holds (sampled segments, both ends included), then a small one again
    nmax = top.STATIC_MAX_SEGMENTS
    run(nmax, 4, 10.0, True, True, True, "hard", segments=[0, 1, 63, 64, 4097, nmax - 2, nmax - 1] + list(rng.integers(0, nmax, 25)))
    run(9, 3, 10.0, False, False, False, "hard")

    # a host pointer in place of the device buffer is refused, not written through
    host = np.zeros(64 * 3)
    with pytest.raises(top.TopError) as ei:
        top.operator_rows_static(np.ones(3), 4, 1.0, host.ctypes.data, stream=stream)
    assert ei.value.status == top.TOP_E_INVALID
