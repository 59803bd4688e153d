"""B200-native CADMM segment sweep of TOP (arXiv 2507.10290).

`paper_2507_10290_b200.top`       thin ctypes binding over the C ABI in include/top.h
`paper_2507_10290_b200.workloads` seeded synthetic inputs (no method arithmetic)

Nothing here imports `oracle/`; the oracle is test infrastructure only.
The binding is imported lazily so that `workloads` stays usable without the
CUDA library being built.
"""

__all__ = ["top", "workloads"]
