"""B200-native hydrostatic free-surface ocean time step (arXiv 2309.06662 hot path).

`paper_2309_06662_b200.workloads` : seeded synthetic inputs (numpy only, no method arithmetic)
`paper_2309_06662_b200.ocn`       : thin binding over the C-ABI CUDA library libocn.so
"""
__all__ = ["workloads", "ocn"]
