"""B200-native SPH interaction sweep of arxiv/paper_2511_11425 (pkdgrav3 SPH, paper I).

`paper_2511_11425_b200.sph`        thin ctypes binding of the C-ABI library (include/sph.h)
`paper_2511_11425_b200.workloads`  seeded synthetic inputs (numpy only; shared with the oracle)

Nothing is imported eagerly: `workloads` must stay importable without the CUDA library.
"""
__all__ = ["sph", "workloads"]
