"""B200-native Splotch per-frame particle rendering path (arxiv 1309.1114).

`paper_1309_1114_b200.workloads` holds the seeded input generators (no CUDA needed);
`paper_1309_1114_b200.binding` is the thin ctypes layer over the C-ABI library
(include/splotch.h) and is imported lazily so that CPU-only tools can use the generators.
"""
__all__ = ["workloads", "binding"]
