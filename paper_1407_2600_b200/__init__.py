"""dsk — B200-native tree gravity: the 2HOT force path of arxiv 1407.2600.

`paper_1407_2600_b200.dsk` is the thin binding over the C-ABI library `libdsk.so` (include/dsk.h);
`paper_1407_2600_b200.workloads` holds the seeded synthetic input generators (no method arithmetic).
Nothing here imports the CPU oracle; there is no CPU fallback.
"""
__all__ = ["dsk", "workloads"]
