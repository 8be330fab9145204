"""lgx — B200-native mass evaluation of biomass-logistics plans (arxiv 1909.10286 hot path).

`paper_1909_10286_b200.binding` is the thin ctypes binding of the C-ABI library
(include/lgx.h); `workloads` holds the seeded synthetic instance generators;
`sharding` the multi-GPU id split.  Importing this package loads nothing native.
"""
__all__ = ["binding", "workloads", "sharding", "build"]
