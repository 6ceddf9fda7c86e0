"""B200-native matrix-free Poisson solvers for self-gravity (arxiv/paper_2605_03563 hot path).

`binding` holds the thin ctypes layer over the C-ABI library (include/poisson.h); `workloads` the seeded inputs.
"""
