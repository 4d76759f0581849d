"""paper_1503_01725_b200 — B200-native PSL source sampling + Monte Carlo dose (arxiv 1503.01725, hot path).

`binding` is the thin ctypes layer over libpslmc.so (C ABI in include/pslmc.h); `workloads` only
generates synthetic inputs; `build` compiles the library in-tree.  Nothing here falls back to a CPU.
"""
__all__ = ["binding", "workloads", "build"]
