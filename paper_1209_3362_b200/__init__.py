"""paper_1209_3362_b200 — B200 (sm_100a) hot path of the double-frame differential analysis of dynamic
near-field-scattering image stacks (arxiv 1209.3362): D(q,tau) and I(q) through a C-ABI CUDA library.

`binding` loads libnfs_b200.so (built in-tree by `build`).  Nothing here imports oracle/ or the input
generator (synth.py at the repo root, harness code).
"""
__all__ = ["binding", "build"]
