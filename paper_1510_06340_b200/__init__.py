"""B200-native MUSTA-FORCE relativistic hydrodynamics step (arXiv 1510.06340), hand-written CUDA for sm_100a.

`paper_1510_06340_b200.binding` is the thin ctypes layer over the C-ABI library (include/mustaforce.h);
`paper_1510_06340_b200.workloads` holds the seeded synthetic input generators;
`paper_1510_06340_b200.build` compiles csrc/ with nvcc.  Nothing is loaded at import time.
"""
__all__ = ["binding", "workloads", "build"]
