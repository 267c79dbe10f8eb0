"""B200-native batched TB-SMA (Au) force / MD hot path of arXiv:1311.3890.

`paper_1311_3890_b200.binding` is the thin ctypes layer over the C-ABI library
(include/tbsma.h, csrc/); it fails loudly if the CUDA library is not built.
`paper_1311_3890_b200.workloads` builds the seeded synthetic inputs (numpy only).
Nothing here imports the CPU oracle.
"""
__all__ = ["binding", "workloads"]
