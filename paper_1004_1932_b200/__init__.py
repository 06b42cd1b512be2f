"""B200-native hot path of arXiv 1004.1932 (active dumbbell suspensions).

`paper_1004_1932_b200.inputs`  seeded workload generators (numpy only, no method arithmetic)
`paper_1004_1932_b200.ds`      thin ctypes binding of the C-ABI in include/ds.h (argument
                               marshalling only; every step runs in the CUDA kernels of csrc/)

Nothing is imported eagerly: `inputs` must stay importable on a box without the CUDA library.
"""
__all__ = ["inputs", "ds"]
