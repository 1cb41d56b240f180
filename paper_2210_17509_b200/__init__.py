"""grx -- B200-native FP64 Valencia GRMHD right-hand side (GRaM-X, arxiv 2210.17509, hot path).

`paper_2210_17509_b200.grx`    thin ctypes binding of the C-ABI library (include/grx.h)
`paper_2210_17509_b200.inputs` seeded synthetic inputs (shared with the oracle's tests; no method arithmetic)
`paper_2210_17509_b200.build`  nvcc build of csrc/ -> libgrx.so (sm_100a)

Nothing is loaded at import time; `grx.lib()` raises if the CUDA library has not been built.
"""
__version__ = "0.1.0"
