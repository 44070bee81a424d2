"""paper_2606_06641_b200 -- B200-native hot path of AFSAT (arxiv/paper_2606_06641).

`binding` is the thin ctypes layer over the C ABI (include/afsat.h) of the in-tree CUDA library
libafsat_b200.so; `instances` holds the seeded synthetic input generators; `build` compiles the
library with nvcc for sm_100a.  Nothing here falls back to the CPU.
"""
__all__ = ["binding", "instances", "build"]
