"""dh — B200-native (sm_100a) Euler finite-volume step and its adjoint (arxiv/paper_2512_13403 hot path).

`from paper_2512_13403_b200 import dh` gives the thin ctypes binding over the C-ABI library
(`include/dh.h`); `workloads` holds the seeded synthetic input generators.  Importing this package
does not load CUDA; `dh.load()` does, and fails loudly if `libdh.so` cannot be built or loaded.
"""
__all__ = ["dh", "workloads", "build"]
