"""B200-native longitudinal tracking hot path of arxiv/paper_1610_05801.

``longtrack``  -- ctypes binding of the C-ABI library (include/longtrack.h); importing it
                  loads ``liblongtrack.so`` and fails loudly when that is missing.
``workloads``  -- seeded synthetic bunches / BASELINE.json configs (numpy only).
``build``      -- nvcc build of the library for sm_100a.
Nothing is imported eagerly so that ``workloads`` is usable without the CUDA library.
"""
__all__ = ["longtrack", "workloads", "build"]
