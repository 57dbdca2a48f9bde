"""B200-native longitudinal tracking hot path of arxiv/paper_1610_05801.

``longtrack``  -- ctypes binding of the C-ABI library (include/longtrack.h); importing it
                  loads ``liblongtrack.so`` and fails loudly when that is missing.
``probe``      -- ctypes binding of ``liblongtrack_probe.so`` (include/longtrack_probe.h): the FP64-pipe
                  probes bench.py uses; measurement tooling, not part of the product ABI.
``workloads``  -- seeded synthetic bunches / BASELINE.json configs (numpy only).
``build``      -- nvcc build of the library for sm_100a.
Nothing is imported eagerly so that ``workloads`` is usable without the CUDA library.
"""
__all__ = ["longtrack", "probe", "workloads", "build"]
