"""paper_2606_01009_b200 -- B200-native (sm_100a) MelT / MFCCT hot path (arxiv/paper_2606_01009).

``binding``   thin ctypes binding over the C-ABI library (include/melt.h); same names as the C calls.
``workloads`` seeded synthetic inputs shaped like BASELINE.json's configs (no method arithmetic).
``build``     in-tree nvcc build of csrc/ -> libmelt_b200.so.

Importing the package loads nothing heavy; the CUDA library is loaded on first use of ``binding`` and
raises if it is missing -- there is no CPU fallback.
"""
__all__ = ["binding", "workloads", "build"]
