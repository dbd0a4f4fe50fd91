"""B200-native short-range molecular-dynamics hot path (arXiv 1009.4330).

Sub-modules:
  workloads  seeded synthetic input generators (numpy only; no method arithmetic)
  md         thin ctypes binding over the C-ABI library ``libmd_b200.so``
  build      nvcc build helper for the library
  dist       rank bookkeeping for ``bench.py`` (independent replicas)

Nothing is imported eagerly: ``workloads`` must stay importable on a machine with
no CUDA library, and ``md`` must fail loudly when the library is missing.
"""

__all__ = ["workloads", "md", "build", "dist"]
