"""GPUSparse hot path (arxiv/paper_2606_26441), B200-native: exact batched top-k sparse scoring.

Sub-modules:
  workload  seeded synthetic inputs (shared with the oracle; no method arithmetic)
  binding   thin ctypes binding over the C-ABI library ``libgpusparse.so`` (include/gpusparse.h)
  build     nvcc/gcc build steps
Importing this package loads nothing native; ``binding`` raises loudly if the CUDA library is missing.
"""
__version__ = "0.1.0"
