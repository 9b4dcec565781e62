"""PULSE skip-local pipeline stage, B200-native (arxiv/paper_2606_19163).

The product is `libpulse.so` (C-ABI, `include/pulse.h`) plus the thin ctypes
binding in `binding.py`.  `workloads.py` holds only stage *structure* and the
seeded synthetic-input recipe (no arithmetic of the method) and is importable
without the CUDA library; `binding` is imported lazily and fails loudly when
the library is missing.
"""
__all__ = ["workloads", "binding"]
