"""paper_1711_10855_b200 -- B200-native FDAS matched-filter hot path (arXiv:1711.10855, eq.(2)).

`binding` is the thin ctypes layer over the C-ABI library declared in include/fdas.h (built from
csrc/ into libfdas.so next to this file); `workload` makes the seeded synthetic inputs.  Nothing here
computes on the CPU: if libfdas.so is missing, `binding` raises on first use.
"""
__all__ = ["binding", "workload"]
