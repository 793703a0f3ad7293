"""paper_1905_05727_b200 -- B200-native hot path of arXiv:1905.05727.

`inputs` holds the workload recipes; `binding` is the thin ctypes layer over libnmsdt.so
(loaded lazily so that CPU-only tools can import `inputs` without a CUDA runtime).
"""
__all__ = ["inputs", "binding"]
