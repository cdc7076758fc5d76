"""B200-native stroke expansion (arxiv 2405.00127): CUDA kernels behind the C-ABI of include/stroke_expand.h.

`scenes` (seeded synthetic inputs) imports nothing heavy; `binding` (torch + ctypes over libstroke_expand.so)
is imported on first use so that CPU-only tools can import the package without a GPU.
"""
__all__ = ["scenes", "binding", "build"]
