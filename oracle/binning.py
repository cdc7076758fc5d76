"""ctypes loader for oracle/bin_oracle.c (tile binning of the line soup).  TEST INFRASTRUCTURE ONLY."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bin_oracle.c")
_SO = os.path.join(_HERE, "libbin_oracle.so")
_lib = None


def build(force=False):
    """gcc -O2 -ffp-contract=off: the walk decides integers in fp32, one rounding per operation."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fPIC", "-shared", "-o", _SO, _SRC, "-lm"])
    return _SO


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.bo_bin_lines.restype = C.c_uint64
        L.bo_bin_lines.argtypes = [C.c_void_p, C.c_uint64, C.c_uint32, C.c_uint32, C.c_void_p, C.c_void_p]
        _lib = L
    return _lib


def bin_lines(lines, tiles_x, tiles_y):
    """lines: float32 [n, 4] (x0 y0 x1 y1).  Returns (tile_offsets uint32 [tiles + 1], tile_lines uint32 [total]), the
    lines of every tile in increasing order."""
    lines = np.ascontiguousarray(lines, dtype=np.float32).reshape(-1, 4)
    tiles = int(tiles_x) * int(tiles_y)
    off = np.zeros(tiles + 1, dtype=np.uint32)
    total = lib().bo_bin_lines(lines.ctypes.data, lines.shape[0], int(tiles_x), int(tiles_y), off.ctypes.data, None)
    out = np.zeros(max(int(total), 1), dtype=np.uint32)
    lib().bo_bin_lines(lines.ctypes.data, lines.shape[0], int(tiles_x), int(tiles_y), off.ctypes.data, out.ctypes.data)
    return off, out[: int(total)]
