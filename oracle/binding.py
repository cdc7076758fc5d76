"""ctypes loader for oracle/stroke_oracle.c (builds it with gcc when the .so is missing or stale)."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "stroke_oracle.c")
_SO = os.path.join(_HERE, "libstroke_oracle.so")
_lib = None

STAT_NAMES = ["fit_iters", "pieces", "ranges_reg", "ranges_sup", "rec_offset", "rec_evolute", "rec_connector",
              "joins", "caps", "line_segs", "curve_segs"]


class _Result(C.Structure):
    _fields_ = [("n_rec", C.c_uint64), ("xy", C.POINTER(C.c_float)), ("angle", C.POINTER(C.c_float)),
                ("kind", C.POINTER(C.c_uint8)), ("seg", C.POINTER(C.c_uint32)), ("seg_count", C.POINTER(C.c_uint32)),
                ("path_off", C.POINTER(C.c_uint64)), ("pt_off", C.POINTER(C.c_uint32)),
                ("path_idx", C.POINTER(C.c_uint32)), ("sp_first", C.POINTER(C.c_uint32)),
                ("stats", C.c_uint64 * 16), ("cap", C.c_uint64)]


def build(force=False):
    """gcc -O2 -ffp-contract=off (no FMA contraction: the oracle's fp32 decisions are plain IEEE ops)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fPIC", "-shared", "-o", _SO, _SRC, "-lm"])
    return _SO


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.so_expand.restype = C.c_int
        L.so_expand.argtypes = [C.c_void_p, C.c_uint64, C.c_void_p, C.c_uint64, C.c_void_p, C.c_uint64, C.c_void_p,
                                C.c_float, C.c_int, C.POINTER(_Result)]
        L.so_expand_dashed.restype = C.c_int
        L.so_expand_dashed.argtypes = [C.c_void_p, C.c_uint64, C.c_void_p, C.c_uint64, C.c_void_p, C.c_uint64, C.c_void_p,
                                       C.c_float, C.c_int, C.c_void_p, C.c_int, C.c_float, C.POINTER(_Result)]
        L.so_free.argtypes = [C.POINTER(_Result)]
        L.so_tag_walk.restype = C.c_int
        L.so_tag_walk.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint64, C.c_void_p, C.c_void_p, C.c_void_p]
        L.so_f_exact.restype = C.c_double
        L.so_f_exact.argtypes = [C.c_double]
        L.so_f_approx.restype = C.c_float
        L.so_f_approx.argtypes = [C.c_float]
        L.so_f_approx_inv.restype = C.c_float
        L.so_f_approx_inv.argtypes = [C.c_float]
        L.so_f_inv_newton.restype = C.c_double
        L.so_f_inv_newton.argtypes = [C.c_float, C.c_int]
        L.so_f_inv_refined.restype = C.c_float
        L.so_f_inv_refined.argtypes = [C.c_float]
        L.so_ghi.argtypes = [C.c_float, C.c_float, C.POINTER(C.c_float), C.POINTER(C.c_float)]
        L.so_es_integral.argtypes = [C.c_double, C.c_double, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.so_piece_expand.restype = C.c_int
        L.so_piece_expand.argtypes = [C.c_float] * 8 + [C.c_int, C.POINTER(_Result)]
        L.so_fit_error_export.argtypes = [C.c_void_p, C.c_void_p, C.c_float, C.c_float, C.c_void_p, C.c_float, C.c_void_p]
        _lib = L
    return _lib


class OracleResult:
    def __init__(self, xy, angle, kind, seg, seg_count, path_off, pt_off, path_idx, sp_first, stats):
        self.xy, self.angle, self.kind, self.seg = xy, angle, kind, seg
        self.seg_count, self.path_off = seg_count, path_off
        self.pt_off, self.path_idx, self.sp_first = pt_off, path_idx, sp_first
        self.stats = stats

    @property
    def n_rec(self):
        return self.xy.shape[0]


def _arr(ptr, n, dtype, width=1):
    if n == 0:
        return np.zeros((0, width) if width > 1 else (0,), dtype=dtype)
    a = np.ctypeslib.as_array(ptr, shape=(n * width,)).astype(dtype, copy=True)
    return a.reshape(n, width) if width > 1 else a


def _collect(r, n, p):
    m = int(r.n_rec)
    res = OracleResult(_arr(r.xy, m, np.float32, 4), _arr(r.angle, m, np.float32), _arr(r.kind, m, np.uint8),
                       _arr(r.seg, m, np.uint32), _arr(r.seg_count, n, np.uint32), _arr(r.path_off, p + 1, np.uint64),
                       _arr(r.pt_off, n, np.uint32), _arr(r.path_idx, n, np.uint32), _arr(r.sp_first, n, np.uint32),
                       dict(zip(STAT_NAMES, [int(x) for x in r.stats[:len(STAT_NAMES)]])))
    lib().so_free(C.byref(r))
    return res


def piece_expand(k0, k1, L, h, tol_fl, mode, x0=0.0, y0=0.0, dir0=0.0):
    """Both sides of ONE Euler-spiral piece given by its parameters (so_piece_expand): for the pins that measure
    the emitted arcs / evolute chords against the exact spiral."""
    r = _Result()
    rc = lib().so_piece_expand(k0, k1, L, x0, y0, dir0, h, tol_fl, int(mode), C.byref(r))
    if rc != 0:
        raise ValueError(f"oracle so_piece_expand failed: {rc}")
    return _collect(r, 1, 1)


def expand(tags, points, styles, affine, tolerance, mode, dash=None, phase=0.0):
    """Run the oracle on host numpy streams; returns OracleResult (copies; C buffers are freed).  dash: the call's dash
    pattern (2, 4, 6 or 8 positive lengths in output px) for the paths whose style has bit 1 of `fill` set; phase >= 0."""
    L = lib()
    tags = np.ascontiguousarray(tags, dtype=np.uint8)
    points = np.ascontiguousarray(points, dtype=np.float32)
    styles = np.ascontiguousarray(styles)
    affine = np.ascontiguousarray(affine, dtype=np.float32)
    assert styles.dtype.itemsize == 16 and affine.shape == (6,)
    r = _Result()
    n, p = tags.shape[0], styles.shape[0]
    if dash is None:
        rc = L.so_expand(tags.ctypes.data, n, points.ctypes.data, points.shape[0], styles.ctypes.data, p,
                         affine.ctypes.data, float(tolerance), int(mode), C.byref(r))
    else:
        d = np.ascontiguousarray(dash, dtype=np.float32)
        rc = L.so_expand_dashed(tags.ctypes.data, n, points.ctypes.data, points.shape[0], styles.ctypes.data, p,
                                affine.ctypes.data, float(tolerance), int(mode), d.ctypes.data, int(d.shape[0]), float(phase), C.byref(r))
    if rc != 0:
        raise ValueError(f"oracle so_expand failed: {rc}")
    return _collect(r, n, p)
