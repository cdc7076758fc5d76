"""Thin Python binding of include/stroke_expand.h: same names, argument marshalling only.

Every step of the path runs in the CUDA kernels of libstroke_expand.so; torch is used for device memory
and streams.  There is no CPU fallback: loading fails loudly when the library has not been built
(`python -m paper_2405_00127_b200.build`), and sx_create fails when there is no CUDA device.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
SO_PATH = os.path.join(_HERE, "libstroke_expand.so")

SX_OK, SX_E_INVALID_ARG, SX_E_BAD_STREAM, SX_E_CAPACITY, SX_E_CUDA, SX_E_STATE = 0, -1, -2, -3, -4, -5
SX_MODE_LINE, SX_MODE_ARC, SX_MODE_LINE_REFINED = 0, 1, 2
RECORD_BYTES = {SX_MODE_LINE: 16, SX_MODE_ARC: 32, SX_MODE_LINE_REFINED: 16}
ARC_DTYPE = np.dtype([("x0", "<f4"), ("y0", "<f4"), ("x1", "<f4"), ("y1", "<f4"), ("angle", "<f4"), ("seg", "<u4"),
                      ("kind", "<u4"), ("pad", "<u4")])

SX_OPT_KEEP_SEGMENT_INFO, SX_OPT_TILE_SEGMENTS, SX_OPT_TIME_KERNELS = 1, 2, 3

EXPORTS = ["sx_create", "sx_destroy", "sx_count", "sx_write", "stroke_expand", "stroke_expand_into", "stroke_expand_host",
           "sx_bin_lines", "sx_bin_lines_static", "sx_segment_info", "sx_last_error", "sx_set_option", "sx_set_dash", "sx_call_stats", "sx_kernel_times", "sx_measure_issue_peaks", "sx_eval", "sx_launch_count",
           "sx_strerror"]

ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_uint64, C.c_void_p)
_lib = None


class StrokeExpandError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        super().__init__(f"{where}: {sx_strerror(status)} (status {status})")


def lib():
    """Load the C-ABI library (built in-tree by paper_2405_00127_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(SO_PATH):
            raise ImportError(f"{SO_PATH} is missing: build it with `python -m paper_2405_00127_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(SO_PATH)
        vp, u64, i32, f32 = C.c_void_p, C.c_uint64, C.c_int32, C.c_float
        stream_args = [vp, u64, vp, u64, vp, u64, vp, f32, i32]  # tags, n, points, n, styles, n, affine, tol, mode
        L.sx_create.argtypes = [C.POINTER(vp), i32]
        L.sx_destroy.argtypes = [vp]
        L.sx_count.argtypes = [vp] + stream_args + [vp, C.POINTER(u64), vp]
        L.sx_write.argtypes = [vp, vp, u64, vp]
        L.stroke_expand.argtypes = [vp] + stream_args + [ALLOC_FN, vp, C.POINTER(vp), C.POINTER(u64), vp, vp]
        L.stroke_expand_into.argtypes = [vp] + stream_args + [vp, u64, vp, C.POINTER(u64), vp]
        L.stroke_expand_host.argtypes = [vp] + stream_args + [vp, u64, C.POINTER(u64), vp, vp]
        L.sx_segment_info.argtypes = [vp] + [C.POINTER(vp)] * 5
        L.sx_last_error.argtypes = [vp, vp]
        L.sx_set_option.argtypes = [vp, i32, u64]
        L.sx_set_dash.argtypes = [vp, vp, i32, f32]
        L.sx_bin_lines_static.argtypes = [i32, vp, u64, C.c_uint32, C.c_uint32, vp, vp, u64, vp, vp]
        L.sx_call_stats.argtypes = [vp, C.POINTER(u64), vp]
        L.sx_eval.argtypes = [C.c_int32, C.c_int32, vp, vp, u64]
        L.sx_bin_lines.argtypes = [vp, vp, u64, C.c_uint32, C.c_uint32, vp, vp, u64, C.POINTER(u64), vp]
        L.sx_kernel_times.argtypes = [vp, C.POINTER(C.c_float)]
        L.sx_measure_issue_peaks.argtypes = [i32, C.POINTER(C.c_double)]
        L.sx_launch_count.argtypes = [vp]
        L.sx_launch_count.restype = u64
        L.sx_strerror.argtypes = [i32]
        L.sx_strerror.restype = C.c_char_p
        for name in EXPORTS:
            if name not in ("sx_launch_count", "sx_strerror"):
                getattr(L, name).restype = i32
        _lib = L
    return _lib


def sx_strerror(status):
    return lib().sx_strerror(int(status)).decode()


def _check(status, where):
    if status != SX_OK:
        raise StrokeExpandError(status, where)


def _stream_ptr(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _affine(affine):
    a = np.ascontiguousarray(np.asarray(affine, dtype=np.float32).reshape(6))
    return a, C.c_void_p(a.ctypes.data)


def _dev_streams(tags, points, styles):
    """tags u8[N], points f32[Npts,2], styles u8[P,16] (or any 16-byte rows) as contiguous CUDA tensors.  The
    library wants tags / styles 16-byte and points 8-byte aligned (it answers SX_E_INVALID_ARG otherwise)."""
    assert tags.is_cuda and points.is_cuda and styles.is_cuda, "device tensors expected (use stroke_expand_host for host data)"
    assert tags.dtype == torch.uint8 and points.dtype == torch.float32 and styles.dtype == torch.uint8
    assert tags.is_contiguous() and points.is_contiguous() and styles.is_contiguous()
    n_paths = styles.numel() // 16
    return (C.c_void_p(tags.data_ptr()), tags.numel(), C.c_void_p(points.data_ptr()), points.numel() // 2,
            C.c_void_p(styles.data_ptr()), n_paths)


def sx_create(device=0):
    h = C.c_void_p()
    _check(lib().sx_create(C.byref(h), int(device)), "sx_create")
    return h


def sx_destroy(ctx):
    _check(lib().sx_destroy(ctx), "sx_destroy")


def sx_count(ctx, tags, points, styles, affine, tolerance, mode, path_offsets, want_total=True, stream=None):
    """Phase 1.  path_offsets: int64/uint64 CUDA tensor [n_paths+1], written.  Returns the record count (or None
    when want_total is False: the call then stays asynchronous)."""
    args = _dev_streams(tags, points, styles)
    a, ap = _affine(affine)
    assert path_offsets.is_cuda and path_offsets.is_contiguous() and path_offsets.element_size() == 8 and path_offsets.numel() >= args[5] + 1
    total = C.c_uint64(0)
    st = lib().sx_count(ctx, *args, ap, float(tolerance), int(mode), C.c_void_p(path_offsets.data_ptr()),
                        C.byref(total) if want_total else None, _stream_ptr(stream))
    _check(st, "sx_count")
    return int(total.value) if want_total else None


def sx_write(ctx, out_records, cap_records, mode=None, stream=None):
    """Phase 2.  out_records: CUDA tensor with room for cap_records records (16 B line / 32 B arc; pass the mode of
    the count to have the tensor's size checked against cap_records)."""
    assert out_records.is_cuda and out_records.is_contiguous()
    if mode is not None:
        assert out_records.numel() * out_records.element_size() >= int(cap_records) * RECORD_BYTES[int(mode)]
    _check(lib().sx_write(ctx, C.c_void_p(out_records.data_ptr()), int(cap_records), _stream_ptr(stream)), "sx_write")


def stroke_expand_into(ctx, tags, points, styles, affine, tolerance, mode, out_records, path_offsets, want_total=True, stream=None):
    """The whole path in one asynchronous call into a caller-provided CUDA tensor (float32 [cap,4] line / [cap,8] arc).  Returns
    the record count (None when want_total is False: the call stays asynchronous).  Raises SX_E_CAPACITY with the
    needed count in .needed when the records do not fit."""
    args = _dev_streams(tags, points, styles)
    a, ap = _affine(affine)
    width = 8 if mode == SX_MODE_ARC else 4
    assert out_records.is_cuda and out_records.is_contiguous() and out_records.dtype == torch.float32
    cap = out_records.numel() // width
    assert path_offsets.is_cuda and path_offsets.is_contiguous() and path_offsets.element_size() == 8 and path_offsets.numel() >= args[5] + 1
    total = C.c_uint64(0)
    st = lib().stroke_expand_into(ctx, *args, ap, float(tolerance), int(mode), C.c_void_p(out_records.data_ptr()), cap,
                                  C.c_void_p(path_offsets.data_ptr()), C.byref(total) if want_total else None, _stream_ptr(stream))
    if st == SX_E_CAPACITY:
        e = StrokeExpandError(st, "stroke_expand_into")
        e.needed = int(total.value)
        raise e
    _check(st, "stroke_expand_into")
    return int(total.value) if want_total else None


def stroke_expand(ctx, tags, points, styles, affine, tolerance, mode, stream=None):
    """One shot on device tensors.  Returns (records, path_offsets): records is a float32 CUDA tensor [M,4]
    (line mode) or [M,8] (arc mode: x0 y0 x1 y1 angle seg kind pad, the last three as raw bits);
    path_offsets an int64 CUDA tensor [n_paths+1].  The output is allocated by the torch caching allocator
    through the library's allocation callback."""
    args = _dev_streams(tags, points, styles)
    a, ap = _affine(affine)
    dev = tags.device
    path_offsets = torch.empty(args[5] + 1, dtype=torch.int64, device=dev)
    holder = {}
    width = 8 if mode == SX_MODE_ARC else 4

    def _alloc(nbytes, _user):
        t = torch.empty((nbytes // (4 * width), width), dtype=torch.float32, device=dev)
        holder["t"] = t
        return t.data_ptr()

    cb = ALLOC_FN(_alloc)
    out_ptr, n_rec = C.c_void_p(), C.c_uint64(0)
    st = lib().stroke_expand(ctx, *args, ap, float(tolerance), int(mode), cb, None, C.byref(out_ptr), C.byref(n_rec),
                             C.c_void_p(path_offsets.data_ptr()), _stream_ptr(stream))
    _check(st, "stroke_expand")
    rec = holder.get("t")
    if rec is None:
        rec = torch.empty((0, width), dtype=torch.float32, device=dev)
    return rec, path_offsets


def stroke_expand_host(ctx, tags, points, styles, affine, tolerance, mode, out_records, path_offsets, stream=None):
    """One shot on HOST tensors (pin them for asynchronous copies).  out_records: host float32 tensor [cap,4] or
    [cap,8]; path_offsets: host int64 tensor [n_paths+1].  Returns the record count; raises on SX_E_CAPACITY with
    the needed count in the exception's .needed."""
    for t in (tags, points, styles, out_records, path_offsets):
        assert not t.is_cuda and t.is_contiguous()
    assert tags.dtype == torch.uint8 and points.dtype == torch.float32 and styles.dtype == torch.uint8
    a, ap = _affine(affine)
    width = 8 if mode == SX_MODE_ARC else 4
    cap = out_records.numel() // width
    n_paths = styles.numel() // 16
    assert path_offsets.element_size() == 8 and path_offsets.numel() >= n_paths + 1
    n_rec = C.c_uint64(0)
    st = lib().stroke_expand_host(ctx, C.c_void_p(tags.data_ptr()), tags.numel(), C.c_void_p(points.data_ptr()),
                                  points.numel() // 2, C.c_void_p(styles.data_ptr()), n_paths, ap, float(tolerance), int(mode),
                                  C.c_void_p(out_records.data_ptr()), cap, C.byref(n_rec), C.c_void_p(path_offsets.data_ptr()),
                                  _stream_ptr(stream))
    if st == SX_E_CAPACITY:
        e = StrokeExpandError(st, "stroke_expand_host")
        e.needed = int(n_rec.value)
        raise e
    _check(st, "stroke_expand_host")
    return int(n_rec.value)


def sx_bin_lines(ctx, lines, tiles_x, tiles_y, tile_offsets, tile_lines=None, want_total=True, stream=None):
    """Tile binning of line records.  lines: float32 CUDA tensor [n, 4]; tile_offsets: int32 CUDA tensor
    [tiles_x * tiles_y + 1] (written, CSR); tile_lines: int32 CUDA tensor [cap] or None (count and scan only).  Returns the
    number of (tile, record) pairs when want_total (synchronises); raises StrokeExpandError with .needed on SX_E_CAPACITY."""
    assert lines.is_cuda and lines.is_contiguous() and lines.dtype == torch.float32 and lines.dim() == 2 and lines.shape[1] == 4
    assert tile_offsets.is_cuda and tile_offsets.is_contiguous() and tile_offsets.element_size() == 4
    assert tile_offsets.numel() >= int(tiles_x) * int(tiles_y) + 1
    cap = 0
    if tile_lines is not None:
        assert tile_lines.is_cuda and tile_lines.is_contiguous() and tile_lines.element_size() == 4
        cap = tile_lines.numel()
    total = C.c_uint64(0)
    st = lib().sx_bin_lines(ctx, C.c_void_p(lines.data_ptr()), lines.shape[0], int(tiles_x), int(tiles_y), C.c_void_p(tile_offsets.data_ptr()),
                            C.c_void_p(tile_lines.data_ptr() if cap else 0), cap, C.byref(total) if want_total else None, _stream_ptr(stream))
    if st == SX_E_CAPACITY:
        e = StrokeExpandError(st, "sx_bin_lines")
        e.needed = int(total.value)
        raise e
    _check(st, "sx_bin_lines")
    return int(total.value) if want_total else None


SX_STATIC_MAX_TILES, SX_STATIC_FLAG_CAPACITY = 65536, 2


def sx_bin_lines_static(lines, tiles_x, tiles_y, tile_offsets, tile_lines=None, flags=None, stream=None):
    """sx_bin_lines without a context and without any allocation (static device scratch; tiles_x * tiles_y <= 65536; calls that
    overlap on one GPU race).  Asynchronous: the pair total is tile_offsets[tiles_x * tiles_y]; flags: optional int32 CUDA tensor
    [1], written 0 or SX_STATIC_FLAG_CAPACITY.  The device is the tensors' device."""
    assert lines.is_cuda and lines.is_contiguous() and lines.dtype == torch.float32 and lines.dim() == 2 and lines.shape[1] == 4
    assert tile_offsets.is_cuda and tile_offsets.is_contiguous() and tile_offsets.element_size() == 4
    assert tile_offsets.numel() >= int(tiles_x) * int(tiles_y) + 1
    cap = 0
    if tile_lines is not None:
        assert tile_lines.is_cuda and tile_lines.is_contiguous() and tile_lines.element_size() == 4
        cap = tile_lines.numel()
    if flags is not None:
        assert flags.is_cuda and flags.element_size() == 4 and flags.numel() >= 1
    st = lib().sx_bin_lines_static(int(lines.device.index or 0), C.c_void_p(lines.data_ptr()), lines.shape[0], int(tiles_x), int(tiles_y),
                                   C.c_void_p(tile_offsets.data_ptr()), C.c_void_p(tile_lines.data_ptr() if cap else 0), cap,
                                   C.c_void_p(flags.data_ptr() if flags is not None else 0), _stream_ptr(stream))
    _check(st, "sx_bin_lines_static")


def _view(ptr, n, dtype, device):
    """Zero-copy torch view of ctx scratch memory (valid until the next call on the context)."""
    if n == 0 or not ptr:
        return torch.empty(0, dtype=dtype, device=device)
    nbytes = n * torch.empty(0, dtype=dtype).element_size()

    class _Mem:
        __cuda_array_interface__ = {"shape": (nbytes,), "typestr": "|u1", "data": (int(ptr), False), "version": 3}

    return torch.as_tensor(_Mem(), device=device).view(dtype)


def sx_segment_info(ctx, n_tags, device="cuda:0"):
    """Copies of the last sx_count's per-segment scan results: dict of CUDA tensors pt_off, path_idx, sp_first,
    seg_count (int32 views of the u32 data) and seg_offset (int64)."""
    ptrs = [C.c_void_p() for _ in range(5)]
    _check(lib().sx_segment_info(ctx, *[C.byref(p) for p in ptrs]), "sx_segment_info")
    names = ["pt_off", "path_idx", "sp_first", "seg_count", "seg_offset"]
    out = {}
    for name, p in zip(names, ptrs):
        dt = torch.int64 if name == "seg_offset" else torch.int32
        out[name] = _view(p.value, n_tags, dt, device).clone()
    return out


def sx_last_error(ctx, stream=None):
    return int(lib().sx_last_error(ctx, _stream_ptr(stream)))


def sx_set_option(ctx, option, value):
    _check(lib().sx_set_option(ctx, int(option), int(value)), "sx_set_option")


def sx_call_stats(ctx, stream=None):
    """dict(direct_tiles, sub_tiled_tiles, walk_segments, tile_segments) of the last expansion kernel on the context."""
    out = (C.c_uint64 * 4)()
    _check(lib().sx_call_stats(ctx, out, _stream_ptr(stream)), "sx_call_stats")
    return dict(direct_tiles=int(out[0]), sub_tiled_tiles=int(out[1]), walk_segments=int(out[2]), tile_segments=int(out[3]))


def sx_kernel_times(ctx):
    """(tag scan, count pass, allocation scan, writers) in ms of the last call made under SX_OPT_TIME_KERNELS (waits for it)."""
    out = (C.c_float * 4)()
    _check(lib().sx_kernel_times(ctx, out), "sx_kernel_times")
    return tuple(float(x) for x in out)


def sx_measure_issue_peaks(device=0):
    """dict(fp32_ffma, fp32_mix, mufu): measured lane-operations per second (issue-rate microbenchmarks)."""
    out = (C.c_double * 3)()
    _check(lib().sx_measure_issue_peaks(int(device), out), "sx_measure_issue_peaks")
    return dict(fp32_ffma=float(out[0]), fp32_mix=float(out[1]), mufu=float(out[2]))


SX_EVAL_ATAN2, SX_EVAL_NODE_ERROR, SX_EVAL_F_EXACT, SX_EVAL_F_INV_REFINED = 0, 1, 2, 3


def sx_eval(what, values, device=0):
    """Probe of one device function of the kernels (tests): values float32 numpy [n, 2] (atan2: y, x) or [n, 9] (node error:
    u0, u1, |q0|, |q1|, chord, dt); returns float32 numpy [n]."""
    v = np.ascontiguousarray(values, dtype=np.float32)
    n = v.shape[0]
    out = np.zeros(n, dtype=np.float32)
    _check(lib().sx_eval(int(device), int(what), C.c_void_p(v.ctypes.data), C.c_void_p(out.ctypes.data), n), "sx_eval")
    return out


def sx_set_dash(ctx, lengths=None, phase=0.0):
    """Dash pattern of the context: 2, 4, 6 or 8 positive lengths in output px and a phase; None clears it."""
    if lengths is None or len(lengths) == 0:
        _check(lib().sx_set_dash(ctx, None, 0, C.c_float(0.0)), "sx_set_dash")
        return
    v = np.ascontiguousarray(lengths, dtype=np.float32)
    _check(lib().sx_set_dash(ctx, C.c_void_p(v.ctypes.data), int(v.shape[0]), C.c_float(float(phase))), "sx_set_dash")


def sx_launch_count(ctx):
    return int(lib().sx_launch_count(ctx))


def scene_to_torch(scene, device=None, pin=False):
    """Marshal a scenes.Scene (numpy streams) into the tensors the calls above take."""
    tags = torch.from_numpy(np.ascontiguousarray(scene["tags"]))
    points = torch.from_numpy(np.ascontiguousarray(scene["points"], dtype=np.float32))
    styles = torch.from_numpy(np.ascontiguousarray(scene["styles"]).view(np.uint8).reshape(-1, 16).copy())
    if device is not None:
        return tags.to(device), points.to(device), styles.to(device)
    if pin:
        return tags.pin_memory(), points.pin_memory(), styles.pin_memory()
    return tags, points, styles
