"""Seeded synthetic scenes (the C-ABI input streams) for the five BASELINE.json configs.

This module holds NONE of the method's arithmetic: it only draws random control points and styles
(numpy PCG64, float64 draws cast to fp32) and packs them into the tag / point / style streams of
include/stroke_expand.h.  It is the one module that both the oracle-side tests and the CUDA-side
tests import.  The scenes stand in for the paper's own workloads (Nehab "timings", roads.svg,
mmark, long-dash: Tables 2-4), which are not available; the recipes are
DESIGN.md section 4.

Tag byte (Table 1): bits 0-1 coordinate count, bit 2 subpath end, bit 4 path end,
bit 7 closed subpath (R-8).  Point stream (L464, L470, L483): a subpath of k segments owns
1 + sum(count) points; consecutive segments share an end point.
"""
from __future__ import annotations

import numpy as np

STYLE_DTYPE = np.dtype([("width", "<f4"), ("miter_limit", "<f4"), ("join", "u1"), ("cap", "u1"),
                        ("fill", "<u2"), ("rsv", "<u4")])   # fill: bit 0 = the path is filled, not stroked
JOIN_MITER, JOIN_ROUND, JOIN_BEVEL = 0, 1, 2
CAP_BUTT, CAP_SQUARE, CAP_ROUND = 0, 1, 2
MODE_LINE, MODE_ARC = 0, 1
TAG_SUBPATH_END, TAG_PATH_END, TAG_CLOSED = 4, 16, 128

IDENTITY = np.array([1, 0, 0, 1, 0, 0], dtype=np.float32)


class Scene(dict):
    """tags u8[N], points f32[Npts,2], styles STYLE_DTYPE[P], affine f32[6], tolerance, modes."""

    __getattr__ = dict.__getitem__

    @property
    def n_segments(self):
        return int(self["tags"].shape[0])

    @property
    def n_paths(self):
        return int(self["styles"].shape[0])


def make_styles(width, join, cap, miter_limit):
    n = len(width)
    st = np.zeros(n, dtype=STYLE_DTYPE)
    st["width"] = np.asarray(width, dtype=np.float32)
    st["join"] = join
    st["cap"] = cap
    st["miter_limit"] = miter_limit
    return st


def pack_paths(seg_len, cnt, start, ctrl, closed):
    """One subpath per path.  seg_len[P] segments per path; cnt[N] in {1,2,3}; start[P,2] first point;
    ctrl[N,3,2] the (up to 3) points each segment appends; closed[P] bool.  Returns tags, points."""
    seg_len = np.asarray(seg_len, dtype=np.int64)
    n = int(seg_len.sum())
    p = len(seg_len)
    last = np.cumsum(seg_len) - 1
    first = last - seg_len + 1
    tags = cnt.astype(np.uint8).copy()
    tags[last] |= TAG_SUBPATH_END | TAG_PATH_END
    tags[last[np.asarray(closed, dtype=bool)]] |= TAG_CLOSED
    end = np.zeros(n, dtype=np.int64)
    end[last] = 1
    inc = cnt.astype(np.int64) + end
    pt_off = np.cumsum(inc) - inc
    npts = int(inc.sum())
    pts = np.zeros((npts, 2), dtype=np.float32)
    pts[pt_off[first]] = start.astype(np.float32)
    for j in range(3):
        m = cnt > j
        pts[pt_off[m] + j + 1] = ctrl[m, j].astype(np.float32)
    return tags, pts


def _shift_into(start, ctrl, seg_len, lo, hi):
    """Translate whole paths so every control point lies in [lo,hi] (keeps the fp32 ulp below 1e-3 px)."""
    pid = np.repeat(np.arange(len(seg_len)), seg_len)
    ends = np.cumsum(seg_len)
    begs = ends - seg_len
    for ax in range(2):
        c = ctrl[:, :, ax]
        mn = np.minimum(np.minimum.reduceat(c.min(axis=1), begs), start[:, ax])
        mx = np.maximum(np.maximum.reduceat(c.max(axis=1), begs), start[:, ax])
        sh = np.where(mn < lo, lo - mn, 0.0) + np.where(mx > hi, hi - mx, 0.0)
        start[:, ax] += sh
        ctrl[:, :, ax] += sh[pid][:, None]


# ------------------------------------------------------------------ config 1
def config1(n_paths=256, seed=0):
    """256 open paths x 8 cubics, control points U([0,512]^2), G0; width U[1,20]; round join, butt cap."""
    rng = np.random.default_rng(seed)
    seg_len = np.full(n_paths, 8)
    n = int(seg_len.sum())
    start = rng.uniform(0, 512, (n_paths, 2))
    ctrl = rng.uniform(0, 512, (n, 3, 2))
    cnt = np.full(n, 3)
    tags, pts = pack_paths(seg_len, cnt, start, ctrl, np.zeros(n_paths, bool))
    st = make_styles(rng.uniform(1, 20, n_paths), JOIN_ROUND, CAP_BUTT, 4.0)
    return Scene(name="c1", tags=tags, points=pts, styles=st, affine=IDENTITY.copy(), tolerance=0.25, modes=(MODE_LINE,))


# ------------------------------------------------------------------ config 2
def config2(n_paths=2000, seed=1):
    """Style and degeneracy coverage (C2)."""
    rng = np.random.default_rng(seed)
    seg_len = rng.integers(4, 33, n_paths)
    closed = (np.arange(n_paths) % 2) == 0
    n = int(seg_len.sum())
    cnt = rng.integers(1, 4, n)
    start = rng.uniform(64, 960, (n_paths, 2))
    ctrl = np.zeros((n, 3, 2))
    i = 0
    for p in range(n_paths):
        cur = start[p].copy()
        for k in range(seg_len[p]):
            c = cnt[i]
            pts = [cur]
            for _ in range(c):
                pts.append(pts[-1] + rng.normal(0, 60, 2))
            if c == 3:
                r = rng.uniform()
                if r < 0.05:  # cusped: control polygon crosses itself, p1 ~ p3, p2 ~ p0
                    pts[1] = pts[3] + rng.normal(0, 4, 2)
                    pts[2] = pts[0] + rng.normal(0, 4, 2)
                elif r < 0.10:  # coincident inner control points
                    pts[2] = pts[1].copy()
                elif r < 0.15:  # zero-length handle(s)
                    w = rng.integers(0, 3)
                    if w in (0, 2):
                        pts[1] = pts[0].copy()
                    if w in (1, 2):
                        pts[2] = pts[3].copy()
                elif r < 0.20:  # collinear
                    u = rng.uniform(-0.5, 1.5, 2)
                    pts[1] = pts[0] + u[0] * (pts[3] - pts[0])
                    pts[2] = pts[0] + u[1] * (pts[3] - pts[0])
            if closed[p] and k == seg_len[p] - 1:
                pts[c] = start[p].copy()  # ends bit-exactly on the first point
            for j in range(c):
                ctrl[i, j] = pts[j + 1]
            cur = pts[c]
            i += 1
    tags, pts_ = pack_paths(seg_len, cnt, start, ctrl, closed)
    width = np.exp(rng.uniform(np.log(0.5), np.log(64), n_paths))
    st = make_styles(width, rng.integers(0, 3, n_paths), rng.integers(0, 3, n_paths), 4.0)
    return Scene(name="c2", tags=tags, points=pts_, styles=st, affine=IDENTITY.copy(), tolerance=0.25,
                 modes=(MODE_LINE, MODE_ARC))


def _segmented_cumsum(v, seg_len):
    """inclusive cumsum of v[N,...] restarted at each path."""
    cs = np.cumsum(v, axis=0)
    ends = np.cumsum(seg_len)
    begs = ends - seg_len
    base = np.zeros_like(cs[:1]).repeat(len(seg_len), axis=0)
    base[1:] = cs[begs[1:] - 1]
    return cs - np.repeat(base, seg_len, axis=0)


def _dir(a):
    return np.stack([np.cos(a), np.sin(a)], axis=-1)


# ------------------------------------------------------------------ config 3
def config3(n_paths=50000, seed=2):
    """Map-like scene: open polylines-with-curves, small turning angles, random similarity transform."""
    rng = np.random.default_rng(seed)
    seg_len = np.clip(rng.geometric(1.0 / 10.0, n_paths), 2, 40)
    n = int(seg_len.sum())
    cnt = np.where(rng.uniform(size=n) < 0.7, 1, 3)
    start = rng.uniform(256, 3840, (n_paths, 2))
    turn = np.deg2rad(rng.uniform(-30, 30, n))
    h0 = rng.uniform(0, 2 * np.pi, n_paths)
    head_new = _segmented_cumsum(turn, seg_len) + np.repeat(h0, seg_len)
    head_old = head_new - turn
    chord = rng.uniform(5, 40, n)
    step = chord[:, None] * _dir(0.5 * (head_old + head_new))
    endp = _segmented_cumsum(step, seg_len) + np.repeat(start, seg_len, axis=0)
    begp = endp - step
    ctrl = np.zeros((n, 3, 2))
    cub = cnt == 3
    ctrl[~cub, 0] = endp[~cub]
    ctrl[cub, 0] = begp[cub] + (chord[cub] / 3)[:, None] * _dir(head_old[cub])
    ctrl[cub, 1] = endp[cub] - (chord[cub] / 3)[:, None] * _dir(head_new[cub])
    ctrl[cub, 2] = endp[cub]
    tags, pts = pack_paths(seg_len, cnt, start, ctrl, np.zeros(n_paths, bool))
    st = make_styles(rng.uniform(0.5, 3, n_paths), JOIN_ROUND, CAP_ROUND, 4.0)
    ang, sc = rng.uniform(0, 2 * np.pi), rng.uniform(0.5, 2)
    a, b = sc * np.cos(ang), sc * np.sin(ang)
    cx = cy = 2048.0
    aff = np.array([a, b, -b, a, cx - a * cx + b * cy, cy - b * cx - a * cy], dtype=np.float32)
    return Scene(name="c3", tags=tags, points=pts, styles=st, affine=aff, tolerance=0.25, modes=(MODE_LINE,))


# ------------------------------------------------------------------ config 4
def config4(n_paths=100000, seed=3):
    """CAD-scale scene: 10 segments per open path, 50/50 line/cubic, miter joins (limit 10), butt caps."""
    rng = np.random.default_rng(seed)
    seg_len = np.full(n_paths, 10)
    n = int(seg_len.sum())
    cnt = np.where(rng.uniform(size=n) < 0.5, 1, 3)
    start = rng.uniform(512, 15872, (n_paths, 2))
    turn = np.deg2rad(rng.uniform(-90, 90, n))
    h0 = rng.uniform(0, 2 * np.pi, n_paths)
    head = _segmented_cumsum(turn, seg_len) + np.repeat(h0, seg_len)
    chord = np.exp(rng.uniform(np.log(8), np.log(256), n))
    step = chord[:, None] * _dir(head)
    endp = _segmented_cumsum(step, seg_len) + np.repeat(start, seg_len, axis=0)
    begp = endp - step
    hl = chord[:, None] * rng.uniform(0.2, 0.5, (n, 2))
    hd = head[:, None] + np.deg2rad(rng.uniform(-45, 45, (n, 2)))
    ctrl = np.zeros((n, 3, 2))
    cub = cnt == 3
    ctrl[~cub, 0] = endp[~cub]
    ctrl[cub, 0] = begp[cub] + hl[cub, 0, None] * _dir(hd[cub, 0])
    ctrl[cub, 1] = endp[cub] - hl[cub, 1, None] * _dir(hd[cub, 1])
    ctrl[cub, 2] = endp[cub]
    _shift_into(start, ctrl, seg_len, 0.0, 16383.0)
    tags, pts = pack_paths(seg_len, cnt, start, ctrl, np.zeros(n_paths, bool))
    st = make_styles(rng.uniform(0.25, 8, n_paths), JOIN_MITER, CAP_BUTT, 10.0)
    return Scene(name="c4", tags=tags, points=pts, styles=st, affine=IDENTITY.copy(), tolerance=0.1, modes=(MODE_ARC,))


# ------------------------------------------------------------------ config 5
def config5(n_paths=200000, seed=4):
    """Evolute / stress scene: closed paths of 50 cubics, Brownian-bridge control points (sigma 40 px)."""
    rng = np.random.default_rng(seed)
    k = 50
    seg_len = np.full(n_paths, k)
    n = n_paths * k
    start = rng.uniform(2048, 14336, (n_paths, 2))
    steps = rng.normal(0, 40, (n_paths, 3 * k, 2))
    steps -= steps.mean(axis=1, keepdims=True)  # bridge: the walk returns to its start
    pos = np.cumsum(steps, axis=1)
    pos[:, -1] = 0.0
    ctrl = (pos + start[:, None, :]).reshape(n, 3, 2)
    _shift_into(start, ctrl, seg_len, 0.0, 16383.0)
    ctrl.reshape(n_paths, 3 * k, 2)[:, -1] = start  # bit-exact closure after the shift
    cnt = np.full(n, 3)
    tags, pts = pack_paths(seg_len, cnt, start, ctrl, np.ones(n_paths, bool))
    st = make_styles(rng.uniform(20, 100, n_paths), JOIN_ROUND, CAP_BUTT, 4.0)
    return Scene(name="c5", tags=tags, points=pts, styles=st, affine=IDENTITY.copy(), tolerance=0.25,
                 modes=(MODE_LINE, MODE_ARC))


CONFIGS = {"c1": config1, "c2": config2, "c3": config3, "c4": config4, "c5": config5}


def make(name, n_paths=None, seed=None):
    kw = {}
    if n_paths is not None:
        kw["n_paths"] = n_paths
    if seed is not None:
        kw["seed"] = seed
    return CONFIGS[name](**kw)


def with_fill(scene, every=1, offset=0):
    """Copy of the scene in which every `every`-th path (starting at `offset`) is FILLED instead of stroked (Alg. 1
    L309-311: style bit only, no arithmetic here)."""
    st = scene["styles"].copy()
    st["fill"][offset::every] = 1
    out = Scene(scene)
    out["styles"] = st
    out["name"] = scene["name"] + "-fill"
    return out


def with_dash(scene, every=1, offset=0):
    """Copy of the scene in which every `every`-th path (starting at `offset`) is DASHED with the call's dash pattern
    (bit 1 of the style's `fill` field, no arithmetic here)."""
    st = scene["styles"].copy()
    st["fill"][offset::every] |= 2
    out = Scene(scene)
    out["styles"] = st
    out["name"] = scene["name"] + "-dash"
    return out


def subset_paths(scene, path_ids):
    """Sub-scene holding only the given paths (paths are independent units): used to run the oracle on a
    sample of a large scene.  Each path here is one subpath."""
    tags = scene["tags"]
    cnt = (tags & 3).astype(np.int64)
    end = ((tags >> 2) | (tags >> 4)) & 1
    inc = cnt + end
    pt_off = np.cumsum(inc) - inc
    pend = np.flatnonzero(tags & TAG_PATH_END)
    pbeg = np.concatenate([[0], pend[:-1] + 1])
    tsel, psel = [], []
    for p in path_ids:
        a, b = pbeg[p], pend[p] + 1
        tsel.append(np.arange(a, b))
        psel.append(np.arange(pt_off[a], pt_off[b - 1] + inc[b - 1]))
    tsel = np.concatenate(tsel)
    psel = np.concatenate(psel)
    return Scene(name=scene["name"] + "_sub", tags=tags[tsel].copy(), points=scene["points"][psel].copy(),
                 styles=scene["styles"][np.asarray(path_ids)].copy(), affine=scene["affine"].copy(),
                 tolerance=scene["tolerance"], modes=scene["modes"]), tsel


def from_paths(paths, tolerance=0.25, affine=None, modes=(MODE_LINE,)):
    """Hand-built scene.  paths: list of dicts {pts: [P0, seg1 pts..., ...] as a list of segments where each
    segment is a list of 1, 2 or 3 points (the first path point is given as 'start'), closed, width, join, cap,
    miter_limit}."""
    seg_len, cnt, start, ctrl, closed, width, join, cap, ml = [], [], [], [], [], [], [], [], []
    for p in paths:
        segs = p["segs"]
        seg_len.append(len(segs))
        start.append(p["start"])
        closed.append(bool(p.get("closed", False)))
        width.append(p.get("width", 1.0))
        join.append(p.get("join", JOIN_MITER))
        cap.append(p.get("cap", CAP_BUTT))
        ml.append(p.get("miter_limit", 4.0))
        for s in segs:
            cnt.append(len(s))
            c = np.zeros((3, 2))
            c[:len(s)] = np.asarray(s, dtype=np.float64)
            ctrl.append(c)
    tags, pts = pack_paths(np.array(seg_len), np.array(cnt), np.array(start, dtype=np.float64), np.array(ctrl), np.array(closed))
    st = make_styles(width, np.array(join), np.array(cap), np.array(ml, dtype=np.float32))
    aff = IDENTITY.copy() if affine is None else np.asarray(affine, dtype=np.float32)
    return Scene(name="hand", tags=tags, points=pts, styles=st, affine=aff, tolerance=tolerance, modes=modes)
