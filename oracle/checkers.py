"""Double-precision checkers for stroke outlines (TEST INFRASTRUCTURE; numpy only).

They test an outline (from the oracle or from the CUDA path -- "the same checks", north_star) against
what the paper and the mathematics fix, independent of either implementation:

* watertight: per path, the multiset of record start points equals the multiset of end points, bitwise
  ("produce a watertight outline").
* winding numbers: never negative; >= 1 inside the stroked region; 0 outside (L29 strong correctness,
  L191, L197 "All winding numbers are positive").  For round joins + round caps the region is exactly
  {X : dist(X, path) <= h}; distance by dense sampling + brute-force nearest point.
* offset accuracy: every vertex of an offset record lies within tol of the true parallel curve
  C(s) + eta N(s) of its source segment (L37 Frechet tolerance), the true curve sampled densely and
  adaptively from the source cubic itself (not from the Euler spirals).
"""
from __future__ import annotations

import numpy as np

K_OFFSET, K_OFFSET_REV, K_EVOLUTE, K_CONNECTOR, K_JOIN_OUTER, K_JOIN_INNER, K_CAP, K_PLUS = 0, 1, 2, 3, 4, 5, 6, 8


# ------------------------------------------------------------------ watertightness
def watertight_violations(xy, path_off):
    """Number of paths whose start-point multiset differs from the end-point multiset (bitwise)."""
    xy = np.ascontiguousarray(xy, dtype=np.float32)
    m = xy.shape[0]
    if m == 0:
        return 0
    xy = xy + np.float32(0.0)  # -0.0 == +0.0 as points
    bits = xy.view(np.uint32).reshape(m, 4).astype(np.uint64)
    s = (bits[:, 0] << np.uint64(32)) | bits[:, 1]
    e = (bits[:, 2] << np.uint64(32)) | bits[:, 3]
    path_off = np.asarray(path_off, dtype=np.int64)
    pid = np.repeat(np.arange(len(path_off) - 1), np.diff(path_off))
    os_ = np.lexsort((s, pid))
    oe = np.lexsort((e, pid))
    bad = s[os_] != e[oe]
    return int(np.unique(pid[os_][bad]).size)


# ------------------------------------------------------------------ geometry of the source path (double)
def transform_points(points, affine):
    a, b, c, d, e, f = [float(v) for v in affine]
    p = np.asarray(points, dtype=np.float64)
    return np.stack([a * p[:, 0] + c * p[:, 1] + e, b * p[:, 0] + d * p[:, 1] + f], axis=1)


def segment_cubics(tags, points, affine):
    """[N,4,2] cubic control points (device space, double) of every segment, by degree elevation (L349)."""
    tags = np.asarray(tags)
    cnt = (tags & 3).astype(np.int64)
    end = ((tags >> 2) | (tags >> 4)) & 1
    inc = cnt + end
    off = np.cumsum(inc) - inc
    p = transform_points(points, affine)
    n = len(tags)
    cub = np.zeros((n, 4, 2))
    p0 = p[off]
    cub[:, 0] = p0
    l = cnt == 1
    q = cnt == 2
    c = cnt == 3
    p1 = p[off + 1]
    cub[l, 3] = p1[l]
    cub[l, 1] = p0[l] + (p1[l] - p0[l]) / 3
    cub[l, 2] = p0[l] + (p1[l] - p0[l]) * 2 / 3
    p2 = p[np.minimum(off + 2, len(p) - 1)]
    cub[q, 3] = p2[q]
    cub[q, 1] = p0[q] + (p1[q] - p0[q]) * 2 / 3
    cub[q, 2] = p2[q] + (p1[q] - p2[q]) * 2 / 3
    p3 = p[np.minimum(off + 3, len(p) - 1)]
    cub[c, 1] = p1[c]
    cub[c, 2] = p2[c]
    cub[c, 3] = p3[c]
    return cub


def cubic_eval(cb, t):
    t = np.asarray(t, dtype=np.float64)[:, None]
    mt = 1 - t
    return mt ** 3 * cb[0] + 3 * mt * mt * t * cb[1] + 3 * mt * t * t * cb[2] + t ** 3 * cb[3]


def cubic_deriv(cb, t):
    t = np.asarray(t, dtype=np.float64)[:, None]
    mt = 1 - t
    return 3 * (mt * mt * (cb[1] - cb[0]) + 2 * mt * t * (cb[2] - cb[1]) + t * t * (cb[3] - cb[2]))


def adaptive_params(cb, n0=257, max_turn=0.02, rounds=24):
    """Parameters dense enough that the tangent turns < max_turn between neighbours (near-cusps get many)."""
    t = np.linspace(0, 1, n0)
    for _ in range(rounds):
        d = cubic_deriv(cb, t)
        ang = np.arctan2(d[:, 1], d[:, 0])
        turn = np.abs(np.angle(np.exp(1j * np.diff(ang))))
        bad = np.flatnonzero((turn > max_turn) & (np.diff(t) > 1e-12))
        if bad.size == 0:
            break
        t = np.sort(np.concatenate([t, 0.5 * (t[bad] + t[bad + 1])]))
    return t


def true_offset_polyline(cb, eta, **kw):
    """Dense polyline of the true parallel curve C + eta N (N = left normal)."""
    t = adaptive_params(cb, **kw)
    p = cubic_eval(cb, t)
    d = cubic_deriv(cb, t)
    nrm = np.hypot(d[:, 0], d[:, 1])
    ok = nrm > 1e-12
    p, d, nrm = p[ok], d[ok], nrm[ok]
    n = np.stack([-d[:, 1], d[:, 0]], axis=1) / nrm[:, None]
    return p + eta * n


def dist_points_to_polyline(x, poly):
    """min distance from each point x[S,2] to the polyline poly[K,2] (brute force, S x K)."""
    x = np.asarray(x, dtype=np.float64)
    a = poly[:-1]
    ab = poly[1:] - a
    l2 = np.maximum((ab * ab).sum(axis=1), 1e-300)
    out = np.empty(len(x))
    step = max(1, int(4e6 // max(1, len(a))))
    for i in range(0, len(x), step):
        xa = x[i:i + step, None, :] - a[None]
        u = np.clip((xa * ab[None]).sum(axis=2) / l2[None], 0, 1)
        d = xa - u[..., None] * ab[None]
        out[i:i + step] = np.sqrt((d * d).sum(axis=2).min(axis=1))
    return out


def path_polyline(cubs, n=129):
    t = np.linspace(0, 1, n)
    return np.concatenate([cubic_eval(cb, t) for cb in cubs], axis=0)


# ------------------------------------------------------------------ winding numbers
def arcs_to_lines(xy, angle, n=12):
    """Tessellate arc records (end points + signed turning angle) into n chords each."""
    xy = np.asarray(xy, dtype=np.float64)
    angle = np.asarray(angle, dtype=np.float64)
    p0, p1 = xy[:, 0:2], xy[:, 2:4]
    ch = p1 - p0
    out = np.zeros((len(xy), n, 4))
    small = np.abs(angle) < 1e-9
    th = np.where(small, 1.0, angle)
    # centre = midpoint + perp(ch) / (2 tan(th/2)); points rotate about it by th * k / n
    perp = np.stack([-ch[:, 1], ch[:, 0]], axis=1)
    cen = p0 + 0.5 * ch + perp * (0.5 / np.tan(0.5 * th))[:, None]
    r0 = p0 - cen
    for k in range(n + 1):
        a = th * k / n
        ca, sa = np.cos(a), np.sin(a)
        pk = cen + np.stack([ca * r0[:, 0] - sa * r0[:, 1], sa * r0[:, 0] + ca * r0[:, 1]], axis=1)
        pk = np.where(small[:, None], p0 + ch * (k / n), pk)
        if k == n:
            pk = p1
        if k < n:
            out[:, k, 0:2] = pk
        if k > 0:
            out[:, k - 1, 2:4] = pk
    return out.reshape(-1, 4)


def winding_numbers(x, lines):
    """Winding number of each point x[S,2] w.r.t. directed segments lines[M,4] (signed ray crossings)."""
    x = np.asarray(x, dtype=np.float64)
    l = np.asarray(lines, dtype=np.float64)
    x0, y0, x1, y1 = l[:, 0], l[:, 1], l[:, 2], l[:, 3]
    out = np.zeros(len(x), dtype=np.int64)
    step = max(1, int(4e6 // max(1, len(l))))
    for i in range(0, len(x), step):
        px = x[i:i + step, 0, None]
        py = x[i:i + step, 1, None]
        up = (y0[None] <= py) & (py < y1[None])
        dn = (y1[None] <= py) & (py < y0[None])
        side = (x1 - x0)[None] * (py - y0[None]) - (px - x0[None]) * (y1 - y0)[None]
        out[i:i + step] = (up & (side > 0)).sum(axis=1) - (dn & (side < 0)).sum(axis=1)
    return out


# ------------------------------------------------------------------ offset accuracy
def offset_vertex_errors(cb, eta, verts):
    """distance of each vertex to the true parallel curve of cubic cb at signed offset eta."""
    return dist_points_to_polyline(verts, true_offset_polyline(cb, eta))


def check_offsets(scene_cubics, halfw_of_seg, xy, kind, seg, angle=None, segs=None, midpoints=True):
    """Max distance from offset-record vertices (and chord / arc mid-points) to the true parallel curve,
    over the given source segments.  Returns (max_vertex_err, max_mid_err)."""
    kind = np.asarray(kind)
    seg = np.asarray(seg)
    k3 = kind & 7
    is_off = (k3 == K_OFFSET) | (k3 == K_OFFSET_REV)
    vmax = mmax = 0.0
    if segs is None:
        segs = np.unique(seg[is_off])
    for s in segs:
        for plus in (0, 1):
            m = is_off & (seg == s) & (((kind & K_PLUS) != 0) == bool(plus))
            if not m.any():
                continue
            eta = halfw_of_seg[s] * (1 if plus else -1)
            poly = true_offset_polyline(scene_cubics[s], eta)
            r = np.asarray(xy[m], dtype=np.float64)
            v = np.concatenate([r[:, 0:2], r[:, 2:4]])
            vmax = max(vmax, float(dist_points_to_polyline(v, poly).max()))
            if midpoints:
                if angle is not None:
                    sub = arcs_to_lines(r, np.asarray(angle)[m], n=2)
                    mid = sub[0::2, 2:4]
                else:
                    mid = 0.5 * (r[:, 0:2] + r[:, 2:4])
                mmax = max(mmax, float(dist_points_to_polyline(mid, poly).max()))
    return vmax, mmax


def greedy_min_segments(poly, tol):
    """Greedy longest-chord flattening of a dense polyline: fewest chords with max deviation <= tol
    (brute force; tiny inputs only)."""
    n, i, count = len(poly), 0, 0
    while i < n - 1:
        lo, hi = i + 1, n - 1
        # deviation is monotone enough for curves of monotone curvature: binary search the farthest j
        def ok(j):
            return dist_points_to_polyline(poly[i:j + 1], poly[[i, j]]).max() <= tol
        if ok(hi):
            j = hi
        else:
            while hi - lo > 1:
                mid = (lo + hi) // 2
                if ok(mid):
                    lo = mid
                else:
                    hi = mid
            j = lo
        count += 1
        i = j
    return count
