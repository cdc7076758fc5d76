"""Pins for the oracle's whole-outline behaviour: tag walk by brute force, closed forms for lines,
joins, caps and circular arcs, and the strong-correctness / tolerance / watertightness invariants."""
import os

import numpy as np
import pytest

import oracle
from oracle import checkers as ck
from paper_2405_00127_b200 import scenes as S

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def run(sc, mode=0):
    return oracle.expand(sc.tags, sc.points, sc.styles, sc.affine, sc.tolerance, mode)


def recs(r):
    return [tuple(np.round(x, 4)) for x in r.xy.astype(float)]


# ---------------------------------------------------------------- tag walk (L464-470, Table 1)
def test_tag_walk_hand_built_stream():
    # path 0: subpath A = line, cubic(end); subpath B = quad(end, path end).  path 1: line(end,path end, closed)
    tags = np.array([1, 3 | 4, 2 | 4 | 16, 1 | 4 | 16 | 128], dtype=np.uint8)
    n_pts = (1 + 1 + 3) + (1 + 2) + (1 + 1)
    pt, pa, fi = (np.zeros(4, np.uint32) for _ in range(3))
    rc = oracle.lib().so_tag_walk(tags.ctypes.data, 4, n_pts, 2, pt.ctypes.data, pa.ctypes.data, fi.ctypes.data)
    assert rc == 0
    assert pt.tolist() == [0, 1, 5, 8]      # shared end points inside a subpath, +1 at each subpath end (L470)
    assert pa.tolist() == [0, 0, 0, 1]
    assert fi.tolist() == [0, 0, 2, 3]


@pytest.mark.parametrize("bad", ["zero_count", "bit3", "no_path_end", "pts", "paths"])
def test_tag_walk_rejects_bad_streams(bad):
    tags = np.array([1, 3 | 4 | 16], dtype=np.uint8)
    n_pts, n_paths = 5, 1
    if bad == "zero_count":
        tags[0] = 0
    elif bad == "bit3":
        tags[0] |= 8
    elif bad == "no_path_end":
        tags[1] = 3 | 4
    elif bad == "pts":
        n_pts = 6
    else:
        n_paths = 2
    z = np.zeros(2, np.uint32)
    assert oracle.lib().so_tag_walk(tags.ctypes.data, 2, n_pts, n_paths, z.ctypes.data, z.ctypes.data, z.ctypes.data) == -2


def test_tag_walk_matches_generator_identity():
    """point-count identity sum(count + end) = n_points on a generated scene (L470)."""
    sc = S.make("c2", n_paths=50)
    r = run(sc)
    cnt = sc.tags & 3
    end = ((sc.tags >> 2) | (sc.tags >> 4)) & 1
    assert int((cnt + end).sum()) == len(sc.points)
    assert np.array_equal(r.pt_off, (np.cumsum(cnt + end) - (cnt + end)).astype(np.uint32))


# ---------------------------------------------------------------- closed forms: lines, joins, caps
def test_single_line_butt_is_the_rectangle():
    sc = S.from_paths([dict(start=[10, 20], segs=[[[50, 20]]], width=4.0, cap=S.CAP_BUTT)])
    r = run(sc)
    # N = (0,1): -h side (y=18) forward, +h side (y=22) backward, end cap up, start cap down
    assert recs(r) == [(10, 18, 50, 18), (50, 22, 10, 22), (50, 18, 50, 22), (10, 22, 10, 18)]
    assert ck.watertight_violations(r.xy, r.path_off) == 0


def test_square_cap_extends_by_half_width():
    sc = S.from_paths([dict(start=[0, 0], segs=[[[10, 0]]], width=2.0, cap=S.CAP_SQUARE)])
    r = run(sc)
    assert recs(r)[2:5] == [(10, -1, 11, -1), (11, -1, 11, 1), (11, 1, 10, 1)]
    assert recs(r)[5:8] == [(0, 1, -1, 1), (-1, 1, -1, -1), (-1, -1, 0, -1)]


def test_bevel_and_inner_join_left_turn():
    # right angle, left turn at (10,0): outer side is -h; inner (+h) side goes through the vertex (strong correctness)
    sc = S.from_paths([dict(start=[0, 0], segs=[[[10, 0]], [[10, 10]]], width=2.0, join=S.JOIN_BEVEL)])
    r = run(sc)
    rr = recs(r)
    assert rr[2] == (10, -1, 11, 0) and r.kind[2] == ck.K_JOIN_OUTER
    assert rr[3] == (9, 10 - 10, 10, 0) or rr[3] == (9, 0, 10, 0)
    assert rr[3:5] == [(9, 0, 10, 0), (10, 0, 10, 1)]
    assert (r.kind[3] & 7) == ck.K_JOIN_INNER and (r.kind[3] & 8)
    assert ck.watertight_violations(r.xy, r.path_off) == 0


def test_miter_tip_and_limit():
    # 90 degree turn: miter ratio 1/sin(45deg) = 1.414 <= 4: tip at distance h*sqrt(2) on the outer side
    sc = S.from_paths([dict(start=[0, 0], segs=[[[10, 0]], [[10, 10]]], width=2.0, join=S.JOIN_MITER, miter_limit=4.0)])
    rr = recs(run(sc))
    assert rr[2:4] == [(10, -1, 11, -1), (11, -1, 11, 0)]
    # limit 1.2 < 1.414: falls back to a bevel (one record)
    sc = S.from_paths([dict(start=[0, 0], segs=[[[10, 0]], [[10, 10]]], width=2.0, join=S.JOIN_MITER, miter_limit=1.2)])
    rr = recs(run(sc))
    assert rr[2] == (10, -1, 11, 0)
    # right turn mirrors: outer side is +h, emitted backward
    sc = S.from_paths([dict(start=[0, 0], segs=[[[10, 0]], [[10, -10]]], width=2.0, join=S.JOIN_MITER)])
    rr = recs(run(sc))
    assert rr[2:4] == [(10, -1, 10, 0), (10, 0, 9, 0)]           # -h side is inner now
    assert rr[4:6] == [(11, 0, 11, 1), (11, 1, 10, 1)]           # +h side: B' -> tip -> A'


def test_round_cap_and_join_counts_follow_exact_arc_metric():
    """L65-69 exact metric, values in tests/golden/arc_flatten_counts.txt; TOL_FL = 0.8 tol (R-13)."""
    rows = [l.split() for l in open(os.path.join(GOLD, "arc_flatten_counts.txt")) if l.strip() and not l.startswith("#")]
    (r1, a1, d1, n1, s1), (r2, a2, d2, n2, s2) = [[float(v) for v in row] for row in rows]
    assert s1 >= n1 and s2 >= n2   # small-angle form is conservative (L73)
    # half circle R=10: round cap of a width-20 line, flatten tolerance d=0.25 <=> user tol 0.3125
    sc = S.from_paths([dict(start=[0, 0], segs=[[[40, 0]]], width=2 * r1, cap=S.CAP_ROUND)], tolerance=d1 / 0.8)
    r = run(sc)
    assert int((r.kind == ck.K_CAP).sum()) == 2 * int(np.ceil(n1))
    # vertices of the cap lie on the circle, uniformly spaced
    cap = r.xy[r.kind == ck.K_CAP][: int(np.ceil(n1))].astype(float)
    assert np.allclose(np.hypot(cap[:, 0] - 40, cap[:, 1]), r1, atol=1e-4)
    ang = np.unwrap(np.arctan2(cap[:, 1], cap[:, 0] - 40))
    assert np.allclose(np.diff(ang), np.pi / np.ceil(n1), atol=1e-5)
    # quarter circle R=50: round join of a 90 degree turn, width 100
    sc = S.from_paths([dict(start=[0, 0], segs=[[[200, 0]], [[200, 200]]], width=2 * r2, join=S.JOIN_ROUND)], tolerance=d2 / 0.8)
    r = run(sc)
    assert int(((r.kind & 7) == ck.K_JOIN_OUTER).sum()) == int(np.ceil(n2))
    # arc mode: quarter turn is one arc record with angle +pi/2, half-circle cap is two records of pi/2
    r = run(sc, mode=1)
    j = (r.kind & 7) == ck.K_JOIN_OUTER
    assert j.sum() == 1 and abs(r.angle[j][0] - np.pi / 2) < 1e-6


def test_closed_triangle_is_watertight_and_has_three_joins():
    sc = S.from_paths([dict(start=[0, 0], segs=[[[30, 0]], [[15, 20]], [[0, 0]]], closed=True, width=3.0, join=S.JOIN_MITER)])
    r = run(sc)
    assert ck.watertight_violations(r.xy, r.path_off) == 0
    assert (r.kind == ck.K_CAP).sum() == 0
    assert r.seg_count.tolist() == [2 + 4, 2 + 4, 2 + 4]   # 2 offsets + (2 miter + 2 inner) each


def test_zero_width_path_emits_nothing():
    sc = S.from_paths([dict(start=[0, 0], segs=[[[30, 0]]], width=0.0), dict(start=[0, 5], segs=[[[30, 5]]], width=2.0)])
    r = run(sc)
    assert r.seg_count.tolist() == [0, 4] and r.path_off.tolist() == [0, 0, 4]


def test_affine_scales_width_and_maps_points():
    # uniform scale 2 + translation: same outline as stroking the mapped path with twice the width (R-14)
    a = S.from_paths([dict(start=[1, 2], segs=[[[5, 2]], [[5, 7], [9, 9], [12, 3]]], width=1.5, join=S.JOIN_ROUND, cap=S.CAP_ROUND)],
                     affine=[2, 0, 0, 2, 10, -4])
    b = S.from_paths([dict(start=[12, 0], segs=[[[20, 0]], [[20, 10], [28, 14], [34, 2]]], width=3.0, join=S.JOIN_ROUND, cap=S.CAP_ROUND)])
    ra, rb = run(a), run(b)
    assert ra.n_rec == rb.n_rec and np.allclose(ra.xy, rb.xy, atol=1e-5)


# ---------------------------------------------------------------- circular arcs: exact offsets
def _arc_cubic(R, a0, a1):
    """standard cubic approximation of a circular arc (handle 4/3 tan(a/4) R)."""
    k = 4 / 3 * np.tan((a1 - a0) / 4) * R
    p0 = R * np.array([np.cos(a0), np.sin(a0)]); p3 = R * np.array([np.cos(a1), np.sin(a1)])
    t0 = np.array([-np.sin(a0), np.cos(a0)]); t1 = np.array([-np.sin(a1), np.cos(a1)])
    return p0, [p0 + k * t0, p3 - k * t1, p3]


@pytest.mark.parametrize("R,w,mode", [(100.0, 10.0, 0), (100.0, 10.0, 1), (30.0, 40.0, 0)])
def test_circular_arc_offsets_are_concentric(R, w, mode):
    """The parallel curves of a circle are circles (closed form): every offset vertex is at R -/+ h from the
    centre within the ES-fit tolerance, and the line count follows n = s sqrt(kappa/(8d)) (L73)."""
    p0, seg = _arc_cubic(R, 0.0, np.pi / 3)
    sc = S.from_paths([dict(start=p0 + 500, segs=[[q + 500 for q in seg]], width=w)])
    r = run(sc, mode)
    off = (r.kind & 7) == ck.K_OFFSET
    minus = off & ((r.kind & 8) == 0)
    plus = off & ((r.kind & 8) != 0)
    # CCW arc: left normal points to the centre, so the +h side is the inner circle
    for m, rad in ((minus, R + w / 2), (plus, R - w / 2)):
        v = r.xy[m].astype(float).reshape(-1, 2) - 500
        assert np.abs(np.hypot(v[:, 0], v[:, 1]) - rad).max() < 0.03
    if mode == 0:
        for m, rad in ((minus, R + w / 2), (plus, R - w / 2)):
            s = rad * np.pi / 3
            n_pred = s * np.sqrt(1 / rad / (8 * 0.2))
            assert np.ceil(n_pred) <= m.sum() <= np.ceil(n_pred) + r.stats["pieces"]
    else:
        # an arc is its own best approximation: one arc record per ES piece and side, turning = piece angle
        assert minus.sum() == r.stats["pieces"]
        assert abs(r.angle[minus].sum() - np.pi / 3) < 1e-4 and abs(r.angle[plus].sum() + np.pi / 3) < 1e-4


def test_tight_arc_is_supercritical_with_evolute_at_centre():
    """R < h: the +h (inner) side is super-critical everywhere: reversed offset + evolute (the centre, L193:
    evolute of a circle is a point) + connectors, each of the latter twice (L197)."""
    R, w = 10.0, 30.0
    p0, seg = _arc_cubic(R, 0.0, np.pi / 2)
    sc = S.from_paths([dict(start=p0 + 100, segs=[[q + 100 for q in seg]], width=w)])
    r = run(sc)
    k3 = r.kind & 7
    ev = r.xy[k3 == ck.K_EVOLUTE].astype(float).reshape(-1, 2) - 100
    assert len(ev) > 0 and np.abs(ev).max() < 0.05
    assert (k3 == ck.K_EVOLUTE).sum() % 2 == 0 and (k3 == ck.K_CONNECTOR).sum() == 4 * r.stats["pieces"]
    assert (k3 == ck.K_OFFSET_REV).sum() > 0 and ((r.kind[k3 == ck.K_OFFSET_REV] & 8) != 0).all()
    assert ck.watertight_violations(r.xy, r.path_off) == 0


# ---------------------------------------------------------------- invariants on generated scenes
def _winding_band(sc, r, paths, rng, mode, n_pts=1500, margin=0.03):
    cubs = ck.segment_cubics(sc.tags, sc.points, sc.affine)
    det = abs(float(sc.affine[0]) * float(sc.affine[3]) - float(sc.affine[1]) * float(sc.affine[2]))
    tol = sc.tolerance
    stats = dict(neg=0, inside_fail=0, outside_fail=0, inside=0, outside=0)
    for p in paths:
        a, b = int(r.path_off[p]), int(r.path_off[p + 1])
        lines = r.xy[a:b] if mode == 0 else ck.arcs_to_lines(r.xy[a:b], r.angle[a:b])
        segs = np.flatnonzero(r.path_idx == p)
        st = sc.styles[p]
        h = 0.5 * float(st["width"]) * np.sqrt(det)
        poly = ck.path_polyline(cubs[segs], n=257)
        # candidate points just inside / outside the true boundary: C(s) +- (h -/+ (tol+margin)) N(s)
        si = rng.integers(0, len(segs), n_pts)
        tt = rng.uniform(0, 1, n_pts)
        P = np.stack([ck.cubic_eval(cubs[segs[i]], [t])[0] for i, t in zip(si, tt)])
        D = np.stack([ck.cubic_deriv(cubs[segs[i]], [t])[0] for i, t in zip(si, tt)])
        nrm = np.hypot(D[:, 0], D[:, 1])
        ok = nrm > 1e-9
        N = np.stack([-D[ok, 1], D[ok, 0]], 1) / nrm[ok, None]
        sgn = rng.choice([-1.0, 1.0], ok.sum())[:, None]
        rad = np.where(rng.uniform(size=ok.sum()) < 0.5, h - tol - margin, h + tol + margin)[:, None]
        X = np.concatenate([P[ok] + sgn * rad * N, rng.uniform(poly.min(0) - 1.5 * h - 2, poly.max(0) + 1.5 * h + 2, (n_pts // 3, 2))])
        w = ck.winding_numbers(X, lines)
        d = ck.dist_points_to_polyline(X, poly)
        stats["neg"] += int((w < 0).sum())
        round_all = st["join"] == S.JOIN_ROUND and (st["cap"] == S.CAP_ROUND or (sc.tags[segs[-1]] & 128))
        ends = np.stack([poly[0], poly[-1]])
        de = np.minimum(np.hypot(*(X - ends[0]).T), np.hypot(*(X - ends[1]).T))
        closed = bool(sc.tags[segs[-1]] & 128)
        # inside: within h - tol of the path (and, for non-round caps on open paths, not within the end discs)
        inside = (d < h - tol - margin / 2)
        if not closed and st["cap"] != S.CAP_ROUND:
            inside &= de > h + 1e-6
        if not round_all:
            # joins other than round cover at least the bevel triangle, not the full disc: test sweep interiors only
            verts = np.stack([cubs[s][0] for s in segs] + [cubs[segs[-1]][3]])
            dv = np.sqrt(((X[:, None] - verts[None]) ** 2).sum(2)).min(1)
            inside &= dv > h + 1e-6
        kmax = 1.0
        if st["join"] == S.JOIN_MITER:
            kmax = max(kmax, float(st["miter_limit"]))
        if st["cap"] == S.CAP_SQUARE and not closed:
            kmax = max(kmax, np.sqrt(2))
        outside = d > kmax * h + tol + margin / 2
        stats["inside"] += int(inside.sum()); stats["outside"] += int(outside.sum())
        stats["inside_fail"] += int((w[inside] < 1).sum())
        stats["outside_fail"] += int((w[outside] != 0).sum())
    return stats


@pytest.mark.parametrize("name,npaths,mode", [("c1", 64, 0), ("c2", 240, 0), ("c2", 240, 1), ("c3", 300, 0), ("c4", 200, 1), ("c5", 12, 0), ("c5", 12, 1)])
def test_invariants_on_generated_scenes(name, npaths, mode):
    """Strong correctness (L29-35, L191, L197): winding never negative, >= 1 within h - tol of the path, 0 beyond
    h + tol; watertight; every vertex within K h + tol of the path."""
    sc = S.make(name, n_paths=npaths)
    r = run(sc, mode)
    assert np.isfinite(r.xy).all() and np.isfinite(r.angle).all()
    assert ck.watertight_violations(r.xy, r.path_off) == 0
    rng = np.random.default_rng(123)
    paths = rng.choice(npaths, size=min(npaths, 10), replace=False)
    st = _winding_band(sc, r, paths, rng, mode)
    assert st["inside"] > 500 and st["outside"] > 500
    assert st["neg"] == 0, st
    assert st["inside_fail"] == 0 and st["outside_fail"] == 0, st


def test_vertices_within_halfwidth_plus_tol_of_path():
    sc = S.make("c1", n_paths=24)
    r = run(sc)
    cubs = ck.segment_cubics(sc.tags, sc.points, sc.affine)
    for p in range(24):
        a, b = int(r.path_off[p]), int(r.path_off[p + 1])
        segs = np.flatnonzero(r.path_idx == p)
        poly = ck.path_polyline(cubs[segs], n=1025)
        h = 0.5 * float(sc.styles[p]["width"])
        v = r.xy[a:b].astype(float).reshape(-1, 2)
        assert ck.dist_points_to_polyline(v, poly).max() <= h + sc.tolerance


def test_offset_records_track_true_parallel_curve_on_tame_segments():
    """Frechet-type tolerance (L37): on segments whose curvature stays below 2/h the offset vertices lie within
    the ES-fit budget of the true parallel curve and chord mid-points within tol (a 0.1% tail is allowed up to
    1.2 tol: the line metric L77 and f_approx L145 are approximations)."""
    sc = S.make("c1", n_paths=32)
    r = run(sc)
    cubs = ck.segment_cubics(sc.tags, sc.points, sc.affine)
    halfw = 0.5 * sc.styles["width"][r.path_idx]
    k3 = r.kind & 7
    mids, verts = [], []
    for sg in range(sc.n_segments):
        cb, h = cubs[sg], float(halfw[sg])
        t = np.linspace(0, 1, 2001)
        d = ck.cubic_deriv(cb, t)
        dd = 6 * ((1 - t)[:, None] * (cb[2] - 2 * cb[1] + cb[0]) + t[:, None] * (cb[3] - 2 * cb[2] + cb[1]))
        kap = (d[:, 0] * dd[:, 1] - d[:, 1] * dd[:, 0]) / np.hypot(d[:, 0], d[:, 1]) ** 3
        if np.abs(kap).max() * h >= 2.0:
            continue
        for plus in (0, 1):
            m = (r.seg == sg) & (k3 == ck.K_OFFSET) & (((r.kind & 8) != 0) == bool(plus))
            poly = ck.true_offset_polyline(cb, h if plus else -h)
            rr = r.xy[m].astype(float)
            verts.append(ck.dist_points_to_polyline(rr[:, 0:2], poly))
            mids.append(ck.dist_points_to_polyline(0.5 * (rr[:, 0:2] + rr[:, 2:4]), poly))
    verts, mids = np.concatenate(verts), np.concatenate(mids)
    assert len(mids) > 3000
    assert verts.max() < 0.05                      # ES fit tolerance 0.1 tol = 0.025 px plus normal-direction error
    assert mids.max() < 1.2 * sc.tolerance and np.mean(mids > sc.tolerance) < 2e-3
    assert np.quantile(mids, 0.99) > 0.5 * sc.tolerance   # near-minimal: the budget is actually used (L37)


def test_offset_chain_is_continuous_in_t_order():
    """Alg. 2's two-word stack (L444) visits sub-ranges left to right: on a fully regular cubic the -h side
    offset records of consecutive pieces chain end-to-start from the segment's first to last offset point."""
    sc = S.from_paths([dict(start=[100, 100], segs=[[[150, 260], [330, -40], [400, 120]]], width=4.0)])
    r = run(sc)
    m = (r.kind == ck.K_OFFSET)
    a = r.xy[m]
    assert r.stats["pieces"] >= 4 and r.stats["ranges_sup"] == 0
    assert np.array_equal(a[1:, 0:2], a[:-1, 2:4])
    p = (r.kind == (ck.K_OFFSET | ck.K_PLUS))
    # +h side records are emitted per piece, mirrored: as a set they chain backward
    assert ck.watertight_violations(r.xy, r.path_off) == 0 and p.sum() > 0


def test_line_counts_within_factor_of_greedy_minimum():
    """L37/L73: 'near-minimal'.  Brute force: greedy longest-chord flattening of the true parallel curve at the
    same flatten tolerance; the oracle may use at most 1.5x that plus one per ES piece (per-piece round-up)."""
    for seg, w in [([[140, 220], [300, 60], [420, 240]], 12.0), ([[60, 300], [260, 340], [300, 20]], 30.0)]:
        sc = S.from_paths([dict(start=[20, 40], segs=[seg], width=w)])
        r = run(sc)
        cubs = ck.segment_cubics(sc.tags, sc.points, sc.affine)
        if r.stats["ranges_sup"]:
            continue
        for plus in (0, 1):
            m = (r.kind & 7 == ck.K_OFFSET) & (((r.kind & 8) != 0) == bool(plus))
            poly = ck.true_offset_polyline(cubs[0], (w / 2) if plus else (-w / 2), n0=4001)
            g = ck.greedy_min_segments(poly, 0.8 * sc.tolerance)
            assert g <= m.sum() <= 1.5 * g + r.stats["pieces"], (g, m.sum(), r.stats)
