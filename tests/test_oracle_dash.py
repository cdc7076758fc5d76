"""Pins for dashing in the oracle ("the core algorithm is prefix sum applied to
segment length, and the Euler spiral representation is particularly well suited"; reading R-23 of DESIGN.md).

Measured against things the oracle does not compute: hand-placed dashes on straight paths, the true arc length of the
source cubics (Gauss-Legendre on |C'(t)|), the area of a strip of constant width (length x width, whatever the curvature)."""
from collections import Counter

import numpy as np
import pytest

import oracle
from oracle import checkers as ck
from paper_2405_00127_b200 import scenes as S

K_OFFSET, K_JOIN_OUTER, K_JOIN_INNER, K_CAP, K_PLUS = 0, 4, 5, 6, 8


def run(sc, dash, phase=0.0, mode=0):
    return oracle.expand(sc.tags, sc.points, sc.styles, sc.affine, sc.tolerance, mode, dash=dash, phase=phase)


def dash_intervals(total, dash, phase):
    """[(a, b)] of the dashes of a subpath of arc length `total` (the definition, written out once more, in floating point)."""
    out, pos, j = [], -float(phase), 0
    while pos < total:
        ln = dash[j % len(dash)]
        if j % 2 == 0 and pos + ln > 0:
            out.append((max(pos, 0.0), min(pos + ln, total)))
        pos += ln
        j += 1
    return [(a, b) for a, b in out if b > a]


def bits(a):
    return Counter(map(tuple, np.ascontiguousarray(a, dtype=np.float32).view(np.uint32).reshape(len(a), -1)))


def test_straight_path_hand_placed_dashes():
    """A horizontal line of length 100, width 4, pattern 10 on / 5 off, phase 3: dashes [0,7] [12,22] [27,37] ... [87,97];
    each is the rectangle [a,b] x [-2,2] as four records: start cap, -h side, +h side, end cap (butt caps)."""
    sc = S.with_dash(S.from_paths([dict(start=[0, 0], segs=[[[100, 0]]], width=4.0)]))
    r = run(sc, [10, 5], 3.0)
    want = dash_intervals(100.0, [10, 5], 3.0)
    assert want[0] == (0.0, 7.0) and want[-1] == (87.0, 97.0) and len(want) == 7
    assert r.n_rec == 4 * len(want)
    for k, (a, b) in enumerate(want):
        q = r.xy[4 * k:4 * k + 4]
        assert np.allclose(q, np.array([[a, 2, a, -2], [a, -2, b, -2], [b, 2, a, 2], [b, -2, b, 2]]), rtol=0, atol=1e-5), (k, q)   # (t = a / 100 in fp32)
        assert r.kind[4 * k:4 * k + 4].tolist() == [K_CAP, K_OFFSET, K_OFFSET | K_PLUS, K_CAP]
    # a dash that reaches the end of the path ends there: phase 0 -> [90, 100]
    r = run(sc, [10, 5], 0.0)
    assert np.array_equal(r.xy[-1], np.array([100, -2, 100, 2], np.float32)) and r.n_rec == 4 * 7      # (an uncut end: exact)
    # round and square caps: the same dashes with more cap records; the cap extends beyond the dash by h
    for cap, per_cap in ((S.CAP_SQUARE, 3), (S.CAP_ROUND, None)):
        sc2 = S.with_dash(S.from_paths([dict(start=[0, 0], segs=[[[100, 0]]], width=4.0, cap=cap)]))
        r2 = run(sc2, [10, 5], 3.0)
        assert int((r2.kind == K_OFFSET).sum()) == 7 and ck.watertight_violations(r2.xy, r2.path_off) == 0
        assert abs(float(r2.xy[:, [0, 2]].min()) + 2.0) < 1e-6 and abs(float(r2.xy[:, [0, 2]].max()) - 99.0) < 1e-6
        if per_cap:
            assert int(((r2.kind & 7) == K_CAP).sum()) == 2 * 7 * per_cap


def test_pattern_algebra():
    """The pattern is periodic (phase + period changes nothing), [a, b] is the same pattern as [a, b, a, b], and a pattern that
    is on over the whole path gives exactly the records of the undashed open stroke (as a multiset: caps move within the
    order), joins included."""
    base = S.make("c1", n_paths=6)
    sc = S.with_dash(base)
    r1 = run(sc, [17.5, 6.25], 4.0)
    r2 = run(sc, [17.5, 6.25], 4.0 + 23.75)
    r3 = run(sc, [17.5, 6.25, 17.5, 6.25], 4.0)
    assert np.array_equal(r1.xy.view(np.uint32), r2.xy.view(np.uint32)) and np.array_equal(r1.xy.view(np.uint32), r3.xy.view(np.uint32))
    opened = S.Scene(base)
    opened["tags"] = base.tags & ~np.uint8(128)          # the same paths, not closed: the undashed stroke has caps
    plain = oracle.expand(opened.tags, opened.points, opened.styles, opened.affine, opened.tolerance, 0)
    full = run(S.with_dash(opened), [1e6, 1.0], 0.0)
    assert full.n_rec == plain.n_rec and bits(full.xy) == bits(plain.xy)
    # ... and a pattern that is off over the whole path emits nothing
    none = run(S.with_dash(opened), [1.0, 1e6], 2.0)
    assert none.n_rec == 0


def test_joins_only_inside_dashes():
    """An L-shaped polyline, corner at arc length 50: a dash that covers the corner carries the join, a gap over the corner
    leaves it out, and a dash that ends exactly at the corner is capped there."""
    sc = S.with_dash(S.from_paths([dict(start=[0, 0], segs=[[[50, 0]], [[50, 50]]], width=6.0, join=S.JOIN_BEVEL)]))
    joins = lambda r: int(np.isin(r.kind & 7, [K_JOIN_OUTER, K_JOIN_INNER]).sum())
    assert any(a < 50 < b for a, b in dash_intervals(100.0, [20, 20], 0.0))       # dashes [0,20] [40,60] [80,100]: one covers the corner
    r = run(sc, [20, 20], 0.0)
    assert joins(r) == 3 and ck.watertight_violations(r.xy, r.path_off) == 0       # bevel: one outer record, two inner
    assert joins(run(sc, [20, 20], 10.0)) == 0                                      # dashes [0,10] [30,50] [70,90]: one ENDS at the corner
    r = run(sc, [20, 20], 30.0)                           # dashes [10,30] [50,70] [90,100]: the corner starts a dash
    assert not any(a < 50 < b for a, b in dash_intervals(100.0, [20, 20], 30.0))
    assert joins(r) == 0 and ck.watertight_violations(r.xy, r.path_off) == 0
    r = run(sc, [20, 20], 20.0)                           # dashes [20,40] [60,80]: the corner in a gap
    assert joins(r) == 0
    r = run(sc, [25, 25], 0.0)                            # dashes [0,25] [50,75]: the second STARTS at the corner
    assert joins(r) == 0 and int(((r.kind & 7) == K_CAP).sum()) == 4
    r = run(sc, [50, 25], 0.0)                            # dashes [0,50] [75,100]: the first ENDS at the corner: cap there, no join
    assert joins(r) == 0 and int(((r.kind & 7) == K_CAP).sum()) == 4
    caps = r.xy[(r.kind & 7) == K_CAP]
    assert any(np.array_equal(c, np.array([50, -3, 50, 3], np.float32)) for c in caps)


def cubic_length(cb, n=64):
    x, w = np.polynomial.legendre.leggauss(n)
    t = 0.5 * (x + 1.0)
    d = ck.cubic_deriv(cb, t)
    return 0.5 * float(np.sum(w * np.hypot(d[:, 0], d[:, 1])))


def arc_positions(cubs, pts, max_step):
    """Arc length (along the chain of cubics, measured on a dense sampling) of the points pts of the chain, given in the order
    they follow each other along it, no further apart than max_step (the paths cross themselves: the search moves forward)."""
    poly = ck.path_polyline(cubs, n=16385)               # (per cubic: samples ~0.02 px apart)
    seg = np.hypot(*np.diff(poly, axis=0).T)
    cum = np.concatenate([[0.0], np.cumsum(seg)])
    out, prev = [], 0.0
    for p in pts:
        lo, hi = np.searchsorted(cum, prev - 0.25), np.searchsorted(cum, prev + max_step + 0.5)
        d = np.hypot(poly[lo:hi, 0] - p[0], poly[lo:hi, 1] - p[1])
        i = lo + int(np.argmin(d))
        assert d[i - lo] < 0.06, (d[i - lo], prev)        # (the Euler-spiral fit budget, as in test_oracle_outline: 0.05 px; plus the sampling)
        prev = cum[i]
        out.append(prev)
    return np.array(out), cum[-1]


@pytest.mark.parametrize("mode", [0, 1])
def test_dash_ends_sit_at_the_pattern_positions_of_the_true_arc_length(mode):
    """Curved open paths (config 1's cubics, opened; butt caps): the cap records are chords through the path at the dash ends.
    Their mid-points, located on the TRUE curve, sit at the arc lengths the pattern asks for -- the Euler-spiral pieces carry
    the arc length of the cubic to within the fit tolerance -- and there are as many dashes as the true length gives."""
    base = S.make("c1", n_paths=5)
    sc = S.Scene(base)
    sc["tags"] = base.tags & ~np.uint8(128)
    st = sc["styles"].copy(); st["cap"] = S.CAP_BUTT; st["width"] = 3.0
    sc["styles"] = st
    sc = S.with_dash(sc)
    dash, phase = [21.0, 9.5, 4.0, 9.5], 13.0
    r = run(sc, dash, phase, mode)
    assert ck.watertight_violations(r.xy, r.path_off) == 0
    cubs = ck.segment_cubics(sc.tags, sc.points, sc.affine)
    worst = 0.0
    for p in range(5):
        segs = np.flatnonzero(r.path_idx == p)
        a, b = int(r.path_off[p]), int(r.path_off[p + 1])
        caps = r.xy[a:b][(r.kind[a:b] & 7) == K_CAP].astype(np.float64)
        mids = 0.5 * (caps[:, 0:2] + caps[:, 2:4])
        pos, total = arc_positions(cubs[segs], mids, max(dash))
        assert abs(total - sum(cubic_length(cubs[s]) for s in segs)) < 0.02
        want = dash_intervals(total, dash, phase)
        assert len(caps) == 2 * len(want), (p, len(caps), len(want))
        got = pos                                        # (caps come in the order of the dashes: start, end, start, ...)
        exp = np.array(want).ravel()
        worst = max(worst, float(np.abs(got - exp).max()))
    assert worst < 0.1, worst           # px of arc length over paths of ~1000 px (measured 0.055: the pieces carry the arc length to 1e-4)


def test_area_of_the_dashes_is_on_length_times_width():
    """A strip of constant width 2h along a curve has area (length) x (2h) whatever the curvature (no cusps: thin stroke).
    Sum over all records of the shoelace terms = total area of the dash outlines = (sum of the dash lengths) x width."""
    base = S.make("c1", n_paths=4)
    sc = S.Scene(base)
    sc["tags"] = base.tags & ~np.uint8(128)
    st = sc["styles"].copy(); st["cap"] = S.CAP_BUTT; st["width"] = 1.5; st["join"] = S.JOIN_ROUND
    sc["styles"] = st
    sc = S.with_dash(sc)
    dash, phase = [33.0, 14.0], 5.0
    r = run(sc, dash, phase)
    cubs = ck.segment_cubics(sc.tags, sc.points, sc.affine)
    for p in range(4):
        segs = np.flatnonzero(r.path_idx == p)
        a, b = int(r.path_off[p]), int(r.path_off[p + 1])
        q = r.xy[a:b].astype(np.float64)
        area = 0.5 * float(np.sum(q[:, 0] * q[:, 3] - q[:, 2] * q[:, 1]))
        total = sum(cubic_length(cubs[s]) for s in segs)
        on = sum(b2 - a2 for a2, b2 in dash_intervals(total, dash, phase))
        # (round joins inside dashes add their small sectors: at most (turning angle) h^2 / 2 each)
        assert abs(area - on * 1.5) <= 0.01 * on * 1.5 + 0.5 * 0.75 ** 2 * np.pi * len(segs), (p, area, on * 1.5)


def test_splitting_a_segment_does_not_move_the_dashes():
    """The prefix-sum property: the arc length at which a dash starts does not depend on how the path is cut into segments.
    One line of length 240 against the same line in 7 collinear segments of unequal length."""
    one = S.with_dash(S.from_paths([dict(start=[10, 20], segs=[[[250, 20]]], width=2.0)]))
    xs = [25.0, 33.5, 90.25, 91.0, 170.0, 249.0, 250.0]
    many = S.with_dash(S.from_paths([dict(start=[10, 20], segs=[[[x, 20]] for x in xs], width=2.0, join=S.JOIN_BEVEL)]))
    dash, phase = [13.0, 7.0, 2.0, 7.0], 1.0
    r1, r2 = run(one, dash, phase), run(many, dash, phase)
    c1 = r1.xy[(r1.kind & 7) == K_CAP]
    c2 = r2.xy[(r2.kind & 7) == K_CAP]
    assert len(c1) == len(c2) and np.array_equal(np.sort(c1[:, 0]), np.sort(c2[:, 0]))     # bit for bit: lengths are integers in 2^-16 px
    assert ck.watertight_violations(r2.xy, r2.path_off) == 0
    # the dashes of a subpath do not depend on the subpaths before it: the pattern restarts
    two = S.with_dash(S.from_paths([dict(start=[0, 0], segs=[[[37, 0]]], width=2.0), dict(start=[10, 20], segs=[[[250, 20]]], width=2.0)]))
    r3 = run(two, dash, phase)
    a = int(r3.path_off[1])
    assert np.array_equal(r3.xy[a:].view(np.uint32), r1.xy.view(np.uint32))


@pytest.mark.parametrize("name,npaths,mode", [("c1", 24, 0), ("c2", 160, 0), ("c2", 160, 1), ("c5", 4, 0)])
def test_dashed_scenes_are_watertight_and_never_wind_negatively(name, npaths, mode):
    """Every dash is a closed outline (bitwise chains), degenerate segments and evolute patches cut by dash ends included;
    winding numbers are never negative and zero beyond h + tol of the path; only every second path is dashed, the others keep
    their undashed records bit for bit."""
    base = S.make(name, n_paths=npaths)
    sc = S.with_dash(base, every=2, offset=0)
    dash, phase = [26.0, 11.0, 5.0, 11.0], 3.0
    r = run(sc, dash, phase, mode)
    r0 = oracle.expand(base.tags, base.points, base.styles, base.affine, base.tolerance, mode)
    assert np.isfinite(r.xy).all() and ck.watertight_violations(r.xy, r.path_off) == 0
    for p in range(1, npaths, 2):
        a, b, a0, b0 = int(r.path_off[p]), int(r.path_off[p + 1]), int(r0.path_off[p]), int(r0.path_off[p + 1])
        assert np.array_equal(r.xy[a:b].view(np.uint32), r0.xy[a0:b0].view(np.uint32))
    rng = np.random.default_rng(5)
    cubs = ck.segment_cubics(sc.tags, sc.points, sc.affine)
    for p in rng.choice(np.arange(0, npaths, 2), size=min(4, (npaths + 1) // 2), replace=False):
        a, b = int(r.path_off[p]), int(r.path_off[p + 1])
        lines = r.xy[a:b] if mode == 0 else ck.arcs_to_lines(r.xy[a:b], r.angle[a:b])
        segs = np.flatnonzero(r.path_idx == p)
        poly = ck.path_polyline(cubs[segs], n=257)
        h = 0.5 * float(sc.styles[p]["width"])
        X = rng.uniform(poly.min(0) - 1.5 * h - 2, poly.max(0) + 1.5 * h + 2, (800, 2))
        w = ck.winding_numbers(X, lines)
        d = ck.dist_points_to_polyline(X, poly)
        kmax = max(1.0, float(sc.styles[p]["miter_limit"]) if sc.styles[p]["join"] == S.JOIN_MITER else 1.0, np.sqrt(2) if sc.styles[p]["cap"] == S.CAP_SQUARE else 1.0)
        assert (w >= 0).all()
        assert (w[d > kmax * h + sc.tolerance + 0.05] == 0).all()
        assert (w > 0).any()


def test_a_filled_path_is_never_dashed():
    """The pattern applies to stroked paths: a filled path that carries the dash bit, after a dashed stroke in the same call,
    gives the records of the plain fill."""
    base = S.make("c2", n_paths=40)
    filled = S.with_fill(base, every=2, offset=1)
    both = S.with_dash(filled, every=1)
    r = run(both, [9.0, 4.0], 1.0)
    r0 = oracle.expand(filled.tags, filled.points, filled.styles, filled.affine, filled.tolerance, 0)
    for p in range(1, 40, 2):
        a, b, a0, b0 = int(r.path_off[p]), int(r.path_off[p + 1]), int(r0.path_off[p]), int(r0.path_off[p + 1])
        assert np.array_equal(r.xy[a:b].view(np.uint32), r0.xy[a0:b0].view(np.uint32))
    assert int(((r.kind & 7) == K_CAP).sum()) > 0


def edge_scenes():
    """Hand-built paths that stress the position rules: zero-length segments at the start, in the middle and at the end of a
    dashed path, a degenerate cubic, a closed triangle, dashes much shorter than a segment and a pattern longer than the path."""
    z = [40.0, 40.0]
    paths = [
        dict(start=z, segs=[[z], [[90, 40]], [[90, 40]], [[90, 95]], [[90, 95]]], width=5.0, cap=S.CAP_ROUND, join=S.JOIN_ROUND),
        dict(start=[10, 10], segs=[[[10, 10], [10, 10], [10, 10]], [[60, 15], [20, 70], [80, 80]]], width=3.0, cap=S.CAP_SQUARE),
        dict(start=[100, 100], segs=[[[160, 100]], [[130, 150]], [[100, 100]]], width=4.0, closed=True, join=S.JOIN_MITER),
        dict(start=[200, 20], segs=[[[205, 20]]], width=1.0),
        dict(start=[300, 300], segs=[[[340, 380], [420, 260], [460, 340]]], width=30.0, cap=S.CAP_BUTT),
    ]
    return S.with_dash(S.from_paths(paths))


@pytest.mark.parametrize("dash,phase", [([7.0, 3.0], 0.0), ([0.01, 0.02], 0.005), ([1000.0, 5.0], 0.0), ([1000.0, 5.0], 998.0), ([50.0, 50.0], 50.0),
                                        ([2.0 ** -9, 2.0 ** -9], 0.0)])
@pytest.mark.parametrize("mode", [0, 1])
def test_edge_scenes_stay_watertight(dash, phase, mode):
    sc = edge_scenes()
    if dash[0] < 1e-3 and mode == 1:
        pytest.skip("the finest patterns: line mode is enough")
    r = run(sc, dash, phase, mode)
    assert np.isfinite(r.xy).all() and ck.watertight_violations(r.xy, r.path_off) == 0
    # the number of caps is twice the number of dashes; with the pattern longer than every path: one dash or none per subpath
    caps_per_cap = {S.CAP_BUTT: 1, S.CAP_SQUARE: 3}
    if dash[0] >= 1000.0 and phase == 0.0:
        for p in (1, 3, 4):
            a, b = int(r.path_off[p]), int(r.path_off[p + 1])
            assert int(((r.kind[a:b] & 7) == K_CAP).sum()) == 2 * caps_per_cap[int(sc.styles[p]["cap"])]
