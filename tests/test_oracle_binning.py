"""Pins of the tile-binning oracle (oracle/bin_oracle.c, reading R-19 of DESIGN.md) against
what the definition fixes without it: the exact geometry "which 16 x 16 tiles does the segment pass through / touch", evaluated
here in double precision on the fp32 inputs (independently: segment-to-rectangle distance, no row walk), closed forms,
and invariants of the CSR result."""
import numpy as np
import pytest

import oracle

TILE = 16.0


def seg_rect_distance(l, x_lo, y_lo, x_hi, y_hi):
    """Exact-enough (float64) distance between the segment l = (x0, y0, x1, y1) and the closed rectangle: 0 when they meet.
    Liang-Barsky clip for the intersection test; otherwise the minimum over corner-to-segment and end-point-to-rectangle
    distances."""
    x0, y0, x1, y1 = (float(v) for v in l)
    dx, dy = x1 - x0, y1 - y0
    t0, t1 = 0.0, 1.0
    hit = True
    for p, q in ((-dx, x0 - x_lo), (dx, x_hi - x0), (-dy, y0 - y_lo), (dy, y_hi - y0)):
        if p == 0.0:
            if q < 0.0:
                hit = False
                break
        else:
            r = q / p
            if p < 0.0:
                t0 = max(t0, r)
            else:
                t1 = min(t1, r)
            if t0 > t1:
                hit = False
                break
    if hit:
        return 0.0

    def pt_rect(px, py):
        ex = max(x_lo - px, 0.0, px - x_hi)
        ey = max(y_lo - py, 0.0, py - y_hi)
        return float(np.hypot(ex, ey))

    def pt_seg(px, py):
        L2 = dx * dx + dy * dy
        t = 0.0 if L2 == 0.0 else min(1.0, max(0.0, ((px - x0) * dx + (py - y0) * dy) / L2))
        return float(np.hypot(px - (x0 + t * dx), py - (y0 + t * dy)))

    d = min(pt_rect(x0, y0), pt_rect(x1, y1))
    for cx, cy in ((x_lo, y_lo), (x_lo, y_hi), (x_hi, y_lo), (x_hi, y_hi)):
        d = min(d, pt_seg(cx, cy))
    return d


def tiles_of(off, lines_of_tiles, n_lines):
    """per line: the set of tiles it was binned into"""
    sets = [set() for _ in range(n_lines)]
    for t in range(len(off) - 1):
        for i in lines_of_tiles[off[t]:off[t + 1]]:
            sets[int(i)].add(t)
    return sets


def adversarial_lines(rng, n, size):
    """random segments of mixed lengths, a share of them with end points on grid lines / grid corners, horizontal, vertical,
    degenerate (a point), and reaching outside the viewport"""
    a = rng.uniform(-20.0, size + 20.0, (n, 4))
    short = rng.random(n) < 0.6
    a[short, 2:] = a[short, :2] + rng.normal(0.0, 12.0, (int(short.sum()), 2))
    snap = rng.random((n, 4)) < 0.25
    a[snap] = np.round(a[snap] / TILE) * TILE
    hor = rng.random(n) < 0.1
    a[hor, 3] = a[hor, 1]
    ver = rng.random(n) < 0.1
    a[ver, 2] = a[ver, 0]
    pt = rng.random(n) < 0.03
    a[pt, 2:] = a[pt, :2]
    return a.astype(np.float32)


def test_binning_is_conservative_and_tight_against_exact_geometry():
    """Every tile the exact segment passes through (its square shrunk by the rounding room: half-open tiles) is listed -- a
    mistake in the slab clipping, the slope, a min / max or a floor drops tiles -- and every listed tile's closed square is
    within rounding distance of the segment (a transposed coordinate or an unclipped extent adds tiles)."""
    rng = np.random.default_rng(5)
    tx, ty = 20, 14
    lines = adversarial_lines(rng, 1500, 16.0 * 20)
    off, tl = oracle.bin_lines(lines, tx, ty)
    got = tiles_of(off, tl, len(lines))
    eps = 2e-3
    n_exact = 0
    for i, l in enumerate(lines):
        for r in range(ty):
            for c in range(tx):
                t = r * tx + c
                d = seg_rect_distance(l, TILE * c, TILE * r, TILE * c + TILE, TILE * r + TILE)
                # points exactly on the viewport's far edges belong to no tile (indices come from floor())
                inner = seg_rect_distance(l, TILE * c + eps, TILE * r + eps, TILE * c + TILE - eps, TILE * r + TILE - eps)
                if inner == 0.0:
                    assert t in got[i], (i, l, r, c)
                    n_exact += 1
                if t in got[i]:
                    assert d <= eps, (i, l, r, c, d)
    assert n_exact > 3000


def test_binning_closed_forms():
    # a horizontal line across k tiles, strictly inside its row
    off, tl = oracle.bin_lines(np.array([[3.0, 20.0, 3.0 + 16 * 5, 20.0]], np.float32), 8, 4)
    assert np.flatnonzero(np.diff(off)).tolist() == [8 + c for c in range(0, 6)]
    # a vertical line across rows 0..3 in column 2
    off, tl = oracle.bin_lines(np.array([[40.0, 1.0, 40.0, 63.0]], np.float32), 8, 4)
    assert np.flatnonzero(np.diff(off)).tolist() == [2, 10, 18, 26]
    # a point: one tile; a point on a grid corner belongs to the tile floor() names (half-open tiles)
    off, _ = oracle.bin_lines(np.array([[21.0, 37.0, 21.0, 37.0]], np.float32), 8, 4)
    assert np.flatnonzero(np.diff(off)).tolist() == [2 * 8 + 1]
    off, _ = oracle.bin_lines(np.array([[32.0, 32.0, 32.0, 32.0]], np.float32), 8, 4)
    assert np.flatnonzero(np.diff(off)).tolist() == [2 * 8 + 2]
    # the diagonal of the viewport: the diagonal tiles and, where it leaves a row's closed slab through a grid corner, the
    # tile that corner opens (never the one below-left)
    off, _ = oracle.bin_lines(np.array([[0.0, 0.0, 64.0, 64.0]], np.float32), 4, 4)
    hit = set(np.flatnonzero(np.diff(off)).tolist())
    assert hit == {r * 4 + r for r in range(4)} | {r * 4 + r + 1 for r in range(3)}
    # entirely outside (left, right, above, below), non-finite: nowhere
    out = np.array([[-50, 5, -1, 9], [200, 5, 300, 9], [5, -40, 9, -2], [5, 70, 9, 90], [np.nan, 1, 2, 3], [1, np.inf, 2, 3]], np.float32)
    off, tl = oracle.bin_lines(out, 8, 4)
    assert off[-1] == 0 and len(tl) == 0
    # reaching in from outside: only the inside tiles
    off, _ = oracle.bin_lines(np.array([[-100.0, 8.0, 20.0, 8.0]], np.float32), 8, 4)
    assert np.flatnonzero(np.diff(off)).tolist() == [0, 1]


def test_binning_csr_invariants():
    rng = np.random.default_rng(6)
    lines = adversarial_lines(rng, 4000, 16.0 * 32)
    off, tl = oracle.bin_lines(lines, 32, 32)
    assert off[0] == 0 and off[-1] == len(tl) and np.all(np.diff(off.astype(np.int64)) >= 0)
    for t in np.flatnonzero(np.diff(off))[:200]:
        s = tl[off[t]:off[t + 1]]
        assert np.all(np.diff(s.astype(np.int64)) > 0)   # increasing: no line twice in a tile
    # binning the lines one by one gives the same sets (no cross-talk between records)
    per_line = tiles_of(off, tl, len(lines))
    for i in rng.integers(0, len(lines), 50):
        o1, _ = oracle.bin_lines(lines[i:i + 1], 32, 32)
        assert set(np.flatnonzero(np.diff(o1)).tolist()) == per_line[i]
    # a translation by whole tiles moves the tiles with it
    inner = lines[(lines.min(axis=1) > 40) & (lines.max(axis=1) < 16.0 * 32 - 60)][:300]
    inner = (np.round(inner * 8.0) / 8.0).astype(np.float32)   # (on a 1/8 px lattice the translation is exact in fp32)
    a = tiles_of(*oracle.bin_lines(inner, 32, 32), len(inner))
    shifted = inner + np.array([32.0, 16.0, 32.0, 16.0], np.float32)
    assert np.array_equal((shifted - np.array([32.0, 16.0, 32.0, 16.0], np.float32)), inner)   # (exact in fp32 at these magnitudes)
    b = tiles_of(*oracle.bin_lines(shifted, 32, 32), len(inner))
    for sa, sb in zip(a, b):
        assert {t + 1 * 32 + 2 for t in sa} == sb


def test_binning_of_a_stroke_outline_covers_its_records():
    """On real line soup (config 1, line mode): every record's end points lie in tiles that list the record."""
    from paper_2405_00127_b200 import scenes as S
    sc = S.make("c1", n_paths=24)
    r = oracle.expand(sc.tags, sc.points, sc.styles, sc.affine, sc.tolerance, 0)
    lines = r.xy.astype(np.float32)
    tx = ty = 40
    off, tl = oracle.bin_lines(lines, tx, ty)
    per_line = tiles_of(off, tl, len(lines))
    for i in range(0, len(lines), 7):
        for x, y in ((lines[i, 0], lines[i, 1]), (lines[i, 2], lines[i, 3])):
            c, rr = int(np.floor(x / 16)), int(np.floor(y / 16))
            if 0 <= c < tx and 0 <= rr < ty:
                assert rr * tx + c in per_line[i]
