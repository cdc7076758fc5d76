"""GPU parity for dashing (csrc/sx_dash.cuh) against the oracle's sequential dash walk: per-segment counts,
record coordinates (1e-3 px), angles / kinds / segment ids in arc mode, watertight dashes; the prefix-sum path on a long
polyline of short segments (the paper's "long dash" case, L543), mixed dashed / undashed / filled paths, argument checks."""
import numpy as np
import pytest
import torch

import oracle
from oracle import checkers as ck
from paper_2405_00127_b200 import scenes as S
from test_gpu_parity import B, ctx, gpu_run, compare   # noqa: F401  (fixtures and helpers)

pytestmark = pytest.mark.gpu

# arc angles of dash sub-ranges: phi(tb) - phi(ta) of the cut piece in fp32 against the oracle's double; on config 2's wildest
# pieces (|k1| of a few hundred) the rounding of k1 t alone is 1e-5 rad
DASH_ANGLE_TOL = 5e-5


def dashed_pair(B, ctx, sc, mode, dash, phase, into=True):
    B.sx_set_dash(ctx, dash, phase)
    try:
        g = gpu_run(B, ctx, sc, mode, into=into)
    finally:
        B.sx_set_dash(ctx, None)
    r = oracle.expand(sc.tags, sc.points, sc.styles, sc.affine, sc.tolerance, mode, dash=dash, phase=phase)
    return g, r


@pytest.mark.parametrize("name,npaths,mode,every", [("c1", 96, 0, 1), ("c1", 96, 1, 1), ("c2", 600, 0, 2), ("c2", 600, 1, 1), ("c3", 3000, 0, 1),
                                                    ("c4", 2000, 1, 3), ("c5", 60, 0, 1), ("c5", 60, 1, 2), ("c1", 64, 2, 1)])
def test_dashed_parity_with_oracle(B, ctx, name, npaths, mode, every):
    sc = S.with_dash(S.make(name, n_paths=npaths), every=every)
    dash, phase = [26.0, 11.0, 5.0, 11.0], 3.0
    g, r = dashed_pair(B, ctx, sc, mode, dash, phase)
    parity = compare(sc, mode, g, r, angle_tol=DASH_ANGLE_TOL)
    print(f"dashed {name} mode {mode}: {sc.n_segments} segments -> {len(g.xy)} records, count parity {parity:.6f}")
    assert ck.watertight_violations(g.xy, g.path_off) == 0
    # the two-phase path gives the same bits
    B.sx_set_dash(ctx, dash, phase)
    try:
        g2 = gpu_run(B, ctx, sc, mode)
    finally:
        B.sx_set_dash(ctx, None)
    assert np.array_equal(g.xy.view(np.uint32), g2.xy.view(np.uint32)) and np.array_equal(g.path_off, g2.path_off)


def long_polyline(n_seg, closed=False):
    """One path of n_seg short line segments along a slowly opening spiral (segment lengths 2 .. 6 px) and one of cubics."""
    k = np.arange(n_seg + 1)
    ang = 0.02 * k
    rad = 300.0 + 0.05 * k
    pts = np.stack([2000 + rad * np.cos(ang), 2000 + rad * np.sin(ang)], 1)
    poly = dict(start=pts[0].tolist(), segs=[[p.tolist()] for p in pts[1:]], width=5.0, join=S.JOIN_ROUND, cap=S.CAP_ROUND, closed=closed)
    return poly


def test_long_dash_polyline_uses_the_prefix_sum(B, ctx):
    """PAPER.md L543 ("long dash"): 60,000 short segments in ONE subpath, dashes longer than many segments: a dash start
    depends on the lengths of all the segments before it -- the prefix sum across thousands of blocks -- and must land on the
    same segment, at the same place, as in the sequential walk."""
    sc = S.with_dash(S.from_paths([long_polyline(60000), dict(start=[100, 100], segs=[[[400, 900], [900, -300], [1300, 500]]], width=8.0, cap=S.CAP_SQUARE)]))
    dash, phase = [37.0, 13.5, 3.25, 13.5], 21.0
    g, r = dashed_pair(B, ctx, sc, 0, dash, phase)
    parity = compare(sc, 0, g, r, min_parity=1.0)
    assert parity == 1.0 and ck.watertight_violations(g.xy, g.path_off) == 0
    n_dashes_expected = 2 * int(np.ceil((np.hypot(*np.diff(np.array([long_polyline(60000)["start"]] + [s[0] for s in long_polyline(60000)["segs"]]), axis=0).T).sum() + phase) / sum(dash)))
    caps = int(((r.kind & 7) == 6).sum())
    assert caps > 1000 and abs(len(g.xy) - r.n_rec) == 0
    print(f"long dash: {sc.n_segments} segments -> {len(g.xy)} records, about {n_dashes_expected} dashes")


def test_pattern_cleared_gives_the_undashed_bits_and_bad_patterns_are_refused(B, ctx):
    sc = S.with_dash(S.make("c2", n_paths=200))
    g0 = gpu_run(B, ctx, sc, 0, into=True)                       # no pattern set: the style bit alone does nothing
    r0 = oracle.expand(sc.tags, sc.points, sc.styles, sc.affine, sc.tolerance, 0)
    assert compare(sc, 0, g0, r0) == 1.0
    B.sx_set_dash(ctx, [5.0, 5.0], 0.0)
    B.sx_set_dash(ctx, None)
    g1 = gpu_run(B, ctx, sc, 0, into=True)
    assert np.array_equal(g0.xy.view(np.uint32), g1.xy.view(np.uint32))
    for bad, phase in (([5.0], 0.0), ([5.0, 0.0], 0.0), ([5.0, -1.0], 0.0), ([1.0] * 10, 0.0), ([5.0, 5.0, 5.0], 0.0), ([5.0, 5.0], -1.0), ([5.0, float("nan")], 0.0)):
        with pytest.raises(B.StrokeExpandError) as e:
            B.sx_set_dash(ctx, bad, phase)
        assert e.value.status == B.SX_E_INVALID_ARG
    # an all-on pattern on open paths: the multiset of the undashed records
    opened = S.Scene(S.make("c1", n_paths=12))
    opened["tags"] = opened.tags & ~np.uint8(128)
    und = gpu_run(B, ctx, opened, 0, into=True)
    g, r = dashed_pair(B, ctx, S.with_dash(opened), 0, [1e6, 1.0], 0.0)
    key = lambda a: np.sort(np.ascontiguousarray(a).view(np.uint32).astype(np.uint64).dot(np.array([1, 1 << 16, 1 << 32, 1 << 48], dtype=np.uint64)))
    assert len(g.xy) == len(und.xy)
    d = np.abs(np.sort(g.xy, axis=0) - np.sort(und.xy, axis=0)).max()
    assert d <= 1e-3, d          # (the dashed walk re-bases every piece at its own start vertex: ulps, not bits)


def test_dashed_fill_and_mixed_styles(B, ctx):
    """Filled paths ignore the dash bit; dashed and undashed strokes mix in one call."""
    base = S.make("c2", n_paths=300)
    sc = S.with_dash(S.with_fill(base, every=3), every=1)
    g, r = dashed_pair(B, ctx, sc, 1, [14.0, 6.0], 2.5)
    compare(sc, 1, g, r, angle_tol=DASH_ANGLE_TOL)
    assert ck.watertight_violations(g.xy, g.path_off) == 0


@pytest.mark.parametrize("dash,phase", [([7.0, 3.0], 0.0), ([0.01, 0.02], 0.005), ([1000.0, 5.0], 0.0), ([1000.0, 5.0], 998.0), ([50.0, 50.0], 50.0),
                                        ([2.0 ** -9, 2.0 ** -9], 0.0)])
@pytest.mark.parametrize("mode", [0, 1])
def test_dash_edge_scenes(B, ctx, dash, phase, mode):
    """Zero-length segments at the start, in the middle and at the end of a dashed path, a degenerate cubic, a closed
    triangle, dashes of 1/512 px and a pattern longer than the path (tests/test_oracle_dash.py::edge_scenes): the position
    rules decide caps and joins identically on both sides."""
    from test_oracle_dash import edge_scenes
    sc = edge_scenes()
    g, r = dashed_pair(B, ctx, sc, mode, dash, phase)
    assert compare(sc, mode, g, r, min_parity=1.0, angle_tol=DASH_ANGLE_TOL) == 1.0
    assert ck.watertight_violations(g.xy, g.path_off) == 0
