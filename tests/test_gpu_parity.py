"""GPU parity: the CUDA path (through the C-ABI) against the CPU oracle on the same seeded inputs.

The bar (BASELINE.json north_star): tag-scan results bit-exact; per-segment record counts identical on
>= 99.9 % of input segments; end-point coordinates within 1e-3 px absolute wherever counts match; and the GPU
output passes the same watertightness / winding / tolerance checks as the oracle's.
"""
import numpy as np
import pytest
import torch

import oracle
from oracle import checkers as ck
from paper_2405_00127_b200 import scenes as S

pytestmark = pytest.mark.gpu

COUNT_PARITY = 0.999   # north_star
COORD_TOL = 1e-3       # px, north_star: every end point of every record, whatever its kind
ANGLE_TOL = 2e-5       # rad: fp32 evaluation of an angle of a few radians
KIND_NAMES = {0: "offset", 1: "offset_rev", 2: "evolute", 3: "connector", 4: "join_outer", 5: "join_inner", 6: "cap", 7: "close"}


def check_coords(d, kind, what=""):
    """d[M,4] |gpu - oracle| per coordinate, kind[M] the oracle's record kinds.  One bar for every kind; the
    observed worst case per kind is printed (it lands in the test log)."""
    k3 = np.asarray(kind) & 7
    dm = d.max(axis=1) if len(d) else np.zeros(0)
    report = []
    for k, name in KIND_NAMES.items():
        m = k3 == k
        if m.any():
            report.append(f"{name} {dm[m].max():.2e} ({int(m.sum())})")
    print(f"coordinate parity {what}: max |gpu - oracle| px per kind: " + ", ".join(report))
    assert dm.max(initial=0.0) <= COORD_TOL, (what, float(dm.max()), KIND_NAMES[int(k3[int(dm.argmax())])])


@pytest.fixture(scope="module")
def B():
    from paper_2405_00127_b200 import binding
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return binding


@pytest.fixture(scope="module")
def ctx(B):
    c = B.sx_create(0)
    yield c
    B.sx_destroy(c)


class GpuResult:
    pass


def gpu_run(B, ctx, sc, mode, host=False, into=False):
    """host: stroke_expand_host (pinned host buffers); into: stroke_expand_into (one asynchronous call, per-segment
    results kept); default: stroke_expand = sx_count + allocation callback + sx_write."""
    dev = "cuda:0"
    if into:
        tags, pts, sty = B.scene_to_torch(sc, device=dev)
        B.sx_set_option(ctx, B.SX_OPT_KEEP_SEGMENT_INFO, 1)
        poff_t = torch.empty(sc.n_paths + 1, dtype=torch.int64, device=dev)
        cap = 16 * sc.n_segments + 64
        while True:
            rec_t = torch.full((cap, 8 if mode == 1 else 4), float("nan"), dtype=torch.float32, device=dev)
            try:
                m = B.stroke_expand_into(ctx, tags, pts, sty, sc.affine, sc.tolerance, mode, rec_t, poff_t)
                break
            except B.StrokeExpandError as e:
                assert e.status == B.SX_E_CAPACITY and e.needed > cap
                assert B.sx_last_error(ctx) == B.SX_E_CAPACITY
                cap = e.needed
        torch.cuda.synchronize()
        rec = rec_t[:m].cpu().numpy()
        poff = poff_t.cpu().numpy()
    elif host:
        tags, pts, sty = B.scene_to_torch(sc, pin=True)
        cap = 1 << 16
        while True:
            out = torch.empty((cap, 8 if mode == 1 else 4), dtype=torch.float32).pin_memory()
            poff = torch.empty(sc.n_paths + 1, dtype=torch.int64).pin_memory()
            try:
                m = B.stroke_expand_host(ctx, tags, pts, sty, sc.affine, sc.tolerance, mode, out, poff)
                break
            except B.StrokeExpandError as e:
                assert e.status == B.SX_E_CAPACITY
                cap = e.needed
        rec = out[:m].numpy().copy()
        poff = poff.numpy().copy()
    else:
        tags, pts, sty = B.scene_to_torch(sc, device=dev)
        rec_t, poff_t = B.stroke_expand(ctx, tags, pts, sty, sc.affine, sc.tolerance, mode)
        torch.cuda.synchronize()
        rec = rec_t.cpu().numpy()
        poff = poff_t.cpu().numpy()
    assert B.sx_last_error(ctx) == 0
    if host:
        B.sx_set_option(ctx, B.SX_OPT_KEEP_SEGMENT_INFO, 0)
        tg, pg, sg = B.scene_to_torch(sc, device=dev)
        B.sx_count(ctx, tg, pg, sg, sc.affine, sc.tolerance, mode, torch.empty(sc.n_paths + 1, dtype=torch.int64, device=dev))
    info = B.sx_segment_info(ctx, sc.n_segments)
    if into:
        B.sx_set_option(ctx, B.SX_OPT_KEEP_SEGMENT_INFO, 0)
    g = GpuResult()
    g.xy = np.ascontiguousarray(rec[:, :4])
    if mode == 1:
        g.angle = np.ascontiguousarray(rec[:, 4])
        g.seg = np.ascontiguousarray(rec[:, 5]).view(np.uint32)
        g.kind = np.ascontiguousarray(rec[:, 6]).view(np.uint32).astype(np.uint8)
    else:
        g.angle = np.zeros(len(rec), np.float32)
    g.path_off = poff.astype(np.uint64)
    g.seg_count = info["seg_count"].cpu().numpy().astype(np.uint32)
    g.seg_off = info["seg_offset"].cpu().numpy().astype(np.int64)
    g.pt_off = info["pt_off"].cpu().numpy().astype(np.uint32)
    g.path_idx = info["path_idx"].cpu().numpy().astype(np.uint32)
    g.sp_first = info["sp_first"].cpu().numpy().astype(np.uint32)
    return g


def compare(sc, mode, g, r, min_parity=COUNT_PARITY, angle_tol=ANGLE_TOL):
    """Element-by-element comparison; returns the count-parity fraction."""
    assert np.array_equal(g.pt_off, r.pt_off) and np.array_equal(g.path_idx, r.path_idx) and np.array_equal(g.sp_first, r.sp_first)
    same = g.seg_count == r.seg_count
    parity = float(same.mean()) if len(same) else 1.0
    assert parity >= min_parity, parity
    assert int(g.seg_count.sum()) == len(g.xy)
    assert np.array_equal(g.seg_off, np.cumsum(g.seg_count.astype(np.int64)) - g.seg_count)
    assert np.isfinite(g.xy).all()
    segs = np.flatnonzero(same)
    rep = r.seg_count[segs].astype(np.int64)
    o_off = np.cumsum(r.seg_count.astype(np.int64)) - r.seg_count
    within = np.arange(rep.sum()) - np.repeat(np.cumsum(rep) - rep, rep)
    io = np.repeat(o_off[segs], rep) + within
    ig = np.repeat(g.seg_off[segs], rep) + within
    d = np.abs(g.xy[ig].astype(np.float64) - r.xy[io].astype(np.float64))
    check_coords(d, r.kind[io], f"{sc.name} mode {mode}")
    if mode == 1:
        assert np.abs(g.angle[ig] - r.angle[io]).max(initial=0.0) <= angle_tol
        assert np.array_equal(g.kind[ig], r.kind[io]) and np.array_equal(g.seg[ig], r.seg[io])
    if parity == 1.0:
        assert np.array_equal(g.path_off, r.path_off)
    return parity


def oracle_run(sc, mode):
    return oracle.expand(sc.tags, sc.points, sc.styles, sc.affine, sc.tolerance, mode)


# ---------------------------------------------------------------- element-by-element parity at oracle-sized inputs
CASES = [("c1", None, 0), ("c2", None, 0), ("c2", None, 1), ("c3", 6000, 0), ("c4", 8000, 1), ("c5", 600, 0), ("c5", 600, 1),
         ("c1", None, 2), ("c2", None, 2), ("c3", 6000, 2), ("c5", 600, 2)]   # mode 2: SX_MODE_LINE_REFINED


@pytest.mark.parametrize("name,npaths,mode", CASES)
def test_parity_with_oracle(B, ctx, name, npaths, mode):
    """The one-call path (stroke_expand_into) element by element against the oracle; the two-phase path (sx_count,
    allocation callback, sx_write) must give the same bits."""
    sc = S.make(name, n_paths=npaths)
    g = gpu_run(B, ctx, sc, mode, into=True)
    r = oracle_run(sc, mode)
    compare(sc, mode, g, r)
    assert ck.watertight_violations(g.xy, g.path_off) == 0
    g2 = gpu_run(B, ctx, sc, mode)
    assert np.array_equal(g.xy.view(np.uint32), g2.xy.view(np.uint32)) and np.array_equal(g.path_off, g2.path_off)
    assert np.array_equal(g.seg_count, g2.seg_count) and np.array_equal(g.angle.view(np.uint32), g2.angle.view(np.uint32))


@pytest.mark.parametrize("every,mode", [(1, 0), (1, 1), (2, 0), (2, 1)])
def test_parity_of_filled_paths(B, ctx, every, mode):
    """SURVEY 8(f)-1, Alg. 1: config 2 (every segment kind and degeneracy) with every path, or every second path,
    FILLED instead of stroked -- offset 0, one record chain per segment, the closing line of open subpaths -- element by
    element against the oracle; stroked and filled paths mix in one call."""
    sc = S.with_fill(S.make("c2", n_paths=600), every=every, offset=every - 1)
    g = gpu_run(B, ctx, sc, mode, into=True)
    r = oracle_run(sc, mode)
    assert compare(sc, mode, g, r) >= COUNT_PARITY
    assert ck.watertight_violations(g.xy, g.path_off) == 0
    g2 = gpu_run(B, ctx, sc, mode)
    assert np.array_equal(g.xy.view(np.uint32), g2.xy.view(np.uint32)) and np.array_equal(g.path_off, g2.path_off)
    gh = gpu_run(B, ctx, sc, mode, host=True)
    assert np.array_equal(g.xy.view(np.uint32), gh.xy.view(np.uint32))


@pytest.mark.parametrize("mode", [0, 1])
def test_filled_paths_do_not_depend_on_the_tiling(B, mode):
    """Fills through the sub-tile path and the thread-per-segment walk: the same records, bit for bit."""
    sc = S.with_fill(S.make("c2", n_paths=200), every=2)
    dev = "cuda:0"
    tags, pts, sty = B.scene_to_torch(sc, device=dev)
    width = 8 if mode == 1 else 4
    outs = []
    for tiles in (1, 2, 8, 0):
        c = B.sx_create(0)
        try:
            B.sx_set_option(c, B.SX_OPT_TILE_SEGMENTS, tiles)
            poff = torch.empty(sc.n_paths + 1, dtype=torch.int64, device=dev)
            total = B.sx_count(c, tags, pts, sty, sc.affine, sc.tolerance, mode, poff)
            out = torch.full((total, width), float("nan"), dtype=torch.float32, device=dev)
            B.sx_write(c, out, total, mode)
            torch.cuda.synchronize()
            assert B.sx_last_error(c) == 0
            outs.append((out.cpu().numpy().view(np.uint32), poff.cpu().numpy()))
        finally:
            B.sx_destroy(c)
    for o in outs[1:]:
        assert np.array_equal(outs[0][0], o[0]) and np.array_equal(outs[0][1], o[1])


@pytest.mark.parametrize("name,npaths,mode", [("c1", 64, 0), ("c2", 300, 1)])
def test_host_buffer_entry_point_matches_device_entry_point(B, ctx, name, npaths, mode):
    sc = S.make(name, n_paths=npaths)
    gd = gpu_run(B, ctx, sc, mode)
    gh = gpu_run(B, ctx, sc, mode, host=True)
    assert np.array_equal(gd.xy.view(np.uint32), gh.xy.view(np.uint32)) and np.array_equal(gd.path_off, gh.path_off)
    assert np.array_equal(gd.angle.view(np.uint32), gh.angle.view(np.uint32))


@pytest.mark.parametrize("name,npaths,mode", [("c1", 64, 0), ("c2", 300, 1), ("c4", 2000, 1), ("c5", 40, 0), ("c5", 40, 2)])
def test_tiling_of_the_expansion_kernel_does_not_change_a_bit(B, name, npaths, mode):
    """The warps of the expansion kernel work on tiles of 32, 16 or 8 segments (adapted on the device); a tile that
    does not fit its shared-memory tables is redone in sub-tiles of 8 segments (forced with 2), and a sub-tile that
    still does not fit takes the thread-per-segment reference walk (forced with 1): every choice must give the same
    records, bit for bit."""
    sc = S.make(name, n_paths=npaths)
    dev = "cuda:0"
    tags, pts, sty = B.scene_to_torch(sc, device=dev)
    width = 8 if mode == 1 else 4
    outs = []
    for tiles in (1, 2, 4, 8, 12, 16, 27, 32, 0):
        c = B.sx_create(0)
        try:
            B.sx_set_option(c, B.SX_OPT_TILE_SEGMENTS, tiles)
            poff = torch.empty(sc.n_paths + 1, dtype=torch.int64, device=dev)
            total = B.sx_count(c, tags, pts, sty, sc.affine, sc.tolerance, mode, poff)
            out = torch.full((total, width), float("nan"), dtype=torch.float32, device=dev)
            B.sx_write(c, out, total, mode)
            torch.cuda.synchronize()
            assert B.sx_last_error(c) == 0
            st = B.sx_call_stats(c)
            if tiles == 1:
                assert st["walk_segments"] == sc.n_segments
            if tiles == 2:
                assert st["direct_tiles"] <= 1 and st["sub_tiled_tiles"] > 0
            if tiles >= 4:
                assert st["tile_segments"] == tiles
            outs.append((out.cpu().numpy().view(np.uint32), poff.cpu().numpy(), st))
        finally:
            B.sx_destroy(c)
    print("tiles in one go / in sub-tiles / segments on the walk:", [(o[2]["direct_tiles"], o[2]["sub_tiled_tiles"], o[2]["walk_segments"]) for o in outs])
    for o in outs[1:]:
        assert np.array_equal(outs[0][0], o[0]) and np.array_equal(outs[0][1], o[1])
    assert outs[2][2]["direct_tiles"] > 0   # 4-segment tiles fit on every config


# ---------------------------------------------------------------- the same invariant checks the oracle passes
@pytest.mark.parametrize("name,npaths,mode", [("c1", 128, 0), ("c2", 240, 0), ("c2", 240, 1), ("c3", 300, 0), ("c4", 200, 1), ("c5", 100, 0), ("c5", 100, 1),
                                              ("c1", 128, 2), ("c5", 100, 2)])
def test_gpu_output_passes_the_invariants(B, ctx, name, npaths, mode):
    """Winding / tolerance invariants on 100 paths per config (the same check the oracle's outlines pass)."""
    from test_oracle_outline import _winding_band
    sc = S.make(name, n_paths=npaths)
    g = gpu_run(B, ctx, sc, mode, into=True)
    assert ck.watertight_violations(g.xy, g.path_off) == 0
    rng = np.random.default_rng(123)
    paths = rng.choice(npaths, size=min(npaths, 100), replace=False)
    st = _winding_band(sc, g, paths, rng, 1 if mode == 1 else 0, n_pts=600)
    assert st["inside"] > 5000 and st["outside"] > 5000
    assert st["neg"] == 0 and st["inside_fail"] == 0 and st["outside_fail"] == 0, st


def test_gpu_offsets_track_the_true_parallel_curve(B, ctx):
    """L37: offset vertices within the ES-fit budget of the true parallel curve of the source cubic."""
    sc = S.make("c1", n_paths=16)
    g = gpu_run(B, ctx, sc, 1)  # arc mode carries seg / kind per record
    cubs = ck.segment_cubics(sc.tags, sc.points, sc.affine)
    halfw = 0.5 * sc.styles["width"][g.path_idx]
    tame = []
    for sg in range(sc.n_segments):
        cb, h = cubs[sg], float(halfw[sg])
        t = np.linspace(0, 1, 1001)
        d = ck.cubic_deriv(cb, t)
        dd = 6 * ((1 - t)[:, None] * (cb[2] - 2 * cb[1] + cb[0]) + t[:, None] * (cb[3] - 2 * cb[2] + cb[1]))
        kap = (d[:, 0] * dd[:, 1] - d[:, 1] * dd[:, 0]) / np.hypot(d[:, 0], d[:, 1]) ** 3
        if np.abs(kap).max() * h < 2.0:
            tame.append(sg)
    vmax, mmax = ck.check_offsets(cubs, halfw, g.xy, g.kind, g.seg, angle=g.angle, segs=tame[:40])
    assert vmax < 0.05 and mmax < 1.2 * sc.tolerance


# ---------------------------------------------------------------- edge cases
def test_empty_input(B, ctx):
    dev = "cuda:0"
    tags = torch.empty(0, dtype=torch.uint8, device=dev)
    pts = torch.empty((0, 2), dtype=torch.float32, device=dev)
    sty = torch.empty((0, 16), dtype=torch.uint8, device=dev)
    rec, poff = B.stroke_expand(ctx, tags, pts, sty, S.IDENTITY, 0.25, 0)
    assert rec.shape[0] == 0 and poff.cpu().tolist() == [0]


def test_hand_built_rectangle(B, ctx):
    sc = S.from_paths([dict(start=[10, 20], segs=[[[50, 20]]], width=4.0, cap=S.CAP_BUTT)])
    g = gpu_run(B, ctx, sc, 0)
    assert g.xy.tolist() == [[10, 18, 50, 18], [50, 22, 10, 22], [50, 18, 50, 22], [10, 22, 10, 18]]


def test_zero_width_and_mixed_subpaths(B, ctx):
    # path 0: two subpaths (open polyline + closed triangle); path 1: zero width (emits nothing); path 2: single quad
    tags = np.array([1, 1 | 4, 1, 1, 1 | 4 | 16 | 128, 3 | 4 | 16, 2 | 4 | 16], dtype=np.uint8)
    pts = np.array([[0, 0], [10, 0], [10, 10],  [20, 20], [30, 20], [25, 30], [20, 20],
                    [0, 50], [10, 60], [20, 40], [30, 50],  [50, 50], [60, 70], [70, 50]], dtype=np.float32)
    st = S.make_styles([2.0, 0.0, 3.0], [S.JOIN_MITER, S.JOIN_ROUND, S.JOIN_BEVEL], [S.CAP_SQUARE, S.CAP_ROUND, S.CAP_ROUND], 4.0)
    sc = S.Scene(name="mixed", tags=tags, points=pts, styles=st, affine=S.IDENTITY.copy(), tolerance=0.25, modes=(0, 1))
    for mode in (0, 1):
        g = gpu_run(B, ctx, sc, mode)
        r = oracle_run(sc, mode)
        assert compare(sc, mode, g, r, 1.0) == 1.0
        assert g.seg_count[5] == 0 and g.path_off[1] == g.path_off[2]
        assert ck.watertight_violations(g.xy, g.path_off) == 0


@pytest.mark.parametrize("n", [1, 15, 16, 17, 2047, 2048, 2049, 4095, 4096, 4097, 12289])
def test_scan_tile_boundaries(B, ctx, n):
    """Ragged tails and exact multiples of the scan tiles (4096 tags, 2048 counts): polylines of n line segments
    split into subpaths / paths at irregular places."""
    rng = np.random.default_rng(n)
    tags = np.ones(n, dtype=np.uint8)
    ends = rng.uniform(size=n) < 0.07
    ends[-1] = True
    pends = ends & (rng.uniform(size=n) < 0.5)
    pends[-1] = True
    tags[ends] |= 4
    tags[pends] |= 16
    tags[ends & (rng.uniform(size=n) < 0.5)] |= 128
    npts = int(n + ends.sum())
    pts = rng.uniform(0, 1000, (npts, 2)).astype(np.float32)
    npaths = int(pends.sum())
    st = S.make_styles(rng.uniform(1, 5, npaths), rng.integers(0, 3, npaths), rng.integers(0, 3, npaths), 4.0)
    sc = S.Scene(name="tiles", tags=tags, points=pts, styles=st, affine=S.IDENTITY.copy(), tolerance=0.25, modes=(0,))
    g = gpu_run(B, ctx, sc, 0)
    r = oracle_run(sc, 0)
    compare(sc, 0, g, r)


@pytest.mark.parametrize("bad", ["zero_count", "bit3", "no_path_end", "pts", "paths"])
def test_bad_streams_are_rejected(B, ctx, bad):
    dev = "cuda:0"
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
    t = torch.from_numpy(tags).to(dev)
    p = torch.zeros((n_pts, 2), dtype=torch.float32, device=dev)
    s = torch.from_numpy(S.make_styles([1.0] * n_paths, 0, 0, 4.0).view(np.uint8).reshape(-1, 16).copy()).to(dev)
    with pytest.raises(B.StrokeExpandError) as e:
        B.stroke_expand(ctx, t, p, s, S.IDENTITY, 0.25, 0)
    assert e.value.status == B.SX_E_BAD_STREAM
    B.sx_last_error(ctx)


def test_invalid_arguments_and_capacity(B, ctx):
    sc = S.make("c1", n_paths=4)
    tags, pts, sty = B.scene_to_torch(sc, device="cuda:0")
    poff = torch.empty(sc.n_paths + 1, dtype=torch.int64, device="cuda:0")
    for kw in (dict(tolerance=0.0), dict(mode=7), dict(affine=[1, 0, 2, 0, 0, 0]), dict(affine=[np.nan, 0, 0, 1, 0, 0])):
        a = dict(affine=sc.affine, tolerance=0.25, mode=0)
        a.update(kw)
        with pytest.raises(B.StrokeExpandError) as e:
            B.sx_count(ctx, tags, pts, sty, a["affine"], a["tolerance"], a["mode"], poff)
        assert e.value.status == B.SX_E_INVALID_ARG
    # contiguous but offset views: the kernels' vector loads need 16-byte (tags, styles) / 8-byte (points) alignment
    t1 = torch.cat([tags[:1], tags])[1:]
    p1 = torch.cat([pts.reshape(-1)[:1], pts.reshape(-1)])[1:].reshape(-1, 2)
    for tt, pp in ((t1, pts), (tags, p1)):
        assert tt.is_contiguous() and pp.is_contiguous()
        with pytest.raises(B.StrokeExpandError) as e:
            B.sx_count(ctx, tt, pp, sty, sc.affine, 0.25, 0, poff)
        assert e.value.status == B.SX_E_INVALID_ARG
    out = torch.empty((8, 4), dtype=torch.float32, device="cuda:0")
    with pytest.raises(B.StrokeExpandError) as e:
        B.sx_write(ctx, out, 8)
    assert e.value.status == B.SX_E_STATE
    total = B.sx_count(ctx, tags, pts, sty, sc.affine, 0.25, 0, poff)
    assert total > 8
    with pytest.raises(B.StrokeExpandError) as e:
        B.sx_write(ctx, out, 8)
    assert e.value.status == B.SX_E_CAPACITY
    # asynchronous count (no host total): the kernel itself refuses to write past the capacity
    B.sx_count(ctx, tags, pts, sty, sc.affine, 0.25, 0, poff, want_total=False)
    guard = torch.full((16, 4), 7.0, dtype=torch.float32, device="cuda:0")
    B.sx_write(ctx, guard, 8)
    assert B.sx_last_error(ctx) == B.SX_E_CAPACITY
    assert (guard[8:] == 7.0).all()


# ---------------------------------------------------------------- full-size configs, in the launch configuration bench.py times
def gpu_watertight_violations(rec, poff, chunk_records=48_000_000):
    """Exact bitwise watertightness of EVERY path on the device: per path, the multiset of record start points
    equals the multiset of end points (the same definition as oracle.checkers.watertight_violations, with torch
    sorts; paths are independent, so the check runs over chunks of whole paths)."""
    dev = rec.device
    n_paths = poff.numel() - 1
    po = poff.cpu().numpy()
    bad = 0
    p0 = 0
    while p0 < n_paths:
        p1 = int(np.searchsorted(po, po[p0] + chunk_records, side="right")) - 1
        p1 = max(p1, p0 + 1)
        p1 = min(p1, n_paths)
        a, b = int(po[p0]), int(po[p1])
        if b > a:
            xy = rec[a:b, :4].contiguous() + 0.0   # -0.0 == +0.0 as points
            bits = xy.view(torch.int32).to(torch.int64) & 0xffffffff
            pid = torch.repeat_interleave(torch.arange(p0, p1, device=dev), (poff[p0 + 1:p1 + 1] - poff[p0:p1]))
            keys = []
            for cx, cy in ((0, 1), (2, 3)):
                k = (bits[:, cx] << 32) | bits[:, cy]
                k, order = torch.sort(k)
                _, o2 = torch.sort(pid[order], stable=True)
                keys.append(k[o2])
                del k, order, o2
            diff = keys[0] != keys[1]
            if bool(diff.any()):
                pid_sorted, _ = torch.sort(pid)
                bad += int(torch.unique(pid_sorted[diff]).numel())
            del xy, bits, pid, keys, diff
        p0 = p1
    return bad


def _full_size(B, ctx, name, mode, every, seed):
    """The full-size config through stroke_expand_into (the call bench.py times): every path watertight (exact, on the
    device); the records of every `every`-th path compared with the oracle one by one."""
    sc = S.make(name)
    dev = "cuda:0"
    tags, pts, sty = B.scene_to_torch(sc, device=dev)
    poff = torch.empty(sc.n_paths + 1, dtype=torch.int64, device=dev)
    B.sx_set_option(ctx, B.SX_OPT_KEEP_SEGMENT_INFO, 1)
    try:
        total = B.sx_count(ctx, tags, pts, sty, sc.affine, sc.tolerance, mode, poff)
        width = 8 if mode == 1 else 4
        out = torch.empty((total, width), dtype=torch.float32, device=dev)
        m = B.stroke_expand_into(ctx, tags, pts, sty, sc.affine, sc.tolerance, mode, out, poff)
        torch.cuda.synchronize()
        assert m == total and B.sx_last_error(ctx) == 0
        info = B.sx_segment_info(ctx, sc.n_segments)
        print(f"{name} mode {mode}: {sc.n_segments} segments -> {total} records; tiles {B.sx_call_stats(ctx)}")
    finally:
        B.sx_set_option(ctx, B.SX_OPT_KEEP_SEGMENT_INFO, 0)
    poff_h = poff.cpu().numpy()
    assert poff_h[0] == 0 and poff_h[-1] == total and (np.diff(poff_h) >= 0).all()
    cnt = info["seg_count"]
    assert int(cnt.to(torch.int64).sum()) == total
    assert bool(torch.isfinite(out[:, :4]).all())
    assert gpu_watertight_violations(out, poff) == 0
    if mode == 1:
        assert bool(((out[:, 6].contiguous().view(torch.int32) & 7) <= ck.K_CAP).all())
    paths = np.arange(seed % every, sc.n_paths, every)
    sub, tsel = S.subset_paths(sc, paths)
    r = oracle_run(sub, mode)
    g_cnt = cnt[torch.from_numpy(tsel).to(dev)].cpu().numpy().astype(np.uint32)
    same = g_cnt == r.seg_count
    print(f"{name} mode {mode}: {len(paths)} paths ({len(tsel)} segments) against the oracle: count parity {same.mean():.6f}")
    assert same.mean() >= COUNT_PARITY
    # records of the sampled paths, path by path
    ds, ks = [], []
    for k, p in enumerate(paths):
        a, b = int(poff_h[p]), int(poff_h[p + 1])
        oa, ob = int(r.path_off[k]), int(r.path_off[k + 1])
        segs = np.flatnonzero(r.path_idx == k)
        if not same[segs].all():
            continue
        assert b - a == ob - oa
        got = out[a:b].cpu().numpy()
        ds.append(np.abs(got[:, :4].astype(np.float64) - r.xy[oa:ob].astype(np.float64)))
        ks.append(r.kind[oa:ob])
        if mode == 1:
            assert np.abs(got[:, 4] - r.angle[oa:ob]).max(initial=0.0) <= ANGLE_TOL
    check_coords(np.concatenate(ds), np.concatenate(ks), f"{name} full size mode {mode}")
    del out


def test_full_size_c3(B, ctx):
    _full_size(B, ctx, "c3", 0, 16, 7)


def test_full_size_c3_refined(B, ctx):
    _full_size(B, ctx, "c3", 2, 16, 3)


def test_full_size_c4(B, ctx):
    _full_size(B, ctx, "c4", 1, 64, 8)


@pytest.mark.parametrize("mode", [0, 1])
def test_full_size_c5(B, ctx, mode):
    _full_size(B, ctx, "c5", mode, 64, 9 + mode)


def test_long_chains_tight_tolerance(B, ctx):
    """A tolerance of 0.002 px gives sides with hundreds of records: parts much longer than the 31 records a warp takes
    per iteration and than a tile, non-uniform (f_approx) subdivision, both write-kernel variants' table path."""
    sc = S.make("c1", n_paths=6)
    sc["tolerance"] = 0.002
    for mode in (0, 1, 2):
        g = gpu_run(B, ctx, sc, mode)
        r = oracle_run(sc, mode)
        compare(sc, mode, g, r)
        assert ck.watertight_violations(g.xy, g.path_off) == 0
    assert g.seg_count.max() > 200


def test_very_long_chains(B, ctx):
    """Tolerance 2e-5 px on two paths: thousands of records per side (chains spanning many tiles and ring wrap-arounds)."""
    sc = S.make("c1", n_paths=2)
    sc["tolerance"] = 2e-5
    g = gpu_run(B, ctx, sc, 0)
    r = oracle_run(sc, 0)
    compare(sc, 0, g, r)
    assert ck.watertight_violations(g.xy, g.path_off) == 0
    assert g.seg_count.max() > 5000


def test_arc_records_do_not_depend_on_the_alignment_of_the_buffer(B, ctx):
    """A 32-byte aligned buffer takes arc records as 256-bit stores, a buffer aligned to 16 bytes only as two 16-byte stores:
    the same bits."""
    sc = S.make("c2", n_paths=150)
    dev = "cuda:0"
    tags, pts, sty = B.scene_to_torch(sc, device=dev)
    poff = torch.empty(sc.n_paths + 1, dtype=torch.int64, device=dev)
    total = B.sx_count(ctx, tags, pts, sty, sc.affine, sc.tolerance, 1, poff)
    raw = torch.full((total * 8 + 8,), float("nan"), dtype=torch.float32, device=dev)
    assert raw.data_ptr() % 32 == 0
    a = raw[:total * 8].view(total, 8)
    B.sx_write(ctx, a, total, 1)
    torch.cuda.synchronize()
    wide = a.cpu().numpy().view(np.uint32).copy()
    raw.fill_(float("nan"))
    b = raw[4:4 + total * 8].view(total, 8)
    assert b.data_ptr() % 32 == 16
    B.sx_write(ctx, b, total, 1)
    torch.cuda.synchronize()
    assert B.sx_last_error(ctx) == 0
    assert np.array_equal(wide, b.cpu().numpy().view(np.uint32))
