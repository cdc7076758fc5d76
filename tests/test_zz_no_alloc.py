"""sx_bin_lines_static -- the tile binning for callers that cannot allocate (static device scratch, csrc/sx_static.cu) --
against the existing path sx_bin_lines on the same inputs: CSR offsets bit for bit, every tile's records equal as sets (the
tolerance the binning tests use: integer work, exact).  Two calls in a row on the shared static array (the second with another
viewport and other lines: what must start at zero is cleared), the capacity flag, the limit.  Collected last on purpose."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from paper_2405_00127_b200 import scenes as S


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2405_00127_b200 import binding
    return binding


def synthetic_lines(rng, n, extent):
    """Segments of mixed length, some on grid lines, some outside the viewport, some degenerate."""
    a = rng.uniform(-0.1 * extent, 1.1 * extent, (n, 2))
    d = rng.normal(0.0, 1.0, (n, 2)) * rng.choice([0.0, 2.0, 20.0, 200.0], (n, 1))
    lines = np.concatenate([a, a + d], 1).astype(np.float32)
    snap = rng.random(n) < 0.2
    lines[snap] = np.round(lines[snap] / 16.0) * 16.0
    return lines


def existing_path(B, lines_t, tx, ty):
    ctx = B.sx_create(0)
    try:
        off = torch.empty(tx * ty + 1, dtype=torch.int32, device="cuda:0")
        try:
            B.sx_bin_lines(ctx, lines_t, tx, ty, off, None)
            total = 0
        except B.StrokeExpandError as e:
            assert e.status == B.SX_E_CAPACITY
            total = e.needed
        out = torch.full((max(total, 1),), -1, dtype=torch.int32, device="cuda:0")
        assert B.sx_bin_lines(ctx, lines_t, tx, ty, off, out) == total
        return off.cpu().numpy().view(np.uint32), out.cpu().numpy().view(np.uint32)[:total]
    finally:
        B.sx_destroy(ctx)


def tile_keys(off, tl):
    tile_of = np.repeat(np.arange(len(off) - 1, dtype=np.uint64), np.diff(off.astype(np.int64)))
    return np.sort((tile_of << np.uint64(32)) | tl.astype(np.uint64))


def static_path(B, lines_t, tx, ty, cap):
    off = torch.full((tx * ty + 1,), -1, dtype=torch.int32, device="cuda:0")
    out = torch.full((max(cap, 1),), -1, dtype=torch.int32, device="cuda:0")
    flags = torch.full((1,), 77, dtype=torch.int32, device="cuda:0")
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    B.sx_bin_lines_static(lines_t, tx, ty, off, out if cap else None, flags)
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    return off.cpu().numpy().view(np.uint32), out.cpu().numpy().view(np.uint32), int(flags.item()), free_before, free_after


def test_static_binning_matches_the_existing_path_on_two_calls_in_a_row(B):
    rng = np.random.default_rng(2405)
    # call 1: the line-mode records of config 1 (stroke expansion output) on a 64 x 48 viewport; call 2: synthetic segments on a
    # 200 x 150 viewport (more tiles than one scan tile: the look-back words are used and must have been cleared)
    sc = S.make("c1", n_paths=64)
    ctx = B.sx_create(0)
    try:
        tags, pts, sty = B.scene_to_torch(sc, device="cuda:0")
        rec, _ = B.stroke_expand(ctx, tags, pts, sty, sc.affine, sc.tolerance, B.SX_MODE_LINE)
        torch.cuda.synchronize()
        lines1 = rec.clone()
    finally:
        B.sx_destroy(ctx)
    lines2 = torch.from_numpy(synthetic_lines(rng, 150_000, 3200.0)).to("cuda:0")
    frees = []
    for lines_t, tx, ty in ((lines1, 64, 48), (lines2, 200, 150), (lines1, 64, 48)):
        off_e, tl_e = existing_path(B, lines_t, tx, ty)
        total = int(off_e[-1])
        assert total > 1000
        off_s, tl_s, flags, fb, fa = static_path(B, lines_t, tx, ty, total)
        frees.append((fb, fa))
        assert flags == 0
        assert np.array_equal(off_s, off_e)                                  # offsets bit for bit, the total included
        assert np.array_equal(tile_keys(off_s, tl_s[:total]), tile_keys(off_e, tl_e))
    # no device memory was taken by the calls (the first may load the module lazily: judged on the later ones)
    for fb, fa in frees[1:]:
        assert fa == fb, (fb, fa)


def test_static_binning_flags_and_limit(B):
    rng = np.random.default_rng(7)
    lines_t = torch.from_numpy(synthetic_lines(rng, 20_000, 1024.0)).to("cuda:0")
    off_e, tl_e = existing_path(B, lines_t, 64, 64)
    total = int(off_e[-1])
    # count and scan only (capacity 0): offsets still exact, the capacity flag raised by the scan? no: only the scatter checks it
    off_s, _, flags, _, _ = static_path(B, lines_t, 64, 64, 0)
    assert np.array_equal(off_s, off_e) and flags == 0
    # too small a capacity: nothing written past it, the flag says so; the next call starts clean again
    cap = total // 2
    off_s, tl_s, flags, _, _ = static_path(B, lines_t, 64, 64, cap)
    assert np.array_equal(off_s, off_e) and flags == B.SX_STATIC_FLAG_CAPACITY
    off_s, tl_s, flags, _, _ = static_path(B, lines_t, 64, 64, total)
    assert flags == 0 and np.array_equal(tile_keys(off_s, tl_s[:total]), tile_keys(off_e, tl_e))
    # the limit: 65,536 tiles are served, one more row is rejected with a clear error
    off = torch.empty(256 * 257 + 1, dtype=torch.int32, device="cuda:0")
    B.sx_bin_lines_static(lines_t, 256, 256, off)
    torch.cuda.synchronize()
    assert int(off[256 * 256].item()) >= total
    with pytest.raises(B.StrokeExpandError) as e:
        B.sx_bin_lines_static(lines_t, 256, 257, off)
    assert e.value.status == B.SX_E_INVALID_ARG
    # empty input
    empty = torch.empty((0, 4), dtype=torch.float32, device="cuda:0")
    off = torch.full((17,), -1, dtype=torch.int32, device="cuda:0")
    B.sx_bin_lines_static(empty, 4, 4, off)
    torch.cuda.synchronize()
    assert int(off.abs().sum().item()) == 0
