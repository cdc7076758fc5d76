"""GPU parity of the tile binning (sx_bin_lines) against oracle/bin_oracle.c: the CSR offsets bit-exact, the
records of every tile equal as sets (their order within a tile is not defined: PAPER.md L450, the soup is unordered)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

import oracle
from paper_2405_00127_b200 import scenes as S
from test_oracle_binning import adversarial_lines


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2405_00127_b200 import binding
    return binding


def gpu_bin(B, ctx, lines, tx, ty):
    dev = "cuda:0"
    lt = torch.from_numpy(np.ascontiguousarray(lines, dtype=np.float32)).to(dev)
    off = torch.empty(tx * ty + 1, dtype=torch.int32, device=dev)
    total = None
    try:
        B.sx_bin_lines(ctx, lt, tx, ty, off, None)           # count + scan only: capacity 0
        total = 0
    except B.StrokeExpandError as e:
        assert e.status == B.SX_E_CAPACITY
        total = e.needed
        assert B.sx_last_error(ctx) in (0, B.SX_E_CAPACITY)
    out = torch.full((max(total, 1),), -1, dtype=torch.int32, device=dev)
    m = B.sx_bin_lines(ctx, lt, tx, ty, off, out)
    assert m == total and B.sx_last_error(ctx) == 0
    return off.cpu().numpy().view(np.uint32), out.cpu().numpy().view(np.uint32)[:total]


def compare(off_g, tl_g, off_o, tl_o):
    assert np.array_equal(off_g, off_o)
    assert len(tl_g) == len(tl_o)
    # per tile: sort the slice, compare (one segmented sort: key = tile * 2^32 + line)
    tile_of = np.repeat(np.arange(len(off_o) - 1, dtype=np.uint64), np.diff(off_o.astype(np.int64)))
    kg = np.sort((tile_of << np.uint64(32)) | tl_g.astype(np.uint64))
    ko = (tile_of << np.uint64(32)) | tl_o.astype(np.uint64)
    assert np.array_equal(kg, ko)


@pytest.mark.parametrize("n,tx,ty,seed", [(0, 4, 4, 0), (1, 1, 1, 1), (5000, 20, 14, 2), (200000, 64, 64, 3), (70001, 1024, 3, 4)])
def test_binning_random_lines(B, n, tx, ty, seed):
    """Adversarial synthetic segments (end points on grid lines and corners, horizontal, vertical, points, outside the
    viewport), empty input, one tile, a ragged count, a grid wider than the scan tile."""
    rng = np.random.default_rng(seed)
    lines = adversarial_lines(rng, n, 16.0 * max(tx, ty)) if n else np.zeros((0, 4), np.float32)
    ctx = B.sx_create(0)
    try:
        off_g, tl_g = gpu_bin(B, ctx, lines, tx, ty)
    finally:
        B.sx_destroy(ctx)
    off_o, tl_o = oracle.bin_lines(lines, tx, ty)
    compare(off_g, tl_g, off_o, tl_o)


@pytest.mark.parametrize("name,npaths,tiles", [("c1", None, 32), ("c3", 6000, 256), ("c5", 400, 1024)])
def test_binning_of_the_stroke_outlines(B, name, npaths, tiles):
    """The line soup the stroke expansion itself wrote (line mode) binned on the device, against the oracle binning the same
    records."""
    sc = S.make(name, n_paths=npaths)
    ctx = B.sx_create(0)
    try:
        tags, pts, sty = B.scene_to_torch(sc, device="cuda:0")
        rec, _ = B.stroke_expand(ctx, tags, pts, sty, sc.affine, sc.tolerance, 0)
        torch.cuda.synchronize()
        lines = rec.cpu().numpy()
        off_g, tl_g = gpu_bin(B, ctx, lines, tiles, tiles)
    finally:
        B.sx_destroy(ctx)
    off_o, tl_o = oracle.bin_lines(lines, tiles, tiles)
    assert off_o[-1] >= len(lines) * 0.5   # (most of the scene lies inside the viewport)
    compare(off_g, tl_g, off_o, tl_o)


def test_binning_capacity_and_arguments(B):
    rng = np.random.default_rng(9)
    lines = adversarial_lines(rng, 3000, 256.0)
    dev = "cuda:0"
    ctx = B.sx_create(0)
    try:
        lt = torch.from_numpy(lines).to(dev)
        off = torch.empty(16 * 16 + 1, dtype=torch.int32, device=dev)
        small = torch.full((100,), -1, dtype=torch.int32, device=dev)
        guard = small.clone()
        with pytest.raises(B.StrokeExpandError) as ei:
            B.sx_bin_lines(ctx, lt, 16, 16, off, small)
        assert ei.value.status == B.SX_E_CAPACITY and ei.value.needed > 100
        assert B.sx_last_error(ctx) == B.SX_E_CAPACITY
        off_o, _ = oracle.bin_lines(lines, 16, 16)
        assert np.array_equal(off.cpu().numpy().view(np.uint32), off_o)      # the count is exact all the same
        assert int((small != guard).sum()) <= 100                                 # nothing past the capacity (by construction of the tensor)
        with pytest.raises(B.StrokeExpandError) as ei:
            B.sx_bin_lines(ctx, lt.view(-1)[1:-3].view(-1, 4), 16, 16, off, small)   # misaligned records
        assert ei.value.status == B.SX_E_INVALID_ARG
    finally:
        B.sx_destroy(ctx)
