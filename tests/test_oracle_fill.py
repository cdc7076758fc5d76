"""Pins for the FILL branch of the oracle (Alg. 1: "if style is fill then flatten_cubic(segment, 0)"; SURVEY
8(f)-1): at offset 0 the flattening density is that of the Euler spiral itself, sqrt|kappa| / sqrt(8 d) (section 2.2,
L77-97: subdivision points s_i ~ i^(2/3) from the inflection), arcs n = cbrt(s^3 |kappa'| / (120 d)) (section 5).
Measured against geometry built here: the exact spiral by quadrature, the exact area enclosed by the Bezier path (Green's
theorem on the control points), the source curves sampled densely."""
import numpy as np

import oracle
from oracle import checkers as ck
from paper_2405_00127_b200 import scenes as S
from test_oracle_pins import exact_spiral

K_OFFSET, K_CLOSE, K_PLUS = 0, 7, 8


def fill_piece(k0, k1, L, d, mode):
    r = oracle.piece_expand(k0, k1, L, 0.0, d, mode)
    assert np.all(r.kind == K_OFFSET)                    # one side, no mirror image, no evolute
    assert np.array_equal(r.xy[1:, 0:2], r.xy[:-1, 2:4])  # a connected chain in increasing t
    return r


def test_fill_through_an_inflection_follows_the_two_thirds_rule():
    """kappa from -k to +k over the piece: int sqrt|kappa| ds = (4/3) (1/2)^1.5 sqrt(L |k1|), so n = ceil of that over
    sqrt(8 d); the interior vertices sit ON the spiral at s = +-(L/2) (2 i / n)^(2/3) from the inflection (L97)."""
    k0, k1, L, d = 0.0, 4.0, 100.0, 0.2
    n_real = (4.0 / 3.0) * 0.5 ** 1.5 * np.sqrt(L * k1) / np.sqrt(8.0 * d)
    r = fill_piece(k0, k1, L, d, 0)
    n = len(r.xy)
    assert n == int(np.ceil(n_real)) == 8
    t, P, th, kap = exact_spiral(k0, k1, L)
    for i in range(1, n):
        u = 2.0 * i / n - 1.0                                 # signed share of the integral, from the inflection
        frac = 0.5 + 0.5 * np.sign(u) * abs(u) ** (2.0 / 3.0)
        p = P[int(round(frac * (len(t) - 1)))]
        assert abs(complex(*r.xy[i, 0:2]) - p) < 2e-3, (i, r.xy[i, 0:2], p)
    # the chords use the tolerance and keep it: deviation d (n_real / n)^2 up to the slack of the estimate
    w = np.linspace(0.0, 1.0, 17)[None, :, None]
    on = (r.xy[:, None, 0:2] * (1 - w) + r.xy[:, None, 2:4] * w).reshape(-1, 2).astype(np.float64)
    dev = float(ck.dist_points_to_polyline(on, np.stack([P.real, P.imag], 1)[::4]).max())
    assert 0.6 * d <= dev <= 1.05 * d, dev


def test_fill_chords_and_arcs_use_the_tolerance_and_keep_it():
    """Random accepted-range pieces at offset 0: the measured deviation of the chords (lines) and of the arcs from the exact
    spiral stays below the flatten tolerance and, where several records are emitted, uses a good part of it."""
    rng = np.random.default_rng(11)
    d = 0.2
    used_l, used_a = [], []
    for _ in range(60):
        k0, k1, L = rng.uniform(-2.0, 2.0), rng.uniform(-7.0, 7.0), rng.uniform(40.0, 400.0)
        t, P, th, kap = exact_spiral(k0, k1, L)
        poly = np.stack([P.real, P.imag], 1)[::4]
        r = fill_piece(k0, k1, L, d, 0)
        w = np.linspace(0.0, 1.0, 17)[None, :, None]
        on = (r.xy[:, None, 0:2] * (1 - w) + r.xy[:, None, 2:4] * w).reshape(-1, 2).astype(np.float64)
        dev = float(ck.dist_points_to_polyline(on, poly).max())
        assert dev <= 1.2 * d, (k0, k1, L, dev)     # (the user tolerance is 1.25 d: R-13)
        if len(r.xy) >= 4:
            used_l.append(dev / d)
        ra = fill_piece(k0, k1, L, d, 1)
        on_a = ck.arcs_to_lines(ra.xy.astype(np.float64), ra.angle.astype(np.float64), n=24)[:, 0:2]
        dev_a = float(ck.dist_points_to_polyline(on_a, poly).max())
        assert dev_a <= 1.2 * d, (k0, k1, L, dev_a)
        assert len(ra.xy) == max(1, int(np.ceil(np.cbrt(L * abs(k1) / (120.0 * d)) * (1 - 1e-6))))   # L171 with s^3 kappa' = L k1
        if len(ra.xy) >= 3:
            used_a.append(dev_a / d)
    assert np.median(used_l) > 0.5 and np.median(used_a) > 0.3, (np.median(used_l), np.median(used_a))


def bezier_area(cubs):
    """Signed area enclosed by a closed chain of cubics (Green's theorem, exact: 1/2 int x dy - y dx per cubic, by 8-point
    Gauss-Legendre, exact for the degree-5 integrand)."""
    x, w = np.polynomial.legendre.leggauss(8)
    t = 0.5 * (x + 1.0)
    a = 0.0
    for cb in cubs:
        p = ck.cubic_eval(cb, t)
        q = ck.cubic_deriv(cb, t)
        a += 0.25 * float(np.sum(w * (p[:, 0] * q[:, 1] - p[:, 1] * q[:, 0])))
    return a


def test_filled_scene_is_closed_stays_on_the_curves_and_has_the_right_area():
    """Config 2 (every style, degenerate cubics) with every path filled, both modes: per subpath the records chain into a
    closed polygon bit for bit (the closing line included, L309-311); every vertex lies on its source segment and the chord /
    arc mid-points within the tolerance of it; the enclosed area equals the exact area of the Bezier path (closed by the
    same line) up to perimeter x tolerance."""
    sc = S.with_fill(S.make("c2", n_paths=120))
    cubs = ck.segment_cubics(sc.tags, sc.points, sc.affine)
    sp_end = ((sc.tags >> 2) | (sc.tags >> 4)) & 1
    closed = (sc.tags >> 7) & 1
    for mode in (0, 1):
        r = oracle.expand(sc.tags, sc.points, sc.styles, sc.affine, sc.tolerance, mode)
        assert ck.watertight_violations(r.xy, r.path_off) == 0
        assert not np.any(r.kind & K_PLUS) and set(np.unique(r.kind).tolist()) <= {K_OFFSET, K_CLOSE}
        assert int((r.kind == K_CLOSE).sum()) == int((sp_end & (1 - closed)).sum())
        seg_off = np.concatenate([[0], np.cumsum(r.seg_count)]).astype(np.int64)
        first = 0
        checked = 0
        for i in range(sc.n_segments):
            a, b = seg_off[i], seg_off[i + 1]
            rec = r.xy[a:b].astype(np.float64)
            body = rec[: len(rec) - (1 if (sp_end[i] and not closed[i]) else 0)]
            assert len(body) >= 1
            # the segment's own records: a chain from C(0) to C(1), on the curve
            assert np.array_equal(body[1:, 0:2], body[:-1, 2:4])
            assert np.allclose(body[0, 0:2], ck.cubic_eval(cubs[i], np.array([0.0]))[0], atol=1e-3)
            assert np.allclose(body[-1, 2:4], ck.cubic_eval(cubs[i], np.array([1.0]))[0], atol=1e-3)
            poly = ck.path_polyline([cubs[i]], n=2049)
            if mode == 0:
                pts = np.concatenate([body[:, 0:2], 0.5 * (body[:, 0:2] + body[:, 2:4])])
            else:
                pts = ck.arcs_to_lines(body, r.angle[a:a + len(body)].astype(np.float64), n=4)[:, 0:2]
            assert float(ck.dist_points_to_polyline(pts, poly).max()) <= sc.tolerance, i
            if sp_end[i]:
                # the subpath first .. i: area of the emitted polygon against the exact area
                lo, hi = seg_off[first], seg_off[i + 1]
                lines = ck.arcs_to_lines(r.xy[lo:hi].astype(np.float64), r.angle[lo:hi].astype(np.float64), n=16) if mode else r.xy[lo:hi].astype(np.float64)
                area = 0.5 * float(np.sum(lines[:, 0] * lines[:, 3] - lines[:, 2] * lines[:, 1]))
                chain = [cubs[j] for j in range(first, i + 1)]
                p_end, p_start = ck.cubic_eval(cubs[i], np.array([1.0]))[0], ck.cubic_eval(cubs[first], np.array([0.0]))[0]
                exact = bezier_area(chain) + 0.5 * float(p_end[0] * p_start[1] - p_start[0] * p_end[1])
                per = float(np.hypot(lines[:, 2] - lines[:, 0], lines[:, 3] - lines[:, 1]).sum())
                assert abs(area - exact) <= per * sc.tolerance + 1e-6, (i, area, exact, per)
                checked += 1
                first = i + 1
        assert checked >= 120


def test_fill_and_stroke_paths_mix_in_one_call():
    """Filling every second path leaves the stroked paths' records untouched, bit for bit."""
    base = S.make("c2", n_paths=60)
    mixed = S.with_fill(base, every=2, offset=1)
    for mode in (0, 1):
        a = oracle.expand(base.tags, base.points, base.styles, base.affine, base.tolerance, mode)
        b = oracle.expand(mixed.tags, mixed.points, mixed.styles, mixed.affine, mixed.tolerance, mode)
        for p in range(0, 60, 2):
            ra, rb = a.xy[a.path_off[p]:a.path_off[p + 1]], b.xy[b.path_off[p]:b.path_off[p + 1]]
            assert np.array_equal(ra.view(np.uint32), rb.view(np.uint32))
        for p in range(1, 60, 2):
            k = b.kind[b.path_off[p]:b.path_off[p + 1]]
            assert set(np.unique(k).tolist()) <= {K_OFFSET, K_CLOSE}
