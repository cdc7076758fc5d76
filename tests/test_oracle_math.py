"""Pins for the oracle's curve mathematics against what the paper and the mathematics fix
(closed forms, quadrature, invariants) -- not against the oracle itself."""
import ctypes as C

import numpy as np
import pytest

import oracle


def ghi(th0, th1):
    k1, c = C.c_float(), C.c_float()
    oracle.lib().so_ghi(th0, th1, C.byref(k1), C.byref(c))
    return k1.value, c.value


def es_z(k0, k1, t):
    x, y = C.c_double(), C.c_double()
    oracle.lib().so_es_integral(k0, k1, t, C.byref(x), C.byref(y))
    return x.value + 1j * y.value


def integrate_spiral(k0, k1, n=200001):
    """independent quadrature (composite Simpson) of the unit-arc spiral kappa = k0 + k1 s, s in [-1/2,1/2]."""
    s = np.linspace(-0.5, 0.5, n)
    th = k0 * s + 0.5 * k1 * s * s
    w = np.ones(n)
    w[1:-1:2] = 4
    w[2:-1:2] = 2
    z = (w * np.exp(1j * th)).sum() * (s[1] - s[0]) / 3
    return z, th[0], th[-1]


# ---------------------------------------------------------------- Appendix A
@pytest.mark.parametrize("th0,th1,tol", [(0.1, 0.2, 2e-6), (0.3, -0.2, 2e-6), (-0.5, 0.45, 2e-6), (1.0, 0.3, 3e-6), (0.0, 0.7, 2e-6)])
def test_ghi_recovers_end_angles(th0, th1, tol):
    """the spiral with k0 = th0+th1 and the polynomial k1 has end tangents th0, th1
    relative to its chord, and chord/arc = c.  Needs s in [-1/2,1/2] (reading R-1)."""
    k1, c = ghi(th0, th1)
    z, a0, a1 = integrate_spiral(th0 + th1, k1)
    chord_ang = np.angle(z)
    assert abs((chord_ang - a0) - th0) < tol + 5e-7 * abs(k1)
    assert abs((a1 - chord_ang) - th1) < tol + 5e-7 * abs(k1)
    assert abs(abs(z) - c) < 2e-6


def test_ghi_printed_values():
    """values recorded in SURVEY A-1 for (0.1, 0.2) (independent double-precision evaluation)."""
    k1, c = ghi(0.1, 0.2)
    assert abs(k1 - 0.599085156207) < 1e-6
    assert abs(c - 0.996006469645) < 1e-6


@pytest.mark.parametrize("k", [0.0, 0.3, 1.0, 2.0, 3.0])
def test_ghi_delta_zero_is_sinc(k):
    """chord/arc = sinc(k/2) when Delta = 0; and k1 = 0 (circular arc)."""
    k1, c = ghi(k / 2, k / 2)
    assert k1 == 0.0
    ref = 1.0 if k == 0 else np.sin(k / 2) / (k / 2)
    # the polynomial is the sinc series truncated after k^6: the next term (k/2)^8/9! bounds the gap
    assert abs(c - ref) < 3e-6 + 1.05 * (k / 2) ** 8 / 362880


def test_ghi_first_order():
    """L636: k1 -> 6 Delta for small angles."""
    k1, _ = ghi(0.0, 1e-3)
    assert abs(k1 / 1e-3 - 6.0) < 1e-4


# ---------------------------------------------------------------- Euler spiral integral
def test_es_integral_circular_arc_closed_form():
    for k0 in [0.2, 1.0, 2.5]:
        for t in [0.3, 1.0]:
            z = es_z(k0, 0.0, t)
            ref = (np.sin(k0 * t) + 1j * (1 - np.cos(k0 * t))) / k0
            assert abs(z - ref) < 1e-13


def test_es_integral_straight_and_general():
    assert abs(es_z(0.0, 0.0, 0.7) - 0.7) < 1e-15
    # general case against an independent Simpson quadrature
    k0, k1, t = 0.9, 2.2, 0.8
    u = np.linspace(0, t, 100001)
    ph = (k0 - k1 / 2) * u + 0.5 * k1 * u * u
    w = np.ones_like(u); w[1:-1:2] = 4; w[2:-1:2] = 2
    ref = (w * np.exp(1j * ph)).sum() * (u[1] - u[0]) / 3
    assert abs(es_z(k0, k1, t) - ref) < 1e-12


# ---------------------------------------------------------------- section 4.1 / 4.2
def test_f_exact_matches_quadrature_and_values():
    L = oracle.lib()
    assert abs(L.so_f_exact(1.0) - np.pi / 4) < 1e-15           # L139 with reading R-3
    assert abs(L.so_f_exact(-0.4) + L.so_f_exact(0.4)) < 1e-16   # odd, L141
    assert abs(L.so_f_exact(1.5) - 1.1427118299) < 1e-9          # SURVEY A-3 (quadrature of L135)
    assert abs(L.so_f_exact(3.0) - 4.1466652635) < 1e-9
    for x in [0.3, 0.95, 1.0, 1.2, 2.5]:
        u = np.linspace(0, x, 400001)
        g = np.sqrt(np.abs(u * u - 1))
        ref = ((g[:-1] + g[1:]) * 0.5).sum() * (u[1] - u[0])
        assert abs(L.so_f_exact(x) - ref) < 2e-5


def test_f_approx_knots_and_printed_values():
    """L149-157: continuity at 0.8 / 1.25 / 2.1 (values SURVEY sec.4 recorded from the printed formula)."""
    L = oracle.lib()
    for x, v in [(0.8, 0.7010707591), (1.25, 0.9032492936), (2.1, 2.0388577936)]:
        lo = L.so_f_approx(np.nextafter(np.float32(x), np.float32(0)))
        hi = L.so_f_approx(np.float32(x))
        assert abs(lo - v) < 2e-6 and abs(hi - v) < 2e-6
    assert abs(L.so_f_approx(1.0) - np.pi / 4) < 1e-7
    assert L.so_f_approx(-1.7) == -L.so_f_approx(1.7)


def test_f_approx_inverse_roundtrip():
    L = oracle.lib()
    for x in np.concatenate([np.linspace(-4, 4, 801), [0.7999, 0.8001, 1.2499, 1.2501, 2.0999, 2.1001, 50.0, -300.0]]):
        u = L.so_f_approx(float(x))
        xr = L.so_f_approx_inv(u)
        # the inverse is ill-conditioned only at x = +-1 where the density vanishes
        tol = 2e-3 if abs(abs(x) - 1) < 0.02 else 3e-5 * max(1, abs(x))
        assert abs(xr - x) < tol, (x, xr)


def test_f_approx_six_percent():
    """L145: worst-case discrepancy between approximate and exact subdivision counts is 6%."""
    L = oracle.lib()
    rng = np.random.default_rng(5)
    worst_hi, worst_lo = 1.0, 1.0
    for _ in range(20000):
        a, b = np.sort(rng.uniform(-4, 4, 2))
        if b - a < 1e-2:
            continue
        ra = (L.so_f_approx(b) - L.so_f_approx(a)) / (L.so_f_exact(b) - L.so_f_exact(a))
        worst_hi, worst_lo = max(worst_hi, ra), min(worst_lo, ra)
    assert worst_hi < 1.065 and worst_lo > 0.935
    assert worst_hi > 1.02 or worst_lo < 0.98  # it IS an approximation: a pasted exact f would fail here


# ---------------------------------------------------------------- section 7.1
def fit(u0, u1, q0, q1, ch, dt=1.0):
    out = np.zeros(4, dtype=np.float32)
    a = [np.ascontiguousarray(v, dtype=np.float32) for v in (u0, u1, ch)]
    oracle.lib().so_fit_error_export(a[0].ctypes.data, a[1].ctypes.data, q0, q1, a[2].ctypes.data, dt, out.ctypes.data)
    return out


def _bezier_area(pts, n=20001):
    """signed area between the cubic and its chord, by the shoelace formula on a dense sampling."""
    t = np.linspace(0, 1, n)[:, None]
    p = (1 - t) ** 3 * pts[0] + 3 * (1 - t) ** 2 * t * pts[1] + 3 * (1 - t) * t * t * pts[2] + t ** 3 * pts[3]
    x, y = p[:, 0], p[:, 1]
    return 0.5 * np.sum(x[:-1] * y[1:] - x[1:] * y[:-1])


def test_fit_error_terms():
    """L215-229.  With the arm lengths of the ES-fit cubic (d = 2/(3(1+cos th)), L217) terms 2 and 3 vanish
    and the estimate is chord * (4.6255e-6 k^5 + 7.5e-3 k^2 |th0-th1|) (L221); the area term (L225-227) is
    pinned against a shoelace area of the two sampled cubics."""
    th0, th1, chord = 0.3, 0.2, 7.0
    u0 = np.array([np.cos(-th0), np.sin(-th0)])
    u1 = np.array([np.cos(th1), np.sin(th1)])
    db0, db1 = 2 / (3 * (1 + np.cos(th0))), 2 / (3 * (1 + np.cos(th1)))
    r = fit(u0, u1, db0 * chord, db1 * chord, [chord, 0.0])
    assert abs(r[0] - th0) < 1e-6 and abs(r[1] - th1) < 1e-6 and abs(r[2] - chord) < 1e-6
    e1 = 4.6255e-6 * 0.5 ** 5 + 7.5e-3 * 0.25 * 0.1
    assert abs(r[3] / chord - e1) < 2e-7
    # now a different source cubic: arms d0, d1; area difference via sampled shoelace
    d0, d1 = 0.45, 0.25
    r2 = fit(u0, u1, d0 * chord, d1 * chord, [chord, 0.0])

    def unit_cubic(a0, a1):
        return np.array([[0, 0], a0 * u0, np.array([1.0, 0]) - a1 * u1, [1.0, 0]])
    dA = abs(_bezier_area(unit_cubic(d0, d1)) - _bezier_area(unit_cubic(db0, db1)))
    e3 = (0.005 * 0.5 + 0.07 * 0.1) * np.hypot(db0 - d0, db1 - d1)
    assert abs(r2[3] / chord - (e1 + 1.55 * dA + e3)) < 3e-6
    # dt scales the arms: a sub-range of half the parameter length has half the arm
    r3 = fit(u0, u1, 2 * d0 * chord, 2 * d1 * chord, [chord, 0.0], dt=0.5)
    assert abs(r3[3] - r2[3]) < 1e-6


def test_fit_error_guards():
    r = fit([1, 0], [1, 0], 1.0, 1.0, [0.0, 0.0])
    assert np.isinf(r[3])                       # zero chord: force a split (R-4)
    r = fit([-1, 0], [1, 0], 1.0, 1.0, [3.0, 0.0])
    assert r[3] == pytest.approx(6.0)           # |theta| > 120 deg: err = 2 chord (R-4)


def test_fit_error_tracks_true_error():
    """The estimate must be of the size of the true cubic<->ES distance (L231 claims it conservative with mean
    ratio 1.656; SURVEY A-6 could not reproduce that, so the exact ratio is 'parity unpinned').  What is pinned:
    true/estimate stays in a fixed band over the validated box, so a dropped term or a constant off by 10x fails."""
    rng = np.random.default_rng(11)
    ratios = []
    for _ in range(60):
        th0, th1 = rng.uniform(0.05, 0.5, 2)
        d0, d1 = rng.uniform(0.15, 0.55, 2)
        u0 = np.array([np.cos(-th0), np.sin(-th0)]); u1 = np.array([np.cos(th1), np.sin(th1)])
        est = fit(u0, u1, d0, d1, [1.0, 0.0])[3]
        cub = np.array([[0, 0], d0 * u0, np.array([1.0, 0]) - d1 * u1, [1.0, 0]])
        t = np.linspace(0, 1, 1501)[:, None]
        cp = (1 - t) ** 3 * cub[0] + 3 * (1 - t) ** 2 * t * cub[1] + 3 * (1 - t) * t * t * cub[2] + t ** 3 * cub[3]
        k1, _ = ghi(th0, th1)
        k0 = th0 + th1
        z1 = es_z(k0, k1, 1.0)
        zs = np.array([es_z(k0, k1, float(tt)) for tt in np.linspace(0, 1, 301)]) / z1
        es = np.stack([zs.real, zs.imag], 1)
        d_c2e = np.sqrt(((cp[:, None, :] - es[None]) ** 2).sum(2)).min(1).max()
        d_e2c = np.sqrt(((es[:, None, :] - cp[None]) ** 2).sum(2)).min(1).max()
        ratios.append(max(d_c2e, d_e2c) / est)
    ratios = np.array(ratios)
    assert 0.7 < np.median(ratios) < 1.3
    assert ratios.max() < 4.0 and np.mean((ratios > 0.4) & (ratios < 2.0)) >= 0.9
