"""The kernels' own math, probed on the device (sx_eval): the angle function of reading R-17 against the definition
(atan2 in double precision, rounded once to fp32 -- evaluated here with numpy, not with the oracle), and the decision-grade
error estimate of section 7.1 against the oracle's plain fp32 evaluation of the same formulas."""
import ctypes as C

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

import oracle


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2405_00127_b200 import binding
    return binding


def test_angle_function_is_the_rounded_double_atan2(B):
    """R-17: theta = fl32(atan2(y, x)).  Two million arguments -- unit-ish vectors as the fit produces them, all octants,
    tiny and huge magnitudes, the axes, equal components: the kernel's own double-precision evaluation must give the same
    fp32 value except where the exact angle sits within ~1e-16 of a rounding boundary (allowed: 5 in 2 million)."""
    rng = np.random.default_rng(17)
    n = 2_000_000
    ang = rng.uniform(-np.pi, np.pi, n)
    mag = np.where(rng.random(n) < 0.8, 1.0 + rng.normal(0, 1e-7, n), 10.0 ** rng.uniform(-30, 30, n))
    yx = np.stack([mag * np.sin(ang), mag * np.cos(ang)], 1).astype(np.float32)
    small = rng.random(n) < 0.3                      # the accepted pieces' angles: a few tenths of a radian and below
    yx[small, 0] = (yx[small, 1] * np.tan(rng.uniform(-0.5, 0.5, int(small.sum())))).astype(np.float32)
    special = np.array([[0, 1], [0, -1], [1, 0], [-1, 0], [1, 1], [-1, 1], [1, -1], [-1, -1], [0.25, 1], [0.5, 1], [0.75, 1],
                        [1, 0.25], [1e-38, 1], [1, 1e-38], [3e38, 3e38], [1e-45, 1e-45], [0.0, 0.0], [-0.0, 1.0]], np.float32)
    yx = np.concatenate([special, yx])
    got = B.sx_eval(B.SX_EVAL_ATAN2, yx)
    want = np.arctan2(yx[:, 0].astype(np.float64), yx[:, 1].astype(np.float64)).astype(np.float32)
    diff = got.view(np.int32).astype(np.int64) - want.view(np.int32).astype(np.int64)
    bad = np.flatnonzero((got != want) & ~((got == 0) & (want == 0)))
    print(f"angle function: {len(bad)} of {len(yx)} differ from fl32(atan2 in double); max ulp distance {np.abs(diff[bad]).max(initial=0)}")
    assert len(bad) <= 5 and np.abs(diff[bad]).max(initial=0) <= 1
    assert np.array_equal(got[:8], want[:8])         # the axes and the diagonals exactly


def test_node_error_agrees_with_the_plain_formulas(B):
    """Section 7.1: the kernel's estimate (MUFU-grade reciprocals, fused multiply-adds, own atan2, area difference expanded)
    against the oracle's operation-by-operation fp32 evaluation on random nodes of the kind Alg. 2 meets: relative
    difference below 1e-4, below 2e-5 on 99.9 % (an accept / split decision then flips only within that distance of the tolerance), the guards
    (zero chord, |theta| > 120 degrees) identical."""
    rng = np.random.default_rng(18)
    n = 20000
    a0, a1 = rng.uniform(-2.4, 2.4, n), rng.uniform(-2.4, 2.4, n)      # angles of the end tangents against the chord (beyond 120 degrees: the guard)
    phi = rng.uniform(-np.pi, np.pi, n)
    chord = 10.0 ** rng.uniform(-2, 2.5, n)
    ch = np.stack([chord * np.cos(phi), chord * np.sin(phi)], 1)
    u0 = np.stack([np.cos(phi - a0), np.sin(phi - a0)], 1)
    u1 = np.stack([np.cos(phi + a1), np.sin(phi + a1)], 1)
    dt = 2.0 ** -rng.integers(0, 8, n).astype(np.float64)
    q0 = chord / dt * rng.uniform(0.1, 0.7, n)
    q1 = chord / dt * rng.uniform(0.1, 0.7, n)
    rows = np.concatenate([u0, u1, q0[:, None], q1[:, None], ch, dt[:, None]], 1).astype(np.float32)
    rows[0, 6:8] = 0.0                                                   # zero chord: forced split
    got = B.sx_eval(B.SX_EVAL_NODE_ERROR, rows)
    want = np.zeros(n, np.float32)
    out = np.zeros(4, np.float32)
    L = oracle.lib()
    for i in range(n):
        r = rows[i]
        L.so_fit_error_export(r[0:2].ctypes.data, r[2:4].ctypes.data, C.c_float(r[4]), C.c_float(r[5]), r[6:8].ctypes.data, C.c_float(r[8]), out.ctypes.data)
        want[i] = out[3]
    assert np.isinf(got[0]) and np.isinf(want[0])
    guard = np.isclose(want, 2.0 * np.hypot(rows[:, 6], rows[:, 7]), rtol=1e-6)       # the 120-degree guard: err = 2 chord
    fin = np.isfinite(want)
    rel = np.abs(got[fin].astype(np.float64) - want[fin]) / np.maximum(np.abs(want[fin]), 1e-12)
    print(f"node_error: max relative difference to the plain fp32 formulas {rel.max():.2e} over {int(fin.sum())} nodes ({int(guard.sum())} guarded)")
    q = np.quantile(rel, [0.5, 0.999])
    print(f"node_error: relative difference median {q[0]:.1e}, 99.9 % {q[1]:.1e}")
    assert rel.max() <= 1e-4 and q[1] <= 2e-5      # (the worst cases: the two area terms nearly cancel)
    assert guard.sum() > 100


def test_refined_density_integral_and_its_inverse(B):
    """SX_MODE_LINE_REFINED: the kernels' f against the closed form of L139 evaluated in double
    with numpy (not with the oracle), and f(f_inv_refined(u)) = u to fp32 accuracy -- two Newton steps from f_approx_inv --
    over the whole range, next to the zeros of the density (|x| = 1) included; the oracle's fp32 evaluation of the same
    formulas differs by rounding only."""
    def f64(x):
        a = np.abs(x)
        r = np.where(a <= 1, 0.5 * (a * np.sqrt(np.maximum(1 - a * a, 0)) + np.arcsin(np.minimum(a, 1))),
                     np.pi / 4 + 0.5 * (a * np.sqrt(np.maximum(a * a - 1, 0)) - np.arccosh(np.maximum(a, 1))))
        return np.sign(x) * r
    x = np.concatenate([np.linspace(-6, 6, 200001), 1 + np.logspace(-7, -1, 400), 1 - np.logspace(-7, -1, 400), -1 + np.logspace(-7, -1, 400),
                        -1 - np.logspace(-7, -1, 400), np.linspace(6, 300, 5000), [0.0, 1.0, -1.0]]).astype(np.float32)
    got = B.sx_eval(B.SX_EVAL_F_EXACT, x)
    want = f64(x.astype(np.float64))
    rel = np.abs(got - want) / np.maximum(1.0, np.abs(want))
    print(f"f_exact: max relative difference to the closed form in double {rel.max():.2e}")
    assert rel.max() <= 4e-7
    u = want.astype(np.float32)
    xr = B.sx_eval(B.SX_EVAL_F_INV_REFINED, u)
    back = np.abs(f64(xr.astype(np.float64)) - u.astype(np.float64)) / np.maximum(1.0, np.abs(u))
    print(f"f_inv_refined: max |f(f_inv(u)) - u| / max(1, |u|) {back.max():.2e}")
    assert back.max() <= 6e-7
    L = oracle.lib()
    idx = np.linspace(0, len(u) - 1, 4000).astype(int)
    worst = max(abs(float(L.so_f_inv_refined(C.c_float(u[i]))) - float(xr[i])) / max(1.0, abs(float(xr[i]))) * min(1.0, 4 * abs(abs(float(xr[i])) - 1.0) ** 0.5 + 1e-3) for i in idx)
    print(f"f_inv_refined: max difference to the oracle's, weighted by the density {worst:.2e}")
    assert worst <= 2e-6
