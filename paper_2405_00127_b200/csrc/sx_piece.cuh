// sx_piece.cuh -- one accepted Euler-spiral piece: parameters, subdivision plans, vertex evaluation.
//
// PAPER.md section 4 (parallel curve -> lines), 5 (-> arcs), 6 (evolutes), 7.3.1 (cusp), App. A.
// Same arithmetic discipline as sx_math.cuh: plain operators where an integer is decided, explicit
// fmaf in vertex evaluation.
#pragma once
#include "sx_math.cuh"

namespace sx {

// ---------------------------------------------------------------- section 4.2: f_approx and its inverse
// This is the PARAMETER path (curvature -> x -> u -> t): IEEE division / square root and CUDA's accurate sinf, asinf,
// cbrtf, because t is ill-conditioned in x on nearly circular pieces (dt/dx = L / (2 eta k1)): one ulp in f_approx
// moves a vertex by up to ~5e-4 px along the curve, and the oracle evaluates this path in fp32 too.
// f_approx (L149), odd extension (L157), middle piece sign-preserving (R-3b)
// (not inlined: four call sites per side plan; the kernels' working set has to stay inside the instruction cache)
__device__ __noinline__ float f_approx(float x) {
    // All four pieces are evaluated and one is selected: the threads of a warp sit on different pieces, and a
    // branch per piece would serialise them.  sin on [0, 0.88] by its Taylor series to y^11 (truncation 6e-9).
    const float a = fabsf(x);
    const float y = kC1 * fminf(a, 0.8f), y2 = y * y;
    float sn = fmaf(y2, -2.5052108385441720e-8f, 2.7557319223985893e-6f);
    sn = fmaf(sn, y2, -1.9841269841269841e-4f);
    sn = fmaf(sn, y2, 8.3333333333333333e-3f);
    sn = fmaf(sn, y2, -1.6666666666666667e-1f);
    sn = fmaf(sn * y2, y, y);
    const float r0 = sn / kC1;
    const float v = a - 1.0f, w = fabsf(v) * sqrtf(fabsf(v));
    const float r1 = kSqrt8Over3 * (v < 0.0f ? -w : w) + kQuarterPi;
    const float r2 = 0.6406f * a * a - 0.81f * a + kC2;
    const float r3 = 0.5f * a * a - 0.156f * a + kC3;
    const float r = a < 0.8f ? r0 : (a < 1.25f ? r1 : (a < 2.1f ? r2 : r3));
    return x < 0.0f ? -r : r;
}
// each piece of L149 solved for x
SX_DEV float f_approx_inv(float u) {
    float a = fabsf(u), r;
    if (a < kKnot0) r = asinf(kC1 * a) / kC1;
    else if (a < kKnot1) { float v = (a - kQuarterPi) / kSqrt8Over3; float w = cbrtf(fabsf(v)); w = w * w; r = 1.0f + (v < 0.0f ? -w : w); }
    else if (a < kKnot2) r = (0.81f + sqrtf(0.6561f - 2.5624f * (kC2 - a))) / 1.2812f;
    else r = 0.156f + sqrtf(0.024336f - 2.0f * (kC3 - a));
    return u < 0.0f ? -r : r;
}

#if SX_REFINED
// The "higher flattening quality" variant of L145 (reading R-22): the exact integral of L139 in the forward
// direction and, as its inverse, f_approx_inv refined by "two iterations of Newton solving".  Both in DOUBLE, rounded to
// fp32 once (as the angles of R-17): u -> x is ill-conditioned next to the zeros of the density (f' = sqrt|x^2 - 1| at
// |x| = 1), an fp32 evaluation would make the subdivision points depend on the last bit of asinf.  Where the guess lies in
// the middle piece of L149 the iteration runs on w(a) = sgn(e) |e|^(2/3), e = f(a) - pi/4, smooth and nearly linear
// across a = 1, with w'(a) = 2/3 f'(a) / |e|^(1/3) -> 2/3 sqrt(a + 1) / (sqrt(8)/3)^(1/3).
__device__ __noinline__ double f_exact_d(double a, double* deriv) {   // a >= 0
    const double d = sqrt(fabs((1.0 - a) * (1.0 + a)));
    *deriv = d;
    return a <= 1.0 ? 0.5 * (a * d + asin(a)) : 0.78539816339744830962 + 0.5 * (a * d - acosh(a));
}
SX_DEV float f_exact(float x) {
    double d;
    const float r = (float)f_exact_d((double)fabsf(x), &d);
    return x < 0.0f ? -r : r;
}
SX_DEV double signed_pow23(double v) { double c = cbrt(fabs(v)); c = c * c; return v < 0.0 ? -c : c; }
__device__ __noinline__ float f_inv_refined(float u) {
    const double au = fabs((double)u);
    double a = fabs((double)f_approx_inv(u));
    const bool middle = a >= 0.8 && a < 1.25;
    const double wt = signed_pow23(au - 0.78539816339744830962);
#pragma unroll 1
    for (int it = 0; it < 2; it++) {
        double d;
        const double fa = f_exact_d(a, &d);
        if (middle) {
            const double e = fa - 0.78539816339744830962, ce = cbrt(fabs(e));
            const double ratio = fabs(a - 1.0) < 1e-9 ? sqrt(a + 1.0) / 0.98057856349232452 : d / ce;   // cbrt(sqrt(8) / 3)
            a = a - (signed_pow23(e) - wt) / ((2.0 / 3.0) * ratio);
        } else {
            a = a - (fa - au) / d;
        }
    }
    const float r = (float)a;
    return u < 0.0f ? -r : r;
}
#define SX_OFF_REFINED(o) ((o).refined)
#else
#define SX_OFF_REFINED(o) false
#endif

// v -> sgn(v) |v|^1.5 and its inverse: the integral of sqrt|v| and the s ~ i^(2/3) rule of section 2.2 (L97)
SX_DEV float pow15(float v) { const float a = fabsf(v), w = a * sqrtf(a); return v < 0.0f ? -w : w; }
SX_DEV float pow15_inv(float w) { float c = cbrtf(fabsf(w)); c = c * c; return w < 0.0f ? -c : c; }
enum : int { kRuleUniform = 0, kRuleFApprox = 1, kRuleInflection = 2, kRuleCusp = 3 };

SX_DEV float clampf(float x, float lo, float hi) { return x < lo ? lo : (x > hi ? hi : x); }
SX_DEV int count_clamp(float n) { if (!(n >= 1.0f)) return 1; return (int)(n > kNMax ? kNMax : n); }

// ---------------------------------------------------------------- the piece
struct Piece {
    V2 base;         // segment start point P0 (global)
    V2 P3;           // segment end point (global), used when at1
    V2 la, lb;       // piece end points, local to base
    V2 ua, ub;       // unit tangents of the cubic at the piece ends
    V2 ch;           // chord lb - la
    float k0, k1, L; // total turning, GHI k1, arc length chord / c (App. A; kappa(s) = k0 + k1 s, s in [-1/2,1/2], R-1)
    bool at0, at1;   // the piece starts at t=0 / ends at t=1 of the segment
};

SX_DEV void piece_params(Piece& p, float th0, float th1, float chord) {
    float cc;
    ghi(th0, th1, &p.k1, &cc);
    p.k0 = th0 + th1;
    if (!(cc > 0.05f)) cc = 0.05f;
    p.L = chord / cc;
    if (!(p.L > 1e-12f)) p.L = 1e-12f;
}

SX_DEV float es_kappa(const Piece& p, float t) { return (p.k0 + p.k1 * (t - 0.5f)) / (p.L); }
// radius of curvature 1/kappa(t), for evolute points (section 6): one MUFU-grade division (the evolute is
// within |h| <= ~100 px of the curve, 2 ulp of the radius is ~1e-5 px)
SX_DEV float es_radius(const Piece& p, float t) { return div_fast(p.L, p.k0 + p.k1 * (t - 0.5f)); }

// ---------------------------------------------------------------- Euler-spiral integral (R-2)
// Z(t) = int_0^t exp(i phi(u)) du, phi(u) = (k0-k1/2) u + k1 u^2/2.  Evaluated from a per-piece table of
// anchors Z(k/K), k = 0..K (accumulated once per piece by 3-point Gauss-Legendre on each interval), plus a 3-point
// rule from the nearest anchor to t (|t - k/K| <= 1/(2K)).  K = 1, 2, 4 or 8 is chosen per piece so that the phase
// advances by at most ~1 rad per interval (max |phi'| <= |k0 - k1/2| + |k1|; on an accepted piece that is below
// ~20: |k0| <= 4.2 by the 120-degree guard R-4, k1 ~ 6 (th1 - th0)), where the 3-point rule's error, ~Phi^6 / 2e6
// of the interval, is at fp32 round-off.  Typical pieces (CAD scene: total turning ~0.3 rad) take K = 1: three sincos
// for Z(1) and three per interior vertex.
constexpr int kAnchors = 8;
struct Spiral {
    float wr, wi;                          // 1 / Z(1) (complex)
    float K;                               // number of intervals (1, 2, 4, 8)
    float zx[kAnchors + 1], zy[kAnchors + 1];
};
SX_DEV int es_intervals(float k0, float k1) {
    const float span = fabsf(k0 - 0.5f * k1) + fabsf(k1);
    return span <= 1.0f ? 1 : (span <= 2.0f ? 2 : (span <= 4.0f ? 4 : 8));
}

// sin and cos of a moderate argument (|x| < ~1e3): two-constant Cody-Waite reduction by pi/2 and the
// classic single-precision minimax kernels on [-pi/4, pi/4] (errors ~1e-7), all on the FMA pipe.
SX_DEV void sx_sincos(float x, float* s, float* c) {
    float k = rintf(x * 0.63661977236758134f);
    float r = fmaf(k, -1.5707963705062866f, x);
    r = fmaf(k, 4.3711390001862410e-8f, r);
    float z = r * r;
    float ps = fmaf(fmaf(fmaf(-1.9515295891e-4f, z, 8.3321608736e-3f), z, -1.6666654611e-1f), z * r, r);
    float pc = fmaf(fmaf(fmaf(2.443315711809948e-5f, z, -1.388731625493765e-3f), z, 4.166664568298827e-2f), z * z, fmaf(-0.5f, z, 1.0f));
    int q = (int)k;
    float ss = (q & 1) ? pc : ps, cc = (q & 1) ? ps : pc;
    *s = (q & 2) ? -ss : ss;
    *c = ((q + 1) & 2) ? -cc : cc;
}

// int_{m-hd}^{m+hd} exp(i phi(u)) du by 3-point Gauss-Legendre (hd may be negative)
SX_DEV float2 es_gl3_body(float a, float hk, float m, float hd) {
    const float d = hd * 0.77459666924148338f;
    const float u0 = m - d, u2 = m + d;
    float s0, c0, s1, c1, s2, c2;
    sx_sincos(u0 * fmaf(hk, u0, a), &s0, &c0);
    sx_sincos(m * fmaf(hk, m, a), &s1, &c1);
    sx_sincos(u2 * fmaf(hk, u2, a), &s2, &c2);
    return make_float2(hd * fmaf(0.55555555555555556f, c0 + c2, 0.88888888888888889f * c1),
                       hd * fmaf(0.55555555555555556f, s0 + s2, 0.88888888888888889f * s1));
}
// One non-inlined copy for the kernels whose working set has to stay inside the instruction cache (the table
// variant of the write kernel); INL = true inlines instead (the DIRECT variant is small enough, and calls cost
// it register spills).  Same operations either way, hence the same bits.
__device__ __noinline__ float2 es_gl3_call(float a, float hk, float m, float hd) { return es_gl3_body(a, hk, m, hd); }
template <bool INL>
SX_DEV float2 es_gl3(float a, float hk, float m, float hd) { return INL ? es_gl3_body(a, hk, m, hd) : es_gl3_call(a, hk, m, hd); }

// one half of the anchor table: half 0 integrates intervals [0, max(K/2,1)), half 1 intervals [K/2, K) (none when
// K = 1); cumulative sums relative to the half's start in hx/hy[0..count), the half's total in *tx, *ty.
// es_prepare = both halves by one thread; the write kernel gives one half to each of two threads.
template <bool INL = false>
SX_DEV int es_anchor_half(const Piece& p, int K, int half, float* hx, float* hy, float* tx, float* ty) {
    const float a = p.k0 - 0.5f * p.k1, hk = 0.5f * p.k1;
    const float w = 1.0f / (float)K;
    const int first = half ? K / 2 : 0, count = half ? K / 2 : (K > 1 ? K / 2 : 1);
    float zx = 0.0f, zy = 0.0f;
#pragma unroll
    for (int k = 0; k < kAnchors / 2; k++) {
        if (k < count) {
            const float2 in = es_gl3<INL>(a, hk, ((float)(first + k) + 0.5f) * w, 0.5f * w);
            zx += in.x; zy += in.y;
        }
        hx[k] = zx; hy[k] = zy;
    }
    *tx = zx; *ty = zy;
    return count;
}
// stores a half's anchors (offset by the other half's total for half 1) and, by half 0, Z(0), K and 1/Z(1)
SX_DEV void es_anchor_store(Spiral& sp, int K, int half, int count, const float* hx, const float* hy, float tx, float ty, float ox, float oy) {
    const int first = half ? K / 2 : 0;
    const float bx = half ? ox : 0.0f, by = half ? oy : 0.0f;
#pragma unroll
    for (int k = 0; k < kAnchors / 2; k++)
        if (k < count) { sp.zx[first + k + 1] = bx + hx[k]; sp.zy[first + k + 1] = by + hy[k]; }
    if (half == 0) {
        sp.zx[0] = 0.0f; sp.zy[0] = 0.0f;
        sp.K = (float)K;
        const float zx = tx + ox, zy = ty + oy;  // Z(1)
        const float den = 1.0f / fmaf(zx, zx, zy * zy);
        sp.wr = zx * den;
        sp.wi = -zy * den;
    }
}

SX_DEV void es_prepare(const Piece& p, Spiral& sp) {
    const int K = es_intervals(p.k0, p.k1);
    float ax[kAnchors / 2], ay[kAnchors / 2], bx[kAnchors / 2], by[kAnchors / 2], atx, aty, btx, bty;
    const int ca = es_anchor_half(p, K, 0, ax, ay, &atx, &aty);
    const int cb = es_anchor_half(p, K, 1, bx, by, &btx, &bty);
    es_anchor_store(sp, K, 1, cb, bx, by, btx, bty, atx, aty);
    es_anchor_store(sp, K, 0, ca, ax, ay, atx, aty, btx, bty);
}

SX_DEV float es_phi(const Piece& p, float t) { return t * fmaf(0.5f * p.k1, t, p.k0 - 0.5f * p.k1); }
// phi(tb) - phi(ta), evaluated as a difference (no cancellation)
SX_DEV float es_dphi(const Piece& p, float ta, float tb) { return (tb - ta) * fmaf(0.5f * p.k1, ta + tb, p.k0 - 0.5f * p.k1); }

// local position and unit tangent at piece fraction t in [0,1]: la + ch (x) Z(t)/Z(1) (L632)
template <bool INL = false>
SX_DEV void es_eval(const Piece& p, const Spiral& sp, float t, V2* pos, V2* tan) {
    const float a = p.k0 - 0.5f * p.k1, hk = 0.5f * p.k1;
    const float K = sp.K;
    float kf = rintf(t * K);
    kf = kf < 0.0f ? 0.0f : (kf > K ? K : kf);
    const int k = (int)kf;
    const float t0 = kf / K, hd = 0.5f * (t - t0);  // K is a power of two: exact
    const float2 in = es_gl3<INL>(a, hk, t0 + hd, hd);
    const float zx = sp.zx[k] + in.x, zy = sp.zy[k] + in.y;
    float wx = fmaf(zx, sp.wr, -zy * sp.wi), wy = fmaf(zx, sp.wi, zy * sp.wr);
    pos->x = fmaf(p.ch.x, wx, fmaf(-p.ch.y, wy, p.la.x));
    pos->y = fmaf(p.ch.x, wy, fmaf(p.ch.y, wx, p.la.y));
    float s, c;
    sx_sincos(es_phi(p, t), &s, &c);
    tan->x = fmaf(c, p.ua.x, -s * p.ua.y);
    tan->y = fmaf(s, p.ua.x, c * p.ua.y);
}

// canonical offset point of a global vertex V with unit tangent u: V + eta N, N = (-u.y, u.x)
SX_DEV V2 offset_point(V2 V, V2 u, float eta) { return v2(fmaf(eta, -u.y, V.x), fmaf(eta, u.x, V.y)); }

// point at signed normal distance r from the spiral at fraction t (r = eta: parallel curve; r = 1/kappa: evolute).
// At t = 0 and t = 1 the cubic's own point and tangent are used, so that adjacent pieces (and the join of the
// next segment) share bits.  The spiral is evaluated unconditionally and the end-point cases are selected
// afterwards, so that a warp evaluating a mix of interior and end vertices stays converged.
template <bool INL>
SX_DEV V2 normal_point_body(const Piece& p, const Spiral& sp, float t, float r) {
    V2 l, T;
    es_eval<INL>(p, sp, t, &l, &T);
    const bool e0 = t == 0.0f, e1 = t == 1.0f;
    if (e0) { l = p.la; T = p.ua; }
    if (e1) { l = p.lb; T = p.ub; }
    const float ox = fmaf(r, -T.y, l.x), oy = fmaf(r, T.x, l.y);
    V2 g = v2(p.base.x + ox, p.base.y + oy);
    if (e0 && p.at0) g = offset_point(p.base, p.ua, r);
    if (e1 && p.at1) g = offset_point(p.P3, p.ub, r);
    return g;
}
// (one non-inlined copy for the ring, the cusp point and the reference walk; see es_gl3)
__device__ __noinline__ V2 normal_point(const Piece& p, const Spiral& sp, float t, float r) { return normal_point_body<false>(p, sp, t, r); }
template <bool INL>
SX_DEV V2 normal_point_sel(const Piece& p, const Spiral& sp, float t, float r) { return INL ? normal_point_body<true>(p, sp, t, r) : normal_point(p, sp, t, r); }
SX_DEV V2 es_offset(const Piece& p, const Spiral& sp, float t, float eta) { return normal_point(p, sp, t, eta); }
SX_DEV V2 es_evolute(const Piece& p, const Spiral& sp, float t) { return normal_point(p, sp, t, es_radius(p, t)); }  // section 6

// ---------------------------------------------------------------- subdivision plans
struct OffPlan {   // rule: how the interior parameters are spaced (kRule*)
    int n; int rule; float ta, tb, ua, ub;
#if SX_REFINED
    bool refined;   // kRuleFApprox with the exact f and its Newton-refined inverse
#endif
};
struct EvoPlan { int n; bool uniform, cube; float ta, tb, wa, wb, skp; };   // cube: arc mode, the parameters are uniform in cbrt(sigma)

// offset range [ta,tb] of side eta (sections 4, 5): number of records and what the parameters need
SX_DEV OffPlan offset_plan(const Piece& p, float eta, float ta, float tb, int mode, float tol_fl) {
    OffPlan o;
    o.ta = ta; o.tb = tb; o.ua = 0.0f; o.ub = 0.0f; o.rule = kRuleUniform;
#if SX_REFINED
    o.refined = mode == kModeLineRefined;
#endif
    float n_f, ah = fabsf(eta);
    if (mode == kModeArc) {
        // L177 with s = L, kappa' = k1/L^2, scaled by the range fraction (R-12)
        float n_full = cbrt_fast(div_fast(p.L * fabsf(p.k1) * (1.0f + 0.4f * div_fast(fabsf(eta * p.k1), p.L)), 120.0f * tol_fl));
        n_f = ceilf((tb - ta) * n_full);
    } else {
        float ka = es_kappa(p, ta), kb = es_kappa(p, tb);
        float xa = 2.0f * eta * ka - 1.0f, xb = 2.0f * eta * kb - 1.0f;  // L125: inflection -> -1, cusp -> +1
        float xm = 0.5f * (xa + xb);
        float kp = div_fast(fabsf(p.k1), p.L * p.L);
        if (fabsf(xb - xa) < 0.015625f * fmaxf(1.0f, fabsf(xm))) {
            // x varies too little for a difference of two f_approx values in fp32 (R-7): the density sqrt|k (1 - k eta)|
            // is integrated locally.  km, gm: curvature and cusp factor at the middle of the range; m_infl, m_cusp: how far
            // km is from the inflection (k = 0) and from the cusp (k = 1/eta)
            float km = 0.5f * (ka + kb), dk = fabsf(kb - ka);
            float gm = 1.0f - km * eta;
            float m_infl = fabsf(km), m_cusp = fabsf(gm) / ah;
            if (dk <= 0.125f * fminf(m_infl, m_cusp)) {
                n_f = ceilf((tb - ta) * p.L * sqrt_fast(div_fast(fabsf(km * gm), 8.0f * tol_fl)));  // constant density (limit: L73)
            } else if (m_infl <= m_cusp) {
                // an inflection in or next to the range: int sqrt|k| ds = 2/3 |k|^1.5 / k' (section 2.2)
                o.ua = pow15(ka); o.ub = pow15(kb);
                n_f = ceilf(div_fast((2.0f / 3.0f) * fabsf(o.ub - o.ua) * sqrt_fast(fabsf(gm)), kp * sqrt_fast(8.0f * tol_fl)));
                o.rule = kRuleInflection;
            } else {
                // the range ends next to the cusp: the same with g = 1 - k eta
                o.ua = pow15(1.0f - ka * eta); o.ub = pow15(1.0f - kb * eta);
                n_f = ceilf(div_fast((2.0f / 3.0f) * fabsf(o.ub - o.ua) * sqrt_fast(fabsf(km)), ah * kp * sqrt_fast(8.0f * tol_fl)));
                o.rule = kRuleCusp;
            }
        } else {
#if SX_REFINED
            if (o.refined) { o.ua = f_exact(xa); o.ub = f_exact(xb); } else
#endif
            { o.ua = f_approx(xa); o.ub = f_approx(xb); }
            n_f = ceilf(div_fast(fabsf(o.ub - o.ua), 4.0f * kp * ah * sqrt_fast(ah) * sqrt_fast(8.0f * tol_fl)));  // L83
            o.rule = kRuleFApprox;
        }
    }
    o.n = count_clamp(n_f);
    return o;
}
// (ONE out-of-line copy per kernel: the side plan calls it for each of its ranges, the count pass and the simple writer for
// their single range; the kernels' working sets have to stay inside the instruction cache)
__device__ __noinline__ OffPlan offset_plan_call(float k0, float k1, float L, float eta, float ta, float tb, int mode, float tol_fl) {
    Piece p;
    p.k0 = k0; p.k1 = k1; p.L = L;
    return offset_plan(p, eta, ta, tb, mode, tol_fl);
}
// parameter of interior subdivision point i (0 < i < n)
SX_DEV float offset_t(const Piece& p, const OffPlan& o, float eta, int i) {
    float fr = (float)i / (float)o.n, t;
    if (o.rule == kRuleUniform) t = o.ta + fr * (o.tb - o.ta);
    else {
        float u = o.ua + fr * (o.ub - o.ua), kap;
#if SX_REFINED
        if (o.rule == kRuleFApprox && o.refined) kap = (f_inv_refined(u) + 1.0f) / (2.0f * eta); else
#endif
        if (o.rule == kRuleFApprox) kap = (f_approx_inv(u) + 1.0f) / (2.0f * eta);
        else if (o.rule == kRuleInflection) kap = pow15_inv(u);
        else kap = (1.0f - pow15_inv(u)) / eta;
        t = 0.5f + (kap * p.L - p.k0) / (p.k1);
    }
    return clampf(t, o.ta, o.tb);
}

// evolute range [ta,tb].  Lines: density |sigma|^-1/2, integral 2 sqrt(sigma), inverse squaring (L195).  Arcs (SURVEY
// 8(f)-1): the metric of section 5 (L171) applied to the evolute -- arc length element |kappa'| / kappa^2 dsigma, curvature
// kappa^3 / |kappa'|, d kappa_E / d s_E = 3 kappa^4 / |kappa'| -- gives n = 3^(4/3) |cbrt(sigma_b) - cbrt(sigma_a)| / cbrt(80 d),
// uniform in cbrt(sigma), inverse cubing (reading R-20: 80, not 120 -- the evolute's curvature derivative varies along an arc).
SX_DEV EvoPlan evolute_plan(const Piece& p, float ta, float tb, int mode, float tol_fl) {
    EvoPlan e;
    e.ta = ta; e.tb = tb; e.wa = 0.0f; e.wb = 0.0f; e.uniform = true; e.cube = mode == kModeArc;
    float ka = es_kappa(p, ta), kb = es_kappa(p, tb), km = 0.5f * (ka + kb);
    float kp = (fabsf(p.k1)) / (p.L * p.L);
    e.skp = ka < 0.0f ? -kp : kp;
    float n_f;
    const bool flat = fabsf(kb - ka) < 0.015625f * fabsf(km);
    if (mode == kModeArc) {
        if (flat) {
            n_f = ceilf((tb - ta) * p.L * cbrt_fast(div_fast(3.0f * kp * kp, 80.0f * tol_fl * km * km)));
        } else {
            e.wa = cbrtf(fabsf(ka) / kp);
            e.wb = cbrtf(fabsf(kb) / kp);
            n_f = ceilf(div_fast(4.326748710922225f * fabsf(e.wb - e.wa), cbrt_fast(80.0f * tol_fl)));
            e.uniform = false;
        }
        // at least one arc per pi/4 of turning over the range (the evolute turns with the spiral), then uniform in t
        const float dphi = fabsf((tb - ta) * (0.5f * p.k1 * (ta + tb) + (p.k0 - 0.5f * p.k1)));
        const float n_phi = ceilf(dphi / kQuarterPi);
        if (n_phi > n_f) { n_f = n_phi; e.uniform = true; }
    } else if (flat) {
        n_f = ceilf((tb - ta) * p.L * sqrt_fast(div_fast(fabsf(div_fast(kp, km)), 8.0f * tol_fl)));
    } else {
        e.wa = sqrtf(fabsf(ka) / kp);
        e.wb = sqrtf(fabsf(kb) / kp);
        n_f = ceilf(fabsf(2.0f * e.wb - 2.0f * e.wa) * sqrt_fast(div_fast(1.0f, 8.0f * tol_fl)));
        e.uniform = false;
    }
    e.n = count_clamp(n_f);
    return e;
}
SX_DEV float evolute_t(const Piece& p, const EvoPlan& e, int i) {
    float fr = (float)i / (float)e.n, t;
    if (e.uniform) t = e.ta + fr * (e.tb - e.ta);
    else {
        float w = e.wa + fr * (e.wb - e.wa);
        float kap = e.skp * w * w * (e.cube ? w : 1.0f);   // sigma = w^2 (lines) or w^3 (arcs)
        t = 0.5f + (kap * p.L - p.k0) / (p.k1);
    }
    return clampf(t, e.ta, e.tb);
}

// ---------------------------------------------------------------- cusp split of one side (Alg. 2, R-9)
// At most two ranges per side, at most one of them super-critical (L267: at most one cusp).
struct SidePlan {
    int nr;          // 0..2 ranges in increasing t
    bool sup[2];
    OffPlan off[2];
    EvoPlan evo;     // of the super-critical range, if any
    bool cusp_a, cusp_b;
    int total;       // records of this side
    float eta;       // signed offset of the side
    uint32_t seg;    // source segment (filled by the write kernel)
};

__device__ __noinline__ SidePlan side_plan(const Piece& p, float eta, int mode, float tol_fl) {
    SidePlan s;
    s.eta = eta; s.seg = 0u;
    float g0 = 1.0f - es_kappa(p, 0.0f) * eta, g1 = 1.0f - es_kappa(p, 1.0f) * eta;  // cusp0, cusp1 (L382-384)
    // L386.  The cusp is inside the piece iff g0 and g1 have strictly opposite signs (decided from the signs, not from the
    // product: g0 == 0 with g1 < 0 is a piece that is super-critical over its whole length)
    const bool has_cusp = (g0 > 0.0f && g1 < 0.0f) || (g0 < 0.0f && g1 > 0.0f);
    float tc = has_cusp ? g0 / (g0 - g1) : 1.0f;
    // regular on [0,tc], then super-critical on [tc,1] if there is a cusp; or super-critical on [0,tc], then regular on
    // [tc,1] if there is a cusp (L388-411)
    const bool first_sup = g0 < 0.0f || (g0 == 0.0f && g1 < 0.0f);
    s.nr = tc < 1.0f ? 2 : 1;
    s.sup[0] = first_sup;
    s.sup[1] = !first_sup;
    s.total = 0;
    s.cusp_a = s.cusp_b = false;
    s.evo.n = 0;
    s.off[0] = offset_plan_call(p.k0, p.k1, p.L, eta, 0.0f, tc, mode, tol_fl);
    s.total += s.off[0].n;
    float ea = 0.0f, eb = tc;
    if (s.nr == 2) {
        s.off[1] = offset_plan_call(p.k0, p.k1, p.L, eta, tc, 1.0f, mode, tol_fl);
        s.total += s.off[1].n;
        if (!first_sup) { ea = tc; eb = 1.0f; }
    } else {
        s.off[1] = s.off[0];
        s.sup[1] = false;
    }
    if (first_sup || s.nr == 2) {
        s.cusp_a = (ea != 0.0f);
        s.cusp_b = (eb != 1.0f);
        s.evo = evolute_plan(p, ea, eb, mode, tol_fl);
        s.total += 2 * s.evo.n + (s.cusp_a ? 0 : 2) + (s.cusp_b ? 0 : 2);
    }
    return s;
}

}  // namespace sx
