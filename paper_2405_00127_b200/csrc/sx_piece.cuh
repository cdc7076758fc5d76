// sx_piece.cuh -- one accepted Euler-spiral piece: parameters, subdivision plans, vertex evaluation.
//
// PAPER.md section 4 (parallel curve -> lines), 5 (-> arcs), 6 (evolutes), 7.3.1 (cusp), App. A.
// Same arithmetic discipline as sx_math.cuh: plain operators where an integer is decided, explicit
// fmaf in vertex evaluation.
#pragma once
#include "sx_math.cuh"

namespace sx {

// ---------------------------------------------------------------- section 4.2: f_approx and its inverse
// f_approx (L149), odd extension (L157), middle piece sign-preserving (R-3b)
SX_DEV float f_approx(float x) {
    float a = fabsf(x), r;
    if (a < 0.8f) r = sinf(kC1 * a) / kC1;
    else if (a < 1.25f) { float v = a - 1.0f; float w = fabsf(v) * sqrtf(fabsf(v)); r = kSqrt8Over3 * (v < 0.0f ? -w : w) + kQuarterPi; }
    else if (a < 2.1f) r = 0.6406f * a * a - 0.81f * a + kC2;
    else r = 0.5f * a * a - 0.156f * a + kC3;
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
    float wr, wi;    // 1 / Z(1) (complex), filled by es_prepare
    bool at0, at1;   // the piece starts at t=0 / ends at t=1 of the segment
    bool zready;
};

SX_DEV void piece_params(Piece& p, float th0, float th1, float chord) {
    float cc;
    ghi(th0, th1, &p.k1, &cc);
    p.k0 = th0 + th1;
    if (!(cc > 0.05f)) cc = 0.05f;
    p.L = chord / cc;
    if (!(p.L > 1e-12f)) p.L = 1e-12f;
    p.zready = false;
}

SX_DEV float es_kappa(const Piece& p, float t) { return (p.k0 + p.k1 * (t - 0.5f)) / p.L; }

// ---------------------------------------------------------------- Euler-spiral integral (R-2)
// Z(t) = int_0^t exp(i((k0-k1/2)u + k1 u^2/2)) du, 8-point Gauss-Legendre in fp32 (the phase spans at
// most a few radians on an accepted piece, where the 8-point rule is at fp32 round-off).
SX_DEV void es_integral(float k0, float k1, float t, float* zx, float* zy) {
    const float gx[4] = {0.18343464249564980f, 0.52553240991632899f, 0.79666647741362674f, 0.96028985649753623f};
    const float gw[4] = {0.36268378337836198f, 0.31370664587788729f, 0.22238103445337447f, 0.10122853629037626f};
    float a = k0 - 0.5f * k1, hk = 0.5f * k1, ht = 0.5f * t;
    float sx_ = 0.0f, sy_ = 0.0f;
#pragma unroll
    for (int j = 0; j < 4; j++) {
        float u0 = ht * (1.0f - gx[j]), u1 = ht * (1.0f + gx[j]);
        float p0 = u0 * fmaf(hk, u0, a), p1 = u1 * fmaf(hk, u1, a);
        float s0, c0, s1, c1;
        sincosf(p0, &s0, &c0);
        sincosf(p1, &s1, &c1);
        sx_ = fmaf(gw[j], c0 + c1, sx_);
        sy_ = fmaf(gw[j], s0 + s1, sy_);
    }
    *zx = ht * sx_;
    *zy = ht * sy_;
}

SX_DEV void es_prepare(Piece& p) {
    if (p.zready) return;
    float zx, zy;
    es_integral(p.k0, p.k1, 1.0f, &zx, &zy);
    float den = 1.0f / fmaf(zx, zx, zy * zy);
    p.wr = zx * den;
    p.wi = -zy * den;
    p.zready = true;
}

SX_DEV float es_phi(const Piece& p, float t) { return t * fmaf(0.5f * p.k1, t, p.k0 - 0.5f * p.k1); }
// phi(tb) - phi(ta), evaluated as a difference (no cancellation)
SX_DEV float es_dphi(const Piece& p, float ta, float tb) { return (tb - ta) * fmaf(0.5f * p.k1, ta + tb, p.k0 - 0.5f * p.k1); }

// local position and unit tangent at piece fraction t (0 < t < 1): la + ch (x) Z(t)/Z(1) (L632)
SX_DEV void es_eval(Piece& p, float t, V2* pos, V2* tan) {
    es_prepare(p);
    float zx, zy;
    es_integral(p.k0, p.k1, t, &zx, &zy);
    float wx = fmaf(zx, p.wr, -zy * p.wi), wy = fmaf(zx, p.wi, zy * p.wr);
    pos->x = fmaf(p.ch.x, wx, fmaf(-p.ch.y, wy, p.la.x));
    pos->y = fmaf(p.ch.x, wy, fmaf(p.ch.y, wx, p.la.y));
    float s, c;
    sincosf(es_phi(p, t), &s, &c);
    tan->x = fmaf(c, p.ua.x, -s * p.ua.y);
    tan->y = fmaf(s, p.ua.x, c * p.ua.y);
}

// canonical offset point of a global vertex V with unit tangent u: V + eta N, N = (-u.y, u.x)
SX_DEV V2 offset_point(V2 V, V2 u, float eta) { return v2(fmaf(eta, -u.y, V.x), fmaf(eta, u.x, V.y)); }

// point at signed normal distance r from the spiral at fraction t (r = eta: parallel curve; r = 1/kappa: evolute).
// At t = 0 and t = 1 the cubic's own point and tangent are used, so that adjacent pieces (and the join of the
// next segment) share bits.  The spiral is evaluated unconditionally and the end-point cases are selected
// afterwards, so that a warp evaluating a mix of interior and end vertices stays converged.
SX_DEV V2 normal_point(Piece& p, float t, float r) {
    V2 l, T;
    es_eval(p, t, &l, &T);
    const bool e0 = t == 0.0f, e1 = t == 1.0f;
    if (e0) { l = p.la; T = p.ua; }
    if (e1) { l = p.lb; T = p.ub; }
    const float ox = fmaf(r, -T.y, l.x), oy = fmaf(r, T.x, l.y);
    V2 g = v2(p.base.x + ox, p.base.y + oy);
    if (e0 && p.at0) g = offset_point(p.base, p.ua, r);
    if (e1 && p.at1) g = offset_point(p.P3, p.ub, r);
    return g;
}
SX_DEV V2 es_offset(Piece& p, float t, float eta) { return normal_point(p, t, eta); }
SX_DEV V2 es_evolute(Piece& p, float t) { return normal_point(p, t, 1.0f / es_kappa(p, t)); }  // section 6

// ---------------------------------------------------------------- subdivision plans
struct OffPlan { int n; bool uniform; float ta, tb, ua, ub; };
struct EvoPlan { int n; bool uniform; float ta, tb, wa, wb, skp; };

// offset range [ta,tb] of side eta (sections 4, 5): number of records and what the parameters need
SX_DEV OffPlan offset_plan(const Piece& p, float eta, float ta, float tb, int mode, float tol_fl) {
    OffPlan o;
    o.ta = ta; o.tb = tb; o.ua = 0.0f; o.ub = 0.0f; o.uniform = true;
    float n_f, ah = fabsf(eta);
    if (mode == kModeArc) {
        // L177 with s = L, kappa' = k1/L^2, scaled by the range fraction (R-12)
        float n_full = cbrtf(p.L * fabsf(p.k1) * (1.0f + 0.4f * fabsf(eta * p.k1) / p.L) / (120.0f * tol_fl));
        n_f = ceilf((tb - ta) * n_full);
    } else {
        float ka = es_kappa(p, ta), kb = es_kappa(p, tb);
        float xa = 2.0f * eta * ka - 1.0f, xb = 2.0f * eta * kb - 1.0f;  // L125: inflection -> -1, cusp -> +1
        float xm = 0.5f * (xa + xb);
        if (fabsf(xb - xa) < 0.015625f * fmaxf(1.0f, fabsf(xm))) {
            float km = 0.5f * (ka + kb);  // constant density sqrt|k(1-k eta)| (R-7; limit is L73)
            n_f = ceilf((tb - ta) * p.L * sqrtf(fabsf(km * (1.0f - km * eta)) / (8.0f * tol_fl)));
        } else {
            o.ua = f_approx(xa);
            o.ub = f_approx(xb);
            float kp = fabsf(p.k1) / (p.L * p.L);
            n_f = ceilf(fabsf(o.ub - o.ua) / (4.0f * kp * ah * sqrtf(ah) * sqrtf(8.0f * tol_fl)));  // L83
            o.uniform = false;
        }
    }
    o.n = count_clamp(n_f);
    return o;
}
// parameter of interior subdivision point i (0 < i < n)
SX_DEV float offset_t(const Piece& p, const OffPlan& o, float eta, int i) {
    float fr = (float)i / (float)o.n, t;
    if (o.uniform) t = o.ta + fr * (o.tb - o.ta);
    else {
        float u = o.ua + fr * (o.ub - o.ua);
        float x = f_approx_inv(u);
        float kap = (x + 1.0f) / (2.0f * eta);
        t = 0.5f + (kap * p.L - p.k0) / p.k1;
    }
    return clampf(t, o.ta, o.tb);
}

// evolute range [ta,tb]: density |sigma|^-1/2, integral 2 sqrt(sigma), inverse squaring (L195)
SX_DEV EvoPlan evolute_plan(const Piece& p, float ta, float tb, float tol_fl) {
    EvoPlan e;
    e.ta = ta; e.tb = tb; e.wa = 0.0f; e.wb = 0.0f; e.uniform = true;
    float ka = es_kappa(p, ta), kb = es_kappa(p, tb), km = 0.5f * (ka + kb);
    float kp = fabsf(p.k1) / (p.L * p.L);
    e.skp = ka < 0.0f ? -kp : kp;
    float n_f;
    if (fabsf(kb - ka) < 0.015625f * fabsf(km)) {
        n_f = ceilf((tb - ta) * p.L * sqrtf(fabsf(kp / km) / (8.0f * tol_fl)));
    } else {
        e.wa = sqrtf(fabsf(ka) / kp);
        e.wb = sqrtf(fabsf(kb) / kp);
        n_f = ceilf(fabsf(2.0f * e.wb - 2.0f * e.wa) * sqrtf(1.0f / (8.0f * tol_fl)));
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
        float kap = e.skp * w * w;
        t = 0.5f + (kap * p.L - p.k0) / p.k1;
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

SX_DEV SidePlan side_plan(const Piece& p, float eta, int mode, float tol_fl) {
    SidePlan s;
    s.eta = eta; s.seg = 0u;
    float g0 = 1.0f - es_kappa(p, 0.0f) * eta, g1 = 1.0f - es_kappa(p, 1.0f) * eta;  // cusp0, cusp1 (L382-384)
    float tc = (g0 * g1 >= 0.0f) ? 1.0f : g0 / (g0 - g1);                            // L386
    float ra[2], rb[2];
    s.nr = 0;
    s.sup[0] = s.sup[1] = false;
    if (g0 >= 0.0f) { ra[s.nr] = 0.0f; rb[s.nr] = tc; s.sup[s.nr] = false; s.nr++; }
    if (g0 < 0.0f || tc < 1.0f) {
        if (g0 >= 0.0f) { ra[s.nr] = tc; rb[s.nr] = 1.0f; } else { ra[s.nr] = 0.0f; rb[s.nr] = tc; }
        s.sup[s.nr] = true; s.nr++;
    }
    if (g0 < 0.0f && tc < 1.0f) { ra[s.nr] = tc; rb[s.nr] = 1.0f; s.sup[s.nr] = false; s.nr++; }
    s.total = 0;
    s.cusp_a = s.cusp_b = false;
    s.evo.n = 0;
#pragma unroll
    for (int r = 0; r < 2; r++) {
        if (r < s.nr) {
            s.off[r] = offset_plan(p, eta, ra[r], rb[r], mode, tol_fl);
            s.total += s.off[r].n;
            if (s.sup[r]) {
                s.cusp_a = (ra[r] != 0.0f);
                s.cusp_b = (rb[r] != 1.0f);
                s.evo = evolute_plan(p, ra[r], rb[r], tol_fl);
                s.total += 2 * s.evo.n + (s.cusp_a ? 0 : 2) + (s.cusp_b ? 0 : 2);
            }
        }
    }
    return s;
}

}  // namespace sx
