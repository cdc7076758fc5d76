// sx_math.cuh -- device functions of the stroke-expansion kernels (sm_100a).
//
// The curve mathematics of "GPU-friendly Stroke Expansion" (PAPER.md sections 2, 4-7, App. A) as used
// by the count kernel (b) and the write kernel (d).  Citations are PAPER.md line numbers; "R-n" are
// the readings listed in DESIGN.md section 3.
//
// Arithmetic discipline: this translation unit is compiled with -fmad=false, so
// every a*b+c written with plain operators is two IEEE roundings and every fused multiply-add is an
// explicit fmaf().  Everything that decides an integer (accept/split of Alg. 2, the Euler-spiral
// parameters, subdivision counts, subdivision parameters t_i) uses plain operators in a fixed order,
// identical in the count and the write kernel, so the two passes agree bit for bit.  Vertex
// coordinates are evaluated in segment-local coordinates with explicit fmaf and the segment base
// point is added last (fp32 ulp at 16384 px is 9.8e-4 px).
#pragma once
// SX_REFINED: the translation unit sx_refined.cu compiles these headers a second time, in namespace sx_refined, with the
// code of SX_MODE_LINE_REFINED switched on; the kernels of the other modes do not carry it (they are bound
// by the instruction cache: DESIGN.md section 5).
#ifndef SX_REFINED
#define SX_REFINED 0
#endif
#include <stdint.h>
#include <math.h>

#ifndef SX_DEV
#define SX_DEV __device__ __forceinline__
#endif

namespace sx {

// ---------------------------------------------------------------- constants (R-13)
constexpr float kEpsQ2 = 1e-12f;             // (1e-6 px)^2: "near zero" derivative, L251
constexpr float kDeltaT = 1e-4f;             // parameter perturbation relative to dt, L251
constexpr float kDtMin = 1.0f / 65536.0f;    // deepest level of Alg. 2 (paper silent)
constexpr float kNMax = 65535.0f;            // clamp of a single subdivision count
constexpr float kC1 = 1.0976991822760038f;   // L155
constexpr float kC2 = 0.9148117935952064f;
constexpr float kC3 = 0.16145779359520596f;
constexpr float kPi = 3.14159265358979323846f;
constexpr float kQuarterPi = 0.78539816339744830962f;
constexpr float kSqrt8Over3 = 0.94280904158206336587f;  // sqrt(8)/3, L149
constexpr float kKnot0 = 0.70107076f;        // f_approx(0.8), f_approx(1.25), f_approx(2.1)
constexpr float kKnot1 = 0.90324929f;
constexpr float kKnot2 = 2.03885779f;

enum : uint32_t { kOffset = 0, kOffsetRev = 1, kEvolute = 2, kConnector = 3, kJoinOuter = 4, kJoinInner = 5, kCap = 6, kClose = 7, kPlus = 8 };
enum : int { kJoinMiter = 0, kJoinRound = 1, kJoinBevel = 2, kCapButt = 0, kCapSquare = 1, kCapRound = 2, kModeLine = 0, kModeArc = 1, kModeLineRefined = 2 };   // 2: lines with the exact density integral (L145, R-22)

// ---------------------------------------------------------------- float2 helpers (plain operators: no contraction)
struct V2 { float x, y; };
SX_DEV V2 v2(float x, float y) { V2 r; r.x = x; r.y = y; return r; }
SX_DEV V2 operator-(V2 a, V2 b) { return v2(a.x - b.x, a.y - b.y); }
SX_DEV float dot(V2 a, V2 b) { return a.x * b.x + a.y * b.y; }
SX_DEV float cross(V2 a, V2 b) { return a.x * b.y - a.y * b.x; }
SX_DEV float len2(V2 a) { return a.x * a.x + a.y * a.y; }
// Two grades of arithmetic.  Plain operators, sqrtf, sinf, asinf ... are IEEE / CUDA's
// accurate library versions (no -use_fast_math): used for everything a coordinate or a subdivision parameter is
// computed from.  The *_fast helpers below (MUFU approximations, ~2 ulp) are used where a value only feeds a
// tolerance comparison or a ceil(): the cubic -> spiral error estimate and the subdivision-count formulas.
SX_DEV float div_fast(float a, float b) { return __fdividef(a, b); }
SX_DEV float sqrt_fast(float a) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a)); return r; }
SX_DEV float cbrt_fast(float a) { return a > 0.0f ? __powf(a, 0.33333333333333333f) : 0.0f; }
// (not inlined: IEEE square root and two divisions, a dozen call sites)
__device__ __noinline__ V2 unit(V2 a) { float l = sqrtf(len2(a)); return v2(a.x / l, a.y / l); }

SX_DEV float u2f(uint32_t u) { return __uint_as_float(u); }
SX_DEV int ctz32(uint32_t x) { return __ffs((int)x) - 1; }

// ---------------------------------------------------------------- per-call parameters (kernel argument, by value)
struct Params {
    const uint8_t* tags;
    const float* pts;        // xy interleaved
    const uint8_t* styles;   // sx_style[], 16 B each
    const uint32_t* pt_off;  // from the tag scan
    const uint32_t* path_idx;
    const uint32_t* sp_first;
    float A[6];              // affine (L462)
    float scale;             // sqrt|det A| (R-14)
    float tol_es, tol_fl;    // 0.1 / 0.8 of the tolerance (R-13)
    int mode;
    uint32_t n_tags;
};

// ---------------------------------------------------------------- segment in device space, local to P0
struct Seg {
    int kind;         // 1 line, 2 quad, 3 cubic
    V2 P0, P3;        // global end points
    V2 c1, c2, c3;    // control points relative to P0, after degree elevation (L349)
    V2 ts, te;        // unit start / end tangents
    bool degenerate;  // all control points coincide
};

// transform (R-14): x' = fma(a,x,fma(c,y,e)), y' = fma(b,x,fma(d,y,f))
SX_DEV V2 xform(const float* A, float x, float y) {
    return v2(fmaf(A[0], x, fmaf(A[2], y, A[4])), fmaf(A[1], x, fmaf(A[3], y, A[5])));
}

// first control-polygon leg that is not (near) zero, else (1,0) (R-5): the limit tangent of the curve
SX_DEV V2 pick_tangent(V2 a, V2 b, V2 c, bool* degenerate) {
    // the leg is SELECTED first and normalised once (three normalisations behind three branches cost a third of the
    // segment writer's instructions)
    const bool ua = len2(a) >= kEpsQ2, ub = len2(b) >= kEpsQ2, uc = len2(c) >= kEpsQ2;
    const V2 d = ua ? a : (ub ? b : c);
    *degenerate = !(ua || ub || uc);
    const V2 u = unit(d);
    return *degenerate ? v2(1.0f, 0.0f) : u;
}

SX_DEV float2 ldg2(const float* p) { return __ldg(reinterpret_cast<const float2*>(p)); }

// pt = index of the segment's first point (pt_off[i] from the tag scan).  Branch-free: the three kinds (line, quadratic,
// cubic) differ in selects only, so that a warp over a mixed tile stays converged (and the code stays small).
SX_DEV Seg load_segment_at(const Params& P, uint32_t pt, uint32_t tag) {
    Seg s;
    const int cnt = tag & 3;
    const bool quad = cnt == 2, cubic = cnt == 3;
    const float* p = P.pts + 2 * (uint64_t)pt;
    const float2 a0 = ldg2(p), a1 = ldg2(p + 2), a2 = ldg2(p + (cnt >= 2 ? 4 : 2)), a3 = ldg2(p + (cubic ? 6 : (quad ? 4 : 2)));
    const V2 q0 = xform(P.A, a0.x, a0.y), q1 = xform(P.A, a1.x, a1.y), q2 = xform(P.A, a2.x, a2.y), q3 = xform(P.A, a3.x, a3.y);
    s.kind = cnt;
    s.P0 = q0; s.P3 = q3;   // (q3 repeats the last point of a line or a quadratic)
    const V2 a = q1 - q0, b = q2 - q0, d = q3 - q0;
    // degree elevation (L349).  line: c1 = d / 3, c2 = 2/3 d; quadratic: c1 = 2/3 a, c2 = b + 2/3 (a - b); cubic: as given
    const V2 c1l = v2(a.x / 3.0f, a.y / 3.0f), c2l = v2(a.x * (2.0f / 3.0f), a.y * (2.0f / 3.0f));
    const V2 c2q = v2(b.x + (a.x - b.x) * (2.0f / 3.0f), b.y + (a.y - b.y) * (2.0f / 3.0f));
    s.c1 = cubic ? a : (quad ? c2l : c1l);
    s.c2 = cubic ? b : (quad ? c2q : c2l);
    s.c3 = d;
    // the legs the limit tangents are picked from (R-5).  line: d, d, d both ways; quadratic: a, b, b / b - a, b, b;
    // cubic: c1, c2, c3 / c3 - c2, c3 - c1, c3
    bool dg, dg2;
    s.ts = pick_tangent(a, b, d, &dg);
    s.te = pick_tangent(cubic ? d - b : (quad ? b - a : d), cubic ? d - a : d, d, &dg2);
    s.degenerate = dg;
    return s;
}

// start point and start tangent only (join partner / start cap owner)
SX_DEV Seg load_segment(const Params& P, uint32_t i, uint32_t tag) { return load_segment_at(P, P.pt_off[i], tag); }

SX_DEV void load_segment_start_at(const Params& P, uint32_t pt, uint32_t tag, V2* P0, V2* ts) {
    // = load_segment_at(P, pt, tag).{P0, ts} without the end tangent: the same legs in the same order
    const uint32_t cnt = tag & 3u;
    const float* p = P.pts + 2 * (uint64_t)pt;
    auto a0 = ldg2(p), a1 = ldg2(p + 2);
    const V2 q0 = xform(P.A, a0.x, a0.y), q1 = xform(P.A, a1.x, a1.y);
    V2 l1 = q1 - q0, l2 = l1, l3 = l1;  // line: d, d, d
    if (cnt >= 2u) {
        auto a2 = ldg2(p + 4);
        const V2 q2 = xform(P.A, a2.x, a2.y);
        l2 = q2 - q0; l3 = l2;              // quadratic: a, b, b
        if (cnt == 3u) {
            auto a3 = ldg2(p + 6);
            const V2 q3 = xform(P.A, a3.x, a3.y);
            l3 = q3 - q0;                   // cubic: c1, c2, c3
        }
    }
    bool dg;
    *P0 = q0;
    *ts = pick_tangent(l1, l2, l3, &dg);
}
SX_DEV void load_segment_start(const Params& P, uint32_t j, V2* P0, V2* ts) { load_segment_start_at(P, P.pt_off[j], P.tags[j], P0, ts); }

// ---------------------------------------------------------------- cubic evaluation (Alg. 2), Bernstein form
SX_DEV V2 cubic_pos(const Seg& s, float t) {
    float mt = 1.0f - t;
    float a = 3.0f * mt * mt * t, b = 3.0f * mt * t * t, c = t * t * t;
    return v2(a * s.c1.x + b * s.c2.x + c * s.c3.x, a * s.c1.y + b * s.c2.y + c * s.c3.y);
}
SX_DEV V2 cubic_q(const Seg& s, float t) {  // C'(t)/3
    float mt = 1.0f - t;
    float a = mt * mt, b = 2.0f * mt * t, c = t * t;
    V2 d0 = s.c1, d1 = s.c2 - s.c1, d2 = s.c3 - s.c2;
    return v2(a * d0.x + b * d1.x + c * d2.x, a * d0.y + b * d1.y + c * d2.y);
}
// position, |q| and unit tangent at t with the near-zero-derivative rule of L251 (R-5)
SX_DEV void eval_cubic(const Seg& s, float t, float dt, V2* pos, float* qmag, V2* u) {
    V2 q = cubic_q(s, t);
    float q2 = len2(q);
    *qmag = sqrtf(q2);
    if (t == 1.0f) { *pos = s.c3; *u = s.te; return; }
    *pos = cubic_pos(s, t);
    if (q2 >= kEpsQ2) { *u = v2(q.x / *qmag, q.y / *qmag); return; }
    V2 qp = cubic_q(s, t - kDeltaT * dt);
    *u = (len2(qp) > 0.0f) ? unit(qp) : v2(1.0f, 0.0f);
}

// ---------------------------------------------------------------- section 7.1: cubic -> Euler spiral error estimate
// L215 unit-chord normalisation; L217 d-bar; L221 e1; L225 area; L227 e2; L229 e3; guards R-4.
//
// Angles (reading R-17): th = the fp32 value nearest to the angle of (x, y): atan2 in double, rounded once.  The
// oracle computes the same number with its own libm; the two agree unless the double result falls within a few
// ulp(double) of a rounding boundary of fp32 (probability ~1e-8 per call).  th0, th1 fix k0, k1, L and hence every
// subdivision parameter and every evolute radius of the piece.
//
// Own double-precision atan2 (the library's costs ~140 instructions per call, two calls per piece): with
// mn = min(|x|, |y|), mx = max(|x|, |y|) and c = k/4 the quarter nearest to mn/mx,
//     atan(mn/mx) = atan(c) + atan(t),  t = (mn - c mx) / (mx + c mn),  |t| <= 0.125 (+ the rounding of k),
// one division (reciprocal seed from the fp32 unit, two Newton steps, one residual correction: full double accuracy)
// and the Taylor series of atan to t^19 (remainder < 2^-63 / 21): error below 2 ulp(double) in all.
SX_DEV float rcp_fast(float a) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a)); return r; }
SX_DEV float rsqrt_fast(float a) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a)); return r; }

// 1e-30 < max(|x|, |y|) < 1e30 (the kernels' arguments are cross / dot products of unit vectors)
SX_DEV float atan2_r_core(float y, float x) {
    const float ax = fabsf(x), ay = fabsf(y);
    const float mxf = fmaxf(ax, ay), mnf = fminf(ax, ay);
    const float kf = rintf(4.0f * (mnf * rcp_fast(mxf)));   // 0 .. 4
    const double c = 0.25 * (double)kf;
    // atan(k / 4), k = 0 .. 4
    const double at = kf < 0.5f ? 0.0 : (kf < 1.5f ? 0.24497866312686415417 : (kf < 2.5f ? 0.46364760900080611621 : (kf < 3.5f ? 0.64350110879328438680 : 0.78539816339744830962)));
    const double mx = (double)mxf, mn = (double)mnf;
    const double num = fma(-c, mx, mn), den = fma(c, mn, mx);   // den in [mx, 2 mx]
    double r = (double)rcp_fast((float)den);
    r = fma(r, fma(-den, r, 1.0), r);
    r = fma(r, fma(-den, r, 1.0), r);
    double t = num * r;
    t = fma(r, fma(-den, t, num), t);
    const double z = t * t;
    double p = -1.0 / 19.0;
    p = fma(p, z, 1.0 / 17.0);
    p = fma(p, z, -1.0 / 15.0);
    p = fma(p, z, 1.0 / 13.0);
    p = fma(p, z, -1.0 / 11.0);
    p = fma(p, z, 1.0 / 9.0);
    p = fma(p, z, -1.0 / 7.0);
    p = fma(p, z, 1.0 / 5.0);
    p = fma(p, z, -1.0 / 3.0);
    double a = at + fma(t * z, p, t);
    if (ay > ax) a = 1.57079632679489661923 - a;
    if (x < 0.0f) a = 3.14159265358979323846 - a;
    const float f = (float)a;
    return y < 0.0f ? -f : f;
}
// (one out-of-line copy for the call sites that are not hot; the count pass inlines its two calls per piece so that the
// two dependent chains interleave)
__device__ __noinline__ float atan2_r(float y, float x) {
    const float m = fmaxf(fabsf(x), fabsf(y));
    if (!(m > 1e-30f) || !(m < 1e30f)) return (float)atan2((double)y, (double)x);   // zeros, denormals, huge, infinities, NaN: the library
    return atan2_r_core(y, x);
}

// atan2 for the accept/split DECISION of Alg. 2 only (the error estimate of section 7.1 is compared with a tolerance):
// approximate division, odd minimax polynomial on [0, 1] (max error ~1e-7 rad).  The angles a piece is built from come
// from atan2_r.  (x, y) is (cos, sin) of an angle: max(|x|, |y|) >= 0.7.
SX_DEV float atan2_dec(float y, float x) {
    const float ax = fabsf(x), ay = fabsf(y);
    const float mx = fmaxf(ax, ay), mn = fminf(ax, ay);
    const float a = mn * rcp_fast(fmaxf(mx, 1e-30f));
    const float s = a * a;
    float r = fmaf(s, 0.00282363896258175373077393f, -0.0159569028764963150024414f);
    r = fmaf(r, s, 0.0425049886107444763183594f);
    r = fmaf(r, s, -0.0748900920152664184570312f);
    r = fmaf(r, s, 0.106347933411598205566406f);
    r = fmaf(r, s, -0.142027363181114196777344f);
    r = fmaf(r, s, 0.199926957488059997558594f);
    r = fmaf(r, s, -0.333331018686294555664062f);
    r = fmaf(r * s, a, a);
    if (ay > ax) r = 1.57079637050628662109375f - r;
    if (x < 0.0f) r = 3.14159274101257324218750f - r;
    return y < 0.0f ? -r : r;
}

// section 7.1 with the decision-grade angles: the estimated error of the node (u0, q0mag) -> (u1, q1mag) over chord ch.
// Everything here feeds one comparison with the tolerance: MUFU-grade reciprocals and square roots, explicit fused
// multiply-adds, area(d0, d1) - area(db0, db1) expanded term by term (L225-227).
SX_DEV float node_error(V2 u0, V2 u1, float q0mag, float q1mag, V2 ch, float dt) {
    const float chord2 = fmaf(ch.x, ch.x, ch.y * ch.y);
    if (chord2 < kEpsQ2) return INFINITY;
    const float rc = rsqrt_fast(chord2), chord = chord2 * rc;
    const float ucx = ch.x * rc, ucy = ch.y * rc;
    const float s0 = fmaf(u0.x, ucy, -(u0.y * ucx)), c0 = fmaf(u0.x, ucx, u0.y * ucy);
    const float s1 = fmaf(ucx, u1.y, -(ucy * u1.x)), c1 = fmaf(ucx, u1.x, ucy * u1.y);
    if (c0 < -0.5f || c1 < -0.5f) return 2.0f * chord;
    const float th0 = atan2_dec(s0, c0), th1 = atan2_dec(s1, c1);
    const float sc = dt * rc;
    const float dd0 = (2.0f / 3.0f) * rcp_fast(1.0f + c0) - q0mag * sc, dd1 = (2.0f / 3.0f) * rcp_fast(1.0f + c1) - q1mag * sc;   // d-bar - d (L217)
    const float d0 = q0mag * sc, d1 = q1mag * sc, db0 = dd0 + d0, db1 = dd1 + d1;
    const float s01 = fmaf(s0, c1, c0 * s1);
    // area(d0, d1) - area(db0, db1), area(a, b) = 3/20 (2 a s0 + 2 b s1 - a b s01)
    const float darea = fmaf(0.15f * s01, fmaf(db0, db1, -(d0 * d1)), -0.3f * fmaf(dd0, s0, dd1 * s1));
    const float ksum = fabsf(th0 + th1), kdif = fabsf(th0 - th1);
    const float k2 = ksum * ksum;
    const float e1 = k2 * fmaf(4.6255e-6f * k2, ksum, 7.5e-3f * kdif);
    const float e3 = fmaf(0.005f, ksum, 0.07f * kdif) * sqrt_fast(fmaf(dd0, dd0, dd1 * dd1));
    return chord * (e1 + fmaf(1.55f, fabsf(darea), e3));
}


// the end-tangent angles of an ACCEPTED piece (L211-213: th0 from the start tangent to the chord, th1 from the chord to
// the end tangent) and its chord length; a zero chord (accepted at the deepest level only) has th0 = th1 = 0
SX_DEV void piece_angles(V2 u0, V2 u1, V2 ch, float* th0, float* th1, float* chord_out) {
    const float chord2 = len2(ch);
    const float chord = sqrtf(chord2);
    *chord_out = chord;
    *th0 = 0.0f; *th1 = 0.0f;
    if (chord2 < kEpsQ2) return;
    const V2 uc = v2(ch.x / chord, ch.y / chord);
    *th0 = atan2_r(cross(u0, uc), dot(u0, uc));
    *th1 = atan2_r(cross(uc, u1), dot(uc, u1));
}

// ---------------------------------------------------------------- Appendix A: geometric Hermite interpolation
// k = th0+th1, D = th1-th0 (L634); k1 (L636) and chord/arc ratio c (L641-651), terms in the paper's order.
SX_DEV void ghi(float th0, float th1, float* k1_out, float* c_out) {
    float k = th0 + th1, D = th1 - th0;
    float k2 = k * k, k4 = k2 * k2, k6 = k4 * k2;
    float D2 = D * D, D3 = D2 * D, D4 = D2 * D2, D5 = D4 * D, D6 = D4 * D2, D7 = D6 * D;
    float k1 = 6.0f * D;
    k1 -= D3 * (1.0f / 70.0f);
    k1 -= D5 * (1.0f / 10780.0f);
    k1 += D7 * 2.769178184818219e-7f;
    k1 -= k2 * D * (1.0f / 10.0f);
    k1 += k2 * D3 * (1.0f / 4200.0f);
    k1 += k2 * D5 * 1.6959677820260655e-5f;
    k1 -= k4 * D * (1.0f / 1400.0f);
    k1 += k4 * D3 * 6.84915970574303e-5f;
    k1 -= k6 * D * 7.936475029053326e-6f;
    float c = 1.0f;
    c -= D2 * (1.0f / 40.0f);
    c += D4 * 0.00034226190482569864f;
    c -= D6 * 1.9349474568904524e-6f;
    c -= k2 * (1.0f / 24.0f);
    c += k2 * D2 * 0.0024702380951963226f;
    c -= k2 * D4 * 3.7297408997537985e-5f;
    c += k4 * (1.0f / 1920.0f);
    c -= k4 * D2 * 4.87350869747975e-5f;
    c -= k6 * 3.1001936068463107e-6f;
    *k1_out = k1;
    *c_out = c;
}

}  // namespace sx
