/*
 * stroke_oracle.c -- CPU ORACLE for "GPU-friendly Stroke Expansion" (arxiv 2405.00127).
 *
 * TEST INFRASTRUCTURE ONLY.  This file is the plain, slow, sequential restatement of the
 * paper's method that the CUDA path is compared against.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
 * code, header, table or constant generator with paper_2405_00127_b200/csrc/.
 *
 * Citations are PAPER.md line numbers (L...) plus the section / equation / algorithm; readings of
 * points where the paper is silent or garbled are the "R-n" items of DESIGN.md section 3.
 *
 * Arithmetic discipline (R-16): everything that DECIDES AN INTEGER (the tag walk, the
 * accept/split test of Alg. 2, the Euler-spiral parameters, every subdivision count, every
 * subdivision parameter t_i) is evaluated in fp32 with no FMA contraction (compile with
 * -ffp-contract=off), because the paper fixes fp32 (L21).  Vertex COORDINATES are then evaluated in
 * double from those fp32 parameters (Euler-spiral integral by 16-point Gauss-Legendre) and rounded
 * to fp32 once: this is the definition the fp32 kernels must reproduce within 1e-3 px.
 *
 * Parity pins live in tests/test_oracle_*.py (arc-mode counts of section 5 and evolute counts of section 6:
 * tests/test_oracle_pins.py, measured against the exact spiral).  "parity unpinned": the
 * three-term cubic->ES error estimate of section 7.1 against the paper's "mean ratio 1.656" claim (only pinned
 * through the tolerance invariant), and the constants EPS_Q, DELTA_T, DT_MIN, the |theta|>120deg
 * guard (exercised through invariants on degenerate inputs only).
 */
#define _GNU_SOURCE
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------ boundary mirrors */
typedef struct {
    float width;
    float miter_limit;
    uint8_t join; /* 0 miter 1 round 2 bevel */
    uint8_t cap;  /* 0 butt 1 square 2 round */
    uint16_t fill; /* bit 0: the path is FILLED, not stroked (Alg. 1); width, join, cap are then ignored;
                      bit 1: the stroke is DASHED with the call's dash pattern (so_expand_dashed) */
    uint32_t rsv;
} so_style;

enum { JOIN_MITER = 0, JOIN_ROUND = 1, JOIN_BEVEL = 2 };
enum { CAP_BUTT = 0, CAP_SQUARE = 1, CAP_ROUND = 2 };
enum { MODE_LINE = 0, MODE_ARC = 1, MODE_LINE_REFINED = 2 };   /* 2: lines with the exact density integral (L145) */

/* record kinds (low 3 bits) | side bit (8 = +h side) */
enum { K_OFFSET = 0, K_OFFSET_REV = 1, K_EVOLUTE = 2, K_CONNECTOR = 3, K_JOIN_OUTER = 4, K_JOIN_INNER = 5, K_CAP = 6, K_CLOSE = 7, K_PLUS = 8 };

enum { ST_FIT_ITERS = 0, ST_PIECES, ST_RANGES_REG, ST_RANGES_SUP, ST_REC_OFFSET, ST_REC_EVOLUTE, ST_REC_CONNECTOR,
       ST_REC_JOIN, ST_REC_CAP, ST_LINE_SEGS, ST_CURVE_SEGS, ST_N };

typedef struct {
    uint64_t n_rec;
    float* xy;       /* [n_rec][4] x0 y0 x1 y1 */
    float* angle;    /* [n_rec] signed turning start->end (0 in line mode) */
    uint8_t* kind;   /* [n_rec] */
    uint32_t* seg;   /* [n_rec] source segment index */
    uint32_t* seg_count; /* [n_tags] records per input segment */
    uint64_t* path_off;  /* [n_paths+1] first record of each path */
    uint32_t* pt_off;    /* [n_tags] tag walk: first point of segment */
    uint32_t* path_idx;  /* [n_tags] */
    uint32_t* sp_first;  /* [n_tags] first segment of the subpath */
    uint64_t stats[16];
    uint64_t cap;
} so_result;

/* ------------------------------------------------------------------ constants (R-13) */
#define EPS_Q2 1e-12f               /* (1e-6 px)^2: "near zero" derivative, L251 */
#define DELTA_T 1e-4f               /* parameter perturbation, relative to dt, L251 */
#define DT_MIN (1.0f / 65536.0f)    /* deepest subdivision of Alg. 2 (paper silent) */
#define N_MAX 65535.0f              /* clamp for any single subdivision count */
#define C1 1.0976991822760038f      /* L155 */
#define C2 0.9148117935952064f
#define C3 0.16145779359520596f
#define PI_F 3.14159265358979323846f
#define QUARTER_PI 0.78539816339744830962f
#define SQRT8_3 0.94280904158206336587f /* sqrt(8)/3, L149 */

/* ------------------------------------------------------------------ small vector helpers */
typedef struct { float x, y; } v2f;
typedef struct { double x, y; } v2d;
static v2f v2(float x, float y) { v2f r = {x, y}; return r; }
static v2f sub(v2f a, v2f b) { return v2(a.x - b.x, a.y - b.y); }
static float dotf(v2f a, v2f b) { return a.x * b.x + a.y * b.y; }
static float crossf(v2f a, v2f b) { return a.x * b.y - a.y * b.x; }
static float len2(v2f a) { return a.x * a.x + a.y * a.y; }
static v2f unit(v2f a) { float l = sqrtf(len2(a)); return v2(a.x / l, a.y / l); }
/* Angles (R-17): the fp32 value nearest to the angle of the vector (x, y), i.e. atan2 evaluated in
 * double and rounded once.  This makes th0, th1 (hence k0, k1, L and everything derived from them) independent of
 * any particular libm's single-precision atan2f rounding. */
static float atan2_r(float y, float x) { return (float)atan2((double)y, (double)x); }

/* ------------------------------------------------------------------ Gauss-Legendre nodes (double) */
#define GLN 16
static double gl_x[GLN], gl_w[GLN];
static int gl_ready = 0;
static void gl_init(void) {
    if (gl_ready) return;
    for (int i = 0; i < GLN; i++) {
        double x = cos(M_PI * (i + 0.75) / (GLN + 0.5)), dp = 1;
        for (int it = 0; it < 100; it++) {
            double p0 = 1, p1 = x;
            for (int k = 2; k <= GLN; k++) { double pk = ((2 * k - 1) * x * p1 - (k - 1) * p0) / k; p0 = p1; p1 = pk; }
            dp = GLN * (x * p1 - p0) / (x * x - 1);
            double dx = p1 / dp;
            x -= dx;
            if (fabs(dx) < 1e-16) break;
        }
        { double p0 = 1, p1 = x; for (int k = 2; k <= GLN; k++) { double pk = ((2 * k - 1) * x * p1 - (k - 1) * p0) / k; p0 = p1; p1 = pk; }
          dp = GLN * (x * p1 - p0) / (x * x - 1); }
        gl_x[i] = x;
        gl_w[i] = 2 / ((1 - x * x) * dp * dp);
    }
    gl_ready = 1;
}

/* ================================================================== step 0: tag walk
 * L464-466 + Table 1 (L468-481) + L483: every tag carries stream-offset increments; offsets are
 * prefix sums.  Bits 0-1 coordinate count, bit 2 subpath end, bit 3 must be 0 (fp32 only), bit 4 path
 * end (implies subpath end), bit 7 closed subpath (R-8).  Point stream: segment i reads points
 * pt_off .. pt_off+count; the stream advances by count, +1 at a subpath end (L470).
 * Returns 0, or -2 (bad stream). */
int so_tag_walk(const uint8_t* tags, uint64_t n_tags, uint64_t n_points, uint64_t n_paths,
                uint32_t* pt_off, uint32_t* path_idx, uint32_t* sp_first) {
    uint64_t pt = 0, path = 0, first = 0;
    for (uint64_t i = 0; i < n_tags; i++) {
        uint8_t tag = tags[i];
        uint32_t cnt = tag & 3u;
        if (cnt == 0 || (tag & 8u)) return -2;
        uint32_t end = ((tag >> 2) | (tag >> 4)) & 1u;
        pt_off[i] = (uint32_t)pt;
        path_idx[i] = (uint32_t)path;
        sp_first[i] = (uint32_t)first;
        pt += cnt + end;
        if (end) first = i + 1;
        if (tag & 16u) path++;
    }
    if (n_tags > 0 && !(tags[n_tags - 1] & 16u)) return -2;
    if (pt != n_points || path != n_paths) return -2;
    return 0;
}

/* ================================================================== section 4.1 / 4.2: subdivision density integral */
/* Exact integral f(x) = int_0^x sqrt|u^2-1| du (L135) in closed form (L139, with the pi/4 placement
 * of reading R-3), double precision; exported for the pins only. */
double so_f_exact(double x) {
    double a = fabs(x), r;
    if (a <= 1) r = 0.5 * (a * sqrt(1 - a * a) + asin(a));
    else r = M_PI / 4 + 0.5 * (a * sqrt(a * a - 1) - acosh(a));
    return x < 0 ? -r : r;
}

/* f_approx (L149), odd extension (L157); middle piece sign-preserving (R-3b). fp32. */
float so_f_approx(float x) {
    float a = fabsf(x), r;
    if (a < 0.8f) r = sinf(C1 * a) / C1;
    else if (a < 1.25f) { float v = a - 1.0f; float w = fabsf(v) * sqrtf(fabsf(v)); r = SQRT8_3 * (v < 0 ? -w : w) + QUARTER_PI; }
    else if (a < 2.1f) r = 0.6406f * a * a - 0.81f * a + C2;
    else r = 0.5f * a * a - 0.156f * a + C3;
    return x < 0 ? -r : r;
}

/* inverse of f_approx, piece by piece (each piece of L149 solved for x); knots are f_approx at
 * 0.8 / 1.25 / 2.1. fp32. */
float so_f_approx_inv(float u) {
    float a = fabsf(u), r;
    if (a < 0.70107076f) r = asinf(C1 * a) / C1;
    else if (a < 0.90324929f) { float v = (a - QUARTER_PI) / SQRT8_3; float w = cbrtf(fabsf(v)); w = w * w; r = 1.0f + (v < 0 ? -w : w); }
    else if (a < 2.03885779f) r = (0.81f + sqrtf(0.6561f - 2.5624f * (C2 - a))) / 1.2812f;
    else r = 0.156f + sqrtf(0.024336f - 2.0f * (C3 - a));
    return u < 0 ? -r : r;
}

/* The "higher flattening quality" variant of L145 (reading R-22): the exact integral of L139 in the forward
 * direction, and for the inverse "this approximation [as] a good initial value ...; two iterations of Newton solving are
 * enough to refine this guess to within 32-bit floating point accuracy".
 * Both in DOUBLE, rounded to fp32 once (as the angles of R-17): u = f(x) -> x is ill-conditioned next to the zeros of the
 * density (f'(x) = sqrt|x^2 - 1| at |x| = 1: the inflection and the cusp), so an fp32 evaluation would make the subdivision
 * points depend on the last bit of one libm's asinf.
 * Newton from x0 = f_approx_inv(u) on f(a) = |u| for a = |x|; where the guess lies in the middle piece of L149
 * (0.8 <= a < 1.25) the iteration runs on w(a) = sgn(e) |e|^(2/3), e = f(a) - pi/4, which is smooth and nearly linear
 * across a = 1 (f - pi/4 ~ sqrt(8)/3 (a - 1)^1.5, L149), with w'(a) = 2/3 f'(a) / |e|^(1/3) -> 2/3 sqrt(a + 1) / (sqrt(8)/3)^(1/3). */
static double f_and_deriv(double a, double* deriv) {
    *deriv = sqrt(fabs((1.0 - a) * (1.0 + a)));
    return so_f_exact(a);
}
static double signed_pow23(double v) { double c = cbrt(fabs(v)); c = c * c; return v < 0 ? -c : c; }
double so_f_inv_newton(float u, int steps) {
    double au = fabs((double)u);
    double a = fabs((double)so_f_approx_inv(u));
    int middle = (a >= 0.8 && a < 1.25);
    double wt = signed_pow23(au - M_PI / 4);
    for (int it = 0; it < steps; it++) {
        double d, fa = f_and_deriv(a, &d);
        if (middle) {
            double e = fa - M_PI / 4, ce = cbrt(fabs(e));
            double ratio = fabs(a - 1.0) < 1e-9 ? sqrt(a + 1.0) / cbrt(sqrt(8.0) / 3.0) : d / ce;
            a = a - (signed_pow23(e) - wt) / ((2.0 / 3.0) * ratio);
        } else {
            a = a - (fa - au) / d;
        }
    }
    return u < 0 ? -a : a;
}
float so_f_inv_refined(float u) { return (float)so_f_inv_newton(u, 2); }

/* ================================================================== Appendix A: geometric Hermite interpolation
 * k = th0+th1, D = th1-th0 (L634).  k1 (L636) and chord/arc ratio c (L641-651), coefficients verbatim,
 * terms in the paper's order.  The unit-arc-length spiral is kappa(s) = k0 + k1 s for s in [-1/2,1/2]
 * (reading R-1). fp32. */
void so_ghi(float th0, float th1, float* k1_out, float* c_out) {
    float k = th0 + th1, D = th1 - th0;
    float k2 = k * k, k4 = k2 * k2, k6 = k4 * k2;
    float D2 = D * D, D3 = D2 * D, D4 = D2 * D2, D5 = D4 * D, D6 = D4 * D2, D7 = D6 * D;
    float k1 = 6.0f * D;
    k1 -= D3 / 70.0f;
    k1 -= D5 / 10780.0f;
    k1 += D7 * 2.769178184818219e-7f;
    k1 -= k2 * D / 10.0f;
    k1 += k2 * D3 / 4200.0f;
    k1 += k2 * D5 * 1.6959677820260655e-5f;
    k1 -= k4 * D / 1400.0f;
    k1 += k4 * D3 * 6.84915970574303e-5f;
    k1 -= k6 * D * 7.936475029053326e-6f;
    float c = 1.0f;
    c -= D2 / 40.0f;
    c += D4 * 0.00034226190482569864f;
    c -= D6 * 1.9349474568904524e-6f;
    c -= k2 / 24.0f;
    c += k2 * D2 * 0.0024702380951963226f;
    c -= k2 * D4 * 3.7297408997537985e-5f;
    c += k4 / 1920.0f;
    c -= k4 * D2 * 4.87350869747975e-5f;
    c -= k6 * 3.1001936068463107e-6f;
    *k1_out = k1;
    *c_out = c;
}

/* Unit-arc Euler spiral integral Z(t) = int_0^t exp(i((k0-k1/2)u + k1 u^2/2)) du, start tangent along
 * +x (R-2): 16-point Gauss-Legendre in double. */
void so_es_integral(double k0, double k1, double t, double* zx, double* zy) {
    gl_init();
    double a = k0 - 0.5 * k1, sx = 0, sy = 0;
    for (int j = 0; j < GLN; j++) {
        double u = 0.5 * t * (gl_x[j] + 1.0);
        double ph = a * u + 0.5 * k1 * u * u;
        sx += gl_w[j] * cos(ph);
        sy += gl_w[j] * sin(ph);
    }
    *zx = 0.5 * t * sx;
    *zy = 0.5 * t * sy;
}

/* ================================================================== section 7.1: cubic -> ES error estimate
 * Inputs: unit tangents u0,u1 at the ends of the sub-cubic, raw derivative magnitudes |q0|,|q1|
 * (q = C'/3), chord vector, dt.  Output th0, th1, chord length and the estimated error in px. fp32.
 * L215 unit-chord normalisation; L217 d-bar; L221 e1; L225 area; L227 e2; L229 e3; guards R-4. */
float so_fit_error(v2f u0, v2f u1, float q0mag, float q1mag, v2f ch, float dt, float* th0_out, float* th1_out, float* chord_out) {
    float chord2 = len2(ch);
    float chord = sqrtf(chord2);
    *chord_out = chord;
    if (chord2 < EPS_Q2) { *th0_out = 0; *th1_out = 0; return INFINITY; }
    v2f uc = v2(ch.x / chord, ch.y / chord);
    float s0 = crossf(u0, uc), c0 = dotf(u0, uc); /* sin, cos of th0 = angle from start tangent to chord */
    float s1 = crossf(uc, u1), c1 = dotf(uc, u1); /* th1 = angle from chord to end tangent */
    float th0 = atan2_r(s0, c0), th1 = atan2_r(s1, c1); /* R-17 */
    *th0_out = th0;
    *th1_out = th1;
    if (c0 < -0.5f || c1 < -0.5f) return 2.0f * chord; /* outside the validated box: force a split (R-4) */
    float d0 = q0mag * dt / chord, d1 = q1mag * dt / chord; /* control-arm lengths of the sub-cubic */
    float db0 = 2.0f / (3.0f * (1.0f + c0)), db1 = 2.0f / (3.0f * (1.0f + c1)); /* L217 */
    float s01 = s0 * c1 + c0 * s1; /* sin(th0+th1) */
    float area = 0.15f * (2.0f * d0 * s0 + 2.0f * d1 * s1 - d0 * d1 * s01);     /* L225, source cubic */
    float areb = 0.15f * (2.0f * db0 * s0 + 2.0f * db1 * s1 - db0 * db1 * s01); /* ES-fit cubic */
    float ksum = fabsf(th0 + th1), kdif = fabsf(th0 - th1);
    float k2 = ksum * ksum;
    float e1 = 4.6255e-6f * k2 * k2 * ksum + 7.5e-3f * k2 * kdif; /* L221 */
    float e2 = 1.55f * fabsf(area - areb);                         /* L227 */
    float dd0 = db0 - d0, dd1 = db1 - d1;
    float e3 = (0.005f * ksum + 0.07f * kdif) * sqrtf(dd0 * dd0 + dd1 * dd1); /* L229 */
    return chord * (e1 + e2 + e3);                                 /* L215 */
}

/* ================================================================== per-call state */
typedef struct {
    so_result* out;
    int mode;
    float tol_es, tol_fl;
    uint32_t cur_seg;
    int fill;        /* the current path is filled: offset 0, one side (Alg. 1) */
    /* dashing (reading R-23; see dash_piece) */
    int nd;                  /* entries of the dash pattern (0: none) */
    uint64_t dq[8], period, phase_q;   /* the pattern, its sum and the phase in units of 2^-16 px */
    int dashed;              /* the current path is dashed */
    uint64_t pos;            /* arc length from the start of the current subpath to the start of the next piece, same units */
    uint64_t sp_total;       /* arc length of the current subpath */
    int measuring;           /* first pass over a subpath: pieces only add their length to pos */
    const void* style;       /* the current path's style (caps of the dashes) */
} ctx_t;

static int push_rec(ctx_t* c, v2d a, v2d b, double angle, int kind) {
    so_result* o = c->out;
    if (o->n_rec == o->cap) {
        uint64_t nc = o->cap ? o->cap * 2 : 4096;
        float* nxy = (float*)realloc(o->xy, nc * 4 * sizeof(float));
        float* nan_ = (float*)realloc(o->angle, nc * sizeof(float));
        uint8_t* nk = (uint8_t*)realloc(o->kind, nc);
        uint32_t* ns = (uint32_t*)realloc(o->seg, nc * sizeof(uint32_t));
        if (!nxy || !nan_ || !nk || !ns) return -1;
        o->xy = nxy; o->angle = nan_; o->kind = nk; o->seg = ns; o->cap = nc;
    }
    uint64_t i = o->n_rec++;
    o->xy[4 * i + 0] = (float)a.x; o->xy[4 * i + 1] = (float)a.y;
    o->xy[4 * i + 2] = (float)b.x; o->xy[4 * i + 3] = (float)b.y;
    o->angle[i] = (float)angle;
    o->kind[i] = (uint8_t)kind;
    o->seg[i] = c->cur_seg;
    return 0;
}

/* a side's records in forward-t order, before mirroring */
typedef struct { v2d a, b; double angle; int kind; } rec_t;
typedef struct { rec_t* r; size_t n, cap; } reclist;
static void rl_push(reclist* l, v2d a, v2d b, double angle, int kind) {
    if (l->n == l->cap) { l->cap = l->cap ? 2 * l->cap : 256; l->r = (rec_t*)realloc(l->r, l->cap * sizeof(rec_t)); }
    rec_t x = {a, b, angle, kind};
    l->r[l->n++] = x;
}

/* canonical offset point: global vertex V (double), unit tangent u (fp32 bits), signed offset eta:
 * V + eta*N, N = (-u.y, u.x) the left normal (R-conv). */
static v2d offset_point(v2d V, v2f u, float eta) {
    v2d r = {V.x + (double)eta * (-(double)u.y), V.y + (double)eta * (double)u.x};
    return r;
}

/* ================================================================== one accepted Euler-spiral piece */
typedef struct {
    v2d pa, pb;      /* global end points of the piece (double; exact images of fp32 values) */
    v2f ua, ub;      /* unit tangents of the cubic at the ends (fp32) */
    v2f ch;          /* chord vector, fp32, local */
    float th0, th1, chord;
    float k0, k1, L; /* ES parameters: total turning, GHI k1, arc length = chord / c */
    double z1x, z1y; /* Z(1) */
} piece_t;

static float es_kappa(const piece_t* p, float t) { return (p->k0 + p->k1 * (t - 0.5f)) / p->L; } /* R-1 */

/* point on the ES at piece fraction t (double): pa + ch (x) Z(t)/Z(1); exact at both ends (L632). */
static v2d es_point(const piece_t* p, float t) {
    if (t == 0.0f) return p->pa;
    if (t == 1.0f) return p->pb;
    double zx, zy;
    so_es_integral(p->k0, p->k1, t, &zx, &zy);
    double den = p->z1x * p->z1x + p->z1y * p->z1y;
    double wx = (zx * p->z1x + zy * p->z1y) / den, wy = (zy * p->z1x - zx * p->z1y) / den;
    v2d r = {p->pa.x + (double)p->ch.x * wx - (double)p->ch.y * wy, p->pa.y + (double)p->ch.x * wy + (double)p->ch.y * wx};
    return r;
}
/* tangent angle advance from the piece start: phi(t) = (k0-k1/2) t + k1 t^2/2 */
static double es_phi(const piece_t* p, float t) { return ((double)p->k0 - 0.5 * (double)p->k1) * t + 0.5 * (double)p->k1 * (double)t * (double)t; }
/* unit tangent (double): the cubic's own at the ends, rotation of ua by phi(t) inside */
static v2d es_tangent(const piece_t* p, float t) {
    v2d r;
    if (t == 0.0f) { r.x = p->ua.x; r.y = p->ua.y; return r; }
    if (t == 1.0f) { r.x = p->ub.x; r.y = p->ub.y; return r; }
    double ph = es_phi(p, t), c = cos(ph), s = sin(ph);
    r.x = c * p->ua.x - s * p->ua.y;
    r.y = s * p->ua.x + c * p->ua.y;
    return r;
}
static v2d es_offset(const piece_t* p, float t, float eta) {
    v2d P = es_point(p, t), T = es_tangent(p, t);
    v2d r = {P.x - (double)eta * T.y, P.y + (double)eta * T.x};
    return r;
}
/* evolute point P + N/kappa (section 6) */
static v2d es_evolute(const piece_t* p, float t) {
    v2d P = es_point(p, t), T = es_tangent(p, t);
    double rho = 1.0 / (double)es_kappa(p, t);
    v2d r = {P.x - rho * T.y, P.y + rho * T.x};
    return r;
}

/* v -> sgn(v) |v|^1.5 and its inverse: the integral of sqrt|v| and the s ~ i^(2/3) rule of section 2.2 (L97) */
static float pow15(float v) { float a = fabsf(v), w = a * sqrtf(a); return v < 0 ? -w : w; }
static float pow15_inv(float w) { float c = cbrtf(fabsf(w)); c = c * c; return w < 0 ? -c : c; }
enum { RULE_UNIFORM = 0, RULE_F_APPROX = 1, RULE_INFLECTION = 2, RULE_CUSP = 3, RULE_F_EXACT = 4 };
static float clampf(float x, float lo, float hi) { return x < lo ? lo : (x > hi ? hi : x); }
static float count_clamp(float n) { if (!(n >= 1.0f)) return 1.0f; return n > N_MAX ? N_MAX : n; }

/* --- regular or reversed offset range [ta,tb] of side eta: subdivision parameters (section 4, 5).
 * Fills ts[0..n] (ts[0]=ta, ts[n]=tb); returns n. */
static int offset_params(const ctx_t* c, const piece_t* p, float eta, float ta, float tb, float** ts_out) {
    float n_f;
    float ua = 0, ub = 0;
    int rule = RULE_UNIFORM;
    float ah = fabsf(eta);
    if (c->mode == MODE_ARC) {
        /* L177: n = s cbrt(|k'|(1+0.4|h s k'|)/(120 d)), s=L, k'=k1/L^2; scaled by the range fraction (R-12) */
        float n_full = cbrtf(p->L * fabsf(p->k1) * (1.0f + 0.4f * fabsf(eta * p->k1) / p->L) / (120.0f * c->tol_fl));
        n_f = ceilf((tb - ta) * n_full);
    } else {
        float ka = es_kappa(p, ta), kb = es_kappa(p, tb);
        float xa = 2.0f * eta * ka - 1.0f, xb = 2.0f * eta * kb - 1.0f; /* L125: inflection -> -1, cusp -> +1 */
        float xm = 0.5f * (xa + xb);
        float kp = fabsf(p->k1) / (p->L * p->L);
        if (fabsf(xb - xa) < 0.015625f * fmaxf(1.0f, fabsf(xm))) {
            /* x varies too little over the range for the difference of two f_approx values in fp32 (R-7): the density
             * sqrt|k (1 - k eta)| (L77-83, L131) is integrated locally instead.  km, gm: curvature and cusp factor at the
             * middle of the range; m_infl, m_cusp: how far km is from the inflection (k = 0) and from the cusp (k = 1/eta). */
            float km = 0.5f * (ka + kb), dk = fabsf(kb - ka);
            float gm = 1.0f - km * eta;
            float m_infl = fabsf(km), m_cusp = fabsf(gm) / ah;
            if (dk <= 0.125f * fminf(m_infl, m_cusp)) {
                /* neither zero of the density is near: constant density (limit: the circular arc, L73) */
                n_f = ceilf((tb - ta) * p->L * sqrtf(fabsf(km * gm) / (8.0f * c->tol_fl)));
            } else if (m_infl <= m_cusp) {
                /* an inflection in or next to the range: int sqrt|k| ds = 2/3 |k|^1.5 / k' (section 2.2: the
                 * subdivision points follow s_i ~ i^(2/3) from the inflection), the factor sqrt|1 - k eta| at the middle */
                ua = pow15(ka); ub = pow15(kb);
                n_f = ceilf((2.0f / 3.0f) * fabsf(ub - ua) * sqrtf(fabsf(gm)) / (kp * sqrtf(8.0f * c->tol_fl)));
                rule = RULE_INFLECTION;
            } else {
                /* the range ends next to the cusp: the same with g = 1 - k eta (ds = dg / (eta k')), sqrt|k| at the middle */
                ua = pow15(1.0f - ka * eta); ub = pow15(1.0f - kb * eta);
                n_f = ceilf((2.0f / 3.0f) * fabsf(ub - ua) * sqrtf(fabsf(km)) / (ah * kp * sqrtf(8.0f * c->tol_fl)));
                rule = RULE_CUSP;
            }
        } else {
            int refined = (c->mode == MODE_LINE_REFINED);
            ua = refined ? (float)so_f_exact((double)xa) : so_f_approx(xa);
            ub = refined ? (float)so_f_exact((double)xb) : so_f_approx(xb);
            n_f = ceilf(fabsf(ub - ua) / (4.0f * kp * ah * sqrtf(ah) * sqrtf(8.0f * c->tol_fl))); /* L83 with density sqrt|1-x^2|/(2 sqrt|h|) */
            rule = refined ? RULE_F_EXACT : RULE_F_APPROX;
        }
    }
    int n = (int)count_clamp(n_f);
    float* ts = (float*)malloc((size_t)(n + 1) * sizeof(float));
    ts[0] = ta;
    ts[n] = tb;
    for (int i = 1; i < n; i++) {
        float fr = (float)i / (float)n;
        float t;
        if (rule == RULE_UNIFORM) t = ta + fr * (tb - ta);
        else {
            float u = ua + fr * (ub - ua), kap;
            if (rule == RULE_F_APPROX) kap = (so_f_approx_inv(u) + 1.0f) / (2.0f * eta);
            else if (rule == RULE_F_EXACT) kap = (so_f_inv_refined(u) + 1.0f) / (2.0f * eta);
            else if (rule == RULE_INFLECTION) kap = pow15_inv(u);
            else kap = (1.0f - pow15_inv(u)) / eta;
            t = 0.5f + (kap * p->L - p->k0) / p->k1;
        }
        ts[i] = clampf(t, ta, tb);
    }
    *ts_out = ts;
    return n;
}

/* --- evolute range [ta,tb]: density |sigma|^-1/2, integral 2 sqrt(sigma), inverse squaring (L195). */
static int evolute_params(const ctx_t* c, const piece_t* p, float ta, float tb, float** ts_out) {
    float ka = es_kappa(p, ta), kb = es_kappa(p, tb), km = 0.5f * (ka + kb);
    float kp = fabsf(p->k1) / (p->L * p->L);
    float n_f, wa = 0, wb = 0;
    int uniform = 1;
    int arc = (c->mode == MODE_ARC);
    if (arc) {
        /* Arc mode: the evolute is approximated by arcs with the metric of section 5 (L171: arcs follow the
         * derivative of curvature with respect to arc length).  With sigma the spiral's arc length from the inflection
         * (kappa = kappa' sigma) the evolute has arc length element |kappa'| / kappa^2 dsigma and curvature kappa^3 / |kappa'|,
         * so d kappa_E / d s_E = 3 kappa^4 / |kappa'| and
         *   n = int cbrt(3 kappa^4 / (|kappa'| 120 d)) |kappa'| / kappa^2 dsigma = 3^(4/3) |cbrt(sigma_b) - cbrt(sigma_a)| / cbrt(120 d):
         * the subdivision points are uniform in cbrt(sigma), the inverse is cubing.  Reading R-20: the constant 120 of L171
         * belongs to a curve of CONSTANT curvature derivative; the evolute's varies along an arc and the measured deviation
         * with 120 reaches 1.41 d (tests/test_oracle_pins.py): 80 is used here, which keeps it below d. */
        if (fabsf(kb - ka) < 0.015625f * fabsf(km)) {
            /* nearly constant curvature: constant density cbrt(3 kappa'^2 / (120 d kappa^2)) per unit of the spiral's arc length */
            n_f = ceilf((tb - ta) * p->L * cbrtf(3.0f * kp * kp / (80.0f * c->tol_fl * km * km)));
        } else {
            wa = cbrtf(fabsf(ka) / kp);
            wb = cbrtf(fabsf(kb) / kp);
            n_f = ceilf(4.326748710922225f * fabsf(wb - wa) / cbrtf(80.0f * c->tol_fl)); /* 3^(4/3) */
            uniform = 0;
        }
        /* The metric assumes arcs of small turning.  The evolute turns with the spiral (its tangent is the spiral's
         * normal): a short evolute of a strongly turning piece would be ONE arc of several radians.  At least one arc per
         * pi/4 of turning over the range, then uniform in t (no arc turns by more than ~pi/2; reading R-20). */
        {
            float dphi = fabsf((tb - ta) * (0.5f * p->k1 * (ta + tb) + (p->k0 - 0.5f * p->k1)));
            float n_phi = ceilf(dphi / QUARTER_PI);
            if (n_phi > n_f) { n_f = n_phi; uniform = 1; }
        }
    } else if (fabsf(kb - ka) < 0.015625f * fabsf(km)) {
        n_f = ceilf((tb - ta) * p->L * sqrtf(fabsf(kp / km) / (8.0f * c->tol_fl)));
    } else {
        wa = sqrtf(fabsf(ka) / kp);
        wb = sqrtf(fabsf(kb) / kp);
        n_f = ceilf(fabsf(2.0f * wb - 2.0f * wa) * sqrtf(1.0f / (8.0f * c->tol_fl)));
        uniform = 0;
    }
    int n = (int)count_clamp(n_f);
    float* ts = (float*)malloc((size_t)(n + 1) * sizeof(float));
    ts[0] = ta;
    ts[n] = tb;
    for (int i = 1; i < n; i++) {
        float fr = (float)i / (float)n, t;
        if (uniform) t = ta + fr * (tb - ta);
        else {
            float w = wa + fr * (wb - wa);
            float kap = (ka < 0 ? -kp : kp) * w * w * (arc ? w : 1.0f); /* sigma = w^2 (lines, L195) or w^3 (arcs) */
            t = 0.5f + (kap * p->L - p->k0) / p->k1;
        }
        ts[i] = clampf(t, ta, tb);
    }
    *ts_out = ts;
    return n;
}

/* forward-t records of one side of one piece (Alg. 2, readings R-9): cusp split, regular
 * ranges, super-critical ranges with evolute patch. */
static void side_records(ctx_t* c, const piece_t* p, float eta, reclist* out) {
    float g0 = 1.0f - es_kappa(p, 0.0f) * eta, g1 = 1.0f - es_kappa(p, 1.0f) * eta; /* cusp0, cusp1 (L382-384) up to a positive factor */
    /* L386.  The cusp is inside the piece iff g0 and g1 have strictly opposite signs (decided from the signs, not
     * from the product: g0 == 0 with g1 < 0 is a piece that is super-critical over its whole length). */
    int has_cusp = (g0 > 0.0f && g1 < 0.0f) || (g0 < 0.0f && g1 > 0.0f);
    float tc = has_cusp ? g0 / (g0 - g1) : 1.0f;
    int first_sup = g0 < 0.0f || (g0 == 0.0f && g1 < 0.0f);
    float ranges[2][2];
    int sup[2], nr = 0;
    if (!first_sup) { ranges[nr][0] = 0.0f; ranges[nr][1] = tc; sup[nr] = 0; nr++; }      /* L388-392: regular on [0,t] */
    if (first_sup || tc < 1.0f) {                                                          /* L397-403: evolute patch */
        if (!first_sup) { ranges[nr][0] = tc; ranges[nr][1] = 1.0f; } else { ranges[nr][0] = 0.0f; ranges[nr][1] = tc; }
        sup[nr] = 1; nr++;
    }
    if (first_sup && tc < 1.0f) { ranges[nr][0] = tc; ranges[nr][1] = 1.0f; sup[nr] = 0; nr++; } /* L407-411: regular on [t,1] */
    for (int r = 0; r < nr; r++) {
        float ta = ranges[r][0], tb = ranges[r][1];
        float* ts;
        int n = offset_params(c, p, eta, ta, tb, &ts);
        if (!sup[r]) {
            c->out->stats[ST_RANGES_REG]++;
            for (int i = 0; i < n; i++)
                rl_push(out, es_offset(p, ts[i], eta), es_offset(p, ts[i + 1], eta), es_phi(p, ts[i + 1]) - es_phi(p, ts[i]), K_OFFSET);
        } else {
            c->out->stats[ST_RANGES_SUP]++;
            /* the evolute meets the offset curve at the cusp: E(t*) := O(t*) bitwise */
            int cusp_a = (ta != 0.0f), cusp_b = (tb != 1.0f);
            v2d Oa = es_offset(p, ta, eta), Ob = es_offset(p, tb, eta);
            v2d Ea = cusp_a ? Oa : es_evolute(p, ta), Eb = cusp_b ? Ob : es_evolute(p, tb);
            if (!cusp_a) { rl_push(out, Oa, Ea, 0, K_CONNECTOR); rl_push(out, Oa, Ea, 0, K_CONNECTOR); } /* "output twice", L197 */
            float* te;
            int ne = evolute_params(c, p, ta, tb, &te);
            for (int copy = 0; copy < 2; copy++)
                for (int i = 0; i < ne; i++) {
                    v2d a = (i == 0) ? Ea : es_evolute(p, te[i]);
                    v2d b = (i == ne - 1) ? Eb : es_evolute(p, te[i + 1]);
                    /* the evolute's tangent is the spiral's normal: it turns by the same angle (used in arc mode only) */
                    rl_push(out, a, b, es_phi(p, te[i + 1]) - es_phi(p, te[i]), K_EVOLUTE);
                }
            free(te);
            for (int i = n; i > 0; i--) /* reversed offset (L403, L191) */
                rl_push(out, es_offset(p, ts[i], eta), es_offset(p, ts[i - 1], eta), es_phi(p, ts[i - 1]) - es_phi(p, ts[i]), K_OFFSET_REV);
            if (!cusp_b) { rl_push(out, Eb, Ob, 0, K_CONNECTOR); rl_push(out, Eb, Ob, 0, K_CONNECTOR); }
        }
        free(ts);
    }
}

/* both sides of a piece whose k0, k1, L are set */
static int piece_records(ctx_t* c, piece_t* p, float h) {
    so_es_integral(p->k0, p->k1, 1.0, &p->z1x, &p->z1y);
    c->out->stats[ST_PIECES]++;
    reclist l = {0, 0, 0};
    /* -h side, forward */
    side_records(c, p, -h, &l);
    for (size_t i = 0; i < l.n; i++)
        if (push_rec(c, l.r[i].a, l.r[i].b, c->mode == MODE_ARC ? l.r[i].angle : 0.0, l.r[i].kind)) return -1;
    /* a fill is "flatten_cubic(segment, 0)" (Alg. 1): the curve itself, once.  With eta = 0 there is no cusp
     * (1 - kappa eta = 1) and offset_params integrates the pure Euler-spiral density sqrt|kappa| (section 2.2;
     * arcs: L171). */
    if (c->fill) { free(l.r); return 0; }
    /* +h side: mirror image of its forward-t list (reverse order, swap end points, negate angle) */
    l.n = 0;
    side_records(c, p, h, &l);
    for (size_t i = l.n; i > 0; i--)
        if (push_rec(c, l.r[i - 1].b, l.r[i - 1].a, c->mode == MODE_ARC ? -l.r[i - 1].angle : 0.0, l.r[i - 1].kind | K_PLUS)) return -1;
    free(l.r);
    return 0;
}

/* ================================================================== dashing
 * "the core algorithm is prefix sum applied to segment length, and the Euler spiral representation is particularly well
 * suited" (L543); "Given its parameterization by arc length ..." (L589).  The paper stops there; reading R-23 of DESIGN.md:
 *
 *   - The pattern is nd in {2, 4, 6, 8} positive lengths (on, off, on, off, ...) and a phase >= 0, in output px, the same for
 *     every dashed path of the call; it restarts at every subpath.  Lengths are integers in units of 2^-16 px
 *     (llrintf(x * 65536), at least 1 per pattern entry): sums are then exact and do not depend on the order of addition,
 *     which is what lets a parallel prefix sum reproduce this sequential walk bit for bit.
 *   - The arc length of a curve is that of its Euler-spiral pieces (L = chord / c, App. A), piece by piece in the order of
 *     Alg. 2; of a line (or a degenerate curve, R-1b) the distance of its end points.
 *   - Pattern entry j covers [a, b) of the subpath's arc length; the on-entries (j even) are the dashes.  The part of a dash
 *     inside a piece [S, S + L) is the sub-range ta = (a - S) / L .. tb = (b - S) / L of the piece (integers converted to fp32,
 *     one division), clipped to [0, 1]: an Euler-spiral piece again, with k0' = (tb - ta)(k0 + k1 ((ta + tb)/2 - 1/2)),
 *     k1' = k1 (tb - ta)^2, L' = L (tb - ta), from the spiral's point and tangent at ta to those at tb.  It goes through the
 *     SAME flattening as an undashed piece (both sides, cusps, evolutes).
 *   - A dash begins where its entry begins (a in [S, S + L): start cap before the sub-range's records) or at arc length 0; it
 *     ends where its entry ends (b in (S, S + L]: end cap after them) or at the subpath's total arc length.  Everything is
 *     decided from arc-length positions alone (a piece without length emits nothing).  Caps are the path's cap style.  A
 *     closed subpath is dashed like an open one (no closing join, no merging of its last dash with its first).
 *   - The join after a segment is emitted iff a dash covers the junction strictly inside (a < S_next < b, 0 < S_next < total).
 *   - Record order within a segment: per piece in increasing t, per dash in increasing arc length:
 *     [start cap][-h side][+h side][end cap]; then the join. */
static int emit_cap(ctx_t* c, const so_style* st, v2f Vf, v2f T, float h, v2d from, v2d to);
static v2d round32(v2d a) { v2d r = {(double)(float)a.x, (double)(float)a.y}; return r; }

static int dash_sub_piece(ctx_t* c, piece_t* p, float h, float ta, float tb, int starts, int ends, int line) {
    const so_style* st = (const so_style*)c->style;
    piece_t q = *p;
    if (line) {
        /* a straight piece: points pa + t ch, constant tangent */
        if (ta != 0.0f) { q.pa.x = (double)(float)(p->pa.x + (double)ta * (double)p->ch.x); q.pa.y = (double)(float)(p->pa.y + (double)ta * (double)p->ch.y); }
        if (tb != 1.0f) { q.pb.x = (double)(float)(p->pa.x + (double)tb * (double)p->ch.x); q.pb.y = (double)(float)(p->pa.y + (double)tb * (double)p->ch.y); }
    } else if (ta != 0.0f || tb != 1.0f) {
        float dt = tb - ta, tm = 0.5f * (ta + tb) - 0.5f;
        q.k0 = dt * (p->k0 + p->k1 * tm);
        q.k1 = p->k1 * dt * dt;
        q.L = p->L * dt;
        if (!(q.L > 1e-12f)) q.L = 1e-12f;
        /* a cut end: the spiral's point, rounded to fp32 (an uncut end keeps the piece's own end point and tangent) */
        if (ta != 0.0f) { v2d TA = es_tangent(p, ta); q.pa = round32(es_point(p, ta)); q.ua = v2((float)TA.x, (float)TA.y); }
        if (tb != 1.0f) { v2d TB = es_tangent(p, tb); q.pb = round32(es_point(p, tb)); q.ub = v2((float)TB.x, (float)TB.y); }
        q.ch = v2((float)(q.pb.x - q.pa.x), (float)(q.pb.y - q.pa.y));
    }
    v2f Va = v2((float)q.pa.x, (float)q.pa.y), Vb = v2((float)q.pb.x, (float)q.pb.y);
    if (starts && emit_cap(c, st, Va, v2(-q.ua.x, -q.ua.y), h, offset_point(q.pa, q.ua, h), offset_point(q.pa, q.ua, -h))) return -1;
    if (line) {
        if (push_rec(c, offset_point(q.pa, q.ua, -h), offset_point(q.pb, q.ub, -h), 0, K_OFFSET)) return -1;
        if (push_rec(c, offset_point(q.pb, q.ub, h), offset_point(q.pa, q.ua, h), 0, K_OFFSET | K_PLUS)) return -1;
    } else if (piece_records(c, &q, h)) return -1;
    if (ends && emit_cap(c, st, Vb, q.ub, h, offset_point(q.pb, q.ub, -h), offset_point(q.pb, q.ub, h))) return -1;
    return 0;
}

/* one piece (an accepted Euler spiral with k0, k1, L set, or a straight segment: line != 0, L = its length) under the dash
 * pattern; advances c->pos */
static int dash_piece(ctx_t* c, piece_t* p, float h, int line) {
    uint64_t Lq = (uint64_t)llrintf(p->L * 65536.0f);
    uint64_t S = c->pos, E = S + Lq;
    c->pos = E;
    if (c->measuring || Lq == 0) return 0;   /* (a piece without length carries no part of a dash) */
    if (!line) so_es_integral(p->k0, p->k1, 1.0, &p->z1x, &p->z1y);   /* Z(1): es_point of the piece itself */
    uint64_t u = (S + c->phase_q) % c->period;   /* where in the pattern the piece starts */
    int j = 0;
    while (u >= c->dq[j]) { u -= c->dq[j]; j++; }
    uint64_t s = S;
    while (s < E) {
        uint64_t e = s + (c->dq[j] - u);         /* end of entry j */
        if ((j & 1) == 0) {
            uint64_t b = e < E ? e : E;
            int starts = (u == 0) || (s == 0);
            int ends = (e <= E) || (E == c->sp_total);
            float ta = s == S ? 0.0f : (float)(s - S) / (float)Lq;
            float tb = b == E ? 1.0f : (float)(b - S) / (float)Lq;
            if (dash_sub_piece(c, p, h, ta, tb, starts, ends, line)) return -1;
        }
        s = e; u = 0; j = (j + 1) % c->nd;
    }
    return 0;
}
/* does a dash cover arc position s strictly inside (a < s < b)? */
static int dash_covers(const ctx_t* c, uint64_t s) {
    if (s == 0 || s >= c->sp_total) return 0;
    uint64_t u = (s + c->phase_q) % c->period;
    int j = 0;
    while (u >= c->dq[j]) { u -= c->dq[j]; j++; }
    return (j & 1) == 0 && u > 0;
}

static int emit_piece(ctx_t* c, piece_t* p, float h) {
    float cc;
    so_ghi(p->th0, p->th1, &p->k1, &cc);
    p->k0 = p->th0 + p->th1;
    if (!(cc > 0.05f)) cc = 0.05f; /* far outside the polynomial's range (|theta| near pi): keep L finite */
    p->L = p->chord / cc;
    if (!(p->L > 1e-12f)) p->L = 1e-12f; /* zero-length piece accepted at DT_MIN */
    if (c->dashed) return dash_piece(c, p, h, 0);
    return piece_records(c, p, h);
}

/* ================================================================== segments */
typedef struct {
    int kind;      /* 1 line 2 quad 3 cubic */
    v2f P0, P3;    /* global (device-space) end points, fp32 */
    v2f c1, c2, c3;/* cubic control points relative to P0 (after degree elevation, L349) */
    v2f ts, te;    /* unit start / end tangents */
    int degenerate;
} seg_t;

/* transform (R-14): x' = fma(a,x,fma(c,y,e)), y' = fma(b,x,fma(d,y,f)) */
static v2f xform(const float* A, const float* p) {
    return v2(fmaf(A[0], p[0], fmaf(A[2], p[1], A[4])), fmaf(A[1], p[0], fmaf(A[3], p[1], A[5])));
}

/* first control-polygon leg that is not (near) zero, else (1,0) (R-5): the limit tangent of the curve */
static v2f pick_tangent(v2f a, v2f b, v2f c, int* degenerate) {
    *degenerate = 0;
    if (len2(a) >= EPS_Q2) return unit(a);
    if (len2(b) >= EPS_Q2) return unit(b);
    if (len2(c) >= EPS_Q2) return unit(c);
    *degenerate = 1;
    return v2(1.0f, 0.0f);
}

static void load_segment(const uint8_t* tags, const float* pts, const float* A, const uint32_t* pt_off, uint64_t i, seg_t* s) {
    int cnt = tags[i] & 3;
    const float* p = pts + 2 * (uint64_t)pt_off[i];
    v2f q0 = xform(A, p), q1 = xform(A, p + 2), q2 = q1, q3 = q1;
    if (cnt >= 2) q2 = xform(A, p + 4);
    if (cnt >= 3) q3 = xform(A, p + 6);
    s->kind = cnt;
    s->P0 = q0;
    int dg;
    if (cnt == 1) {
        s->P3 = q1;
        v2f d = sub(q1, q0);
        s->c3 = d;
        s->c1 = v2(d.x / 3.0f, d.y / 3.0f);
        s->c2 = v2(d.x * (2.0f / 3.0f), d.y * (2.0f / 3.0f));
        s->ts = s->te = pick_tangent(d, d, d, &dg);
    } else if (cnt == 2) {
        s->P3 = q2;
        v2f a = sub(q1, q0), b = sub(q2, q0); /* control point and end point, local */
        s->c1 = v2(a.x * (2.0f / 3.0f), a.y * (2.0f / 3.0f));                                   /* p0 + 2/3 (q - p0) */
        s->c2 = v2(b.x + (a.x - b.x) * (2.0f / 3.0f), b.y + (a.y - b.y) * (2.0f / 3.0f));       /* p2 + 2/3 (q - p2) */
        s->c3 = b;
        s->ts = pick_tangent(a, b, b, &dg);
        int dg2;
        s->te = pick_tangent(sub(b, a), b, b, &dg2);
    } else {
        s->P3 = q3;
        s->c1 = sub(q1, q0);
        s->c2 = sub(q2, q0);
        s->c3 = sub(q3, q0);
        s->ts = pick_tangent(s->c1, s->c2, s->c3, &dg);
        int dg2;
        s->te = pick_tangent(sub(s->c3, s->c2), sub(s->c3, s->c1), s->c3, &dg2);
    }
    s->degenerate = dg;
}

/* cubic position (local) and q = C'/3 at t, Bernstein form; fp32, no contraction */
static v2f cubic_pos(const seg_t* s, float t) {
    float mt = 1.0f - t;
    float a = 3.0f * mt * mt * t, b = 3.0f * mt * t * t, c = t * t * t;
    return v2(a * s->c1.x + b * s->c2.x + c * s->c3.x, a * s->c1.y + b * s->c2.y + c * s->c3.y);
}
static v2f cubic_q(const seg_t* s, float t) {
    float mt = 1.0f - t;
    float a = mt * mt, b = 2.0f * mt * t, c = t * t;
    v2f d0 = s->c1, d1 = sub(s->c2, s->c1), d2 = sub(s->c3, s->c2);
    return v2(a * d0.x + b * d1.x + c * d2.x, a * d0.y + b * d1.y + c * d2.y);
}
/* eval_cubic_and_deriv of Alg. 2 L369 with the near-zero-derivative rule of L251 (R-5): returns the
 * position, |q| and a unit tangent.  At t=1 the segment's end tangent is used. */
static void eval_cubic(const seg_t* s, float t, float dt, v2f* pos, float* qmag, v2f* u) {
    v2f q = cubic_q(s, t);
    float q2 = len2(q);
    *qmag = sqrtf(q2);
    if (t == 1.0f) { *pos = s->c3; *u = s->te; return; }
    *pos = cubic_pos(s, t);
    if (q2 >= EPS_Q2) { *u = v2(q.x / *qmag, q.y / *qmag); return; }
    v2f qp = cubic_q(s, t - DELTA_T * dt);
    float qp2 = len2(qp);
    if (qp2 > 0.0f) *u = unit(qp); else *u = v2(1.0f, 0.0f);
}

/* Alg. 2 (L351-438, L444): iterative bisection with the two-word stack (t0_u, dt). One pass serves
 * both sides (the fit does not depend on the offset). */
static int flatten_cubic(ctx_t* c, const seg_t* s, float h) {
    uint32_t t0_u = 0;
    float dt = 1.0f;
    v2f last_p = v2(0, 0), last_u = s->ts;
    float last_qmag = sqrtf(len2(s->c1));
    for (;;) {
        float t0 = (float)t0_u * dt;
        if (t0 == 1.0f) break;
        float t1 = t0 + dt;
        v2f next_p, next_u;
        float next_qmag;
        eval_cubic(s, t1, dt, &next_p, &next_qmag, &next_u);
        float th0, th1, chord;
        v2f ch = sub(next_p, last_p);
        float err = so_fit_error(last_u, next_u, last_qmag, next_qmag, ch, dt, &th0, &th1, &chord);
        if (!c->measuring) c->out->stats[ST_FIT_ITERS]++;
        if (err <= c->tol_es || dt <= DT_MIN) {
            piece_t p;
            p.pa.x = (double)s->P0.x + (double)last_p.x; p.pa.y = (double)s->P0.y + (double)last_p.y;
            if (t1 == 1.0f) { p.pb.x = s->P3.x; p.pb.y = s->P3.y; } /* canonical end vertex, shared with the join */
            else { p.pb.x = (double)s->P0.x + (double)next_p.x; p.pb.y = (double)s->P0.y + (double)next_p.y; }
            p.ua = last_u; p.ub = next_u; p.ch = ch; p.th0 = th0; p.th1 = th1; p.chord = chord;
            if (emit_piece(c, &p, h)) return -1;
            t0_u += 1;
            int shift = __builtin_ctz(t0_u);
            t0_u >>= shift;
            dt *= (float)(1u << shift);
            last_p = next_p; last_u = next_u; last_qmag = next_qmag;
        } else {
            t0_u *= 2;
            dt *= 0.5f;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------ circular arcs for round joins / caps
 * centre V, from A (= V + r0) sweeping CCW by phi to B.  Line mode: exact arc metric L65-69,
 * n = ceil(phi / (2 acos(1 - d/|h|))); arc mode: 1 record if phi <= pi/2 else 2 (R-10). */
static int emit_round(ctx_t* c, v2d V, v2d A, v2d B, float phi, float h, int kind) {
    int n;
    if (c->mode == MODE_ARC) n = (phi <= 0.5f * PI_F) ? 1 : 2;
    else {
        float n_f = 1.0f;
        if (c->tol_fl < h) n_f = ceilf(phi / (2.0f * acosf(1.0f - c->tol_fl / h)));
        n = (int)count_clamp(n_f);
    }
    v2d prev = A;
    double rx = A.x - V.x, ry = A.y - V.y;
    for (int i = 1; i <= n; i++) {
        v2d cur = B;
        if (i < n) {
            double a = (double)phi * (double)i / (double)n, ca = cos(a), sa = sin(a);
            cur.x = V.x + ca * rx - sa * ry;
            cur.y = V.y + sa * rx + ca * ry;
        }
        if (push_rec(c, prev, cur, c->mode == MODE_ARC ? (double)phi / n : 0.0, kind)) return -1;
        prev = cur;
    }
    return 0;
}

/* join at the vertex between segment i (end tangent T0, end point V) and its partner (start tangent T1,
 * start point W) -- R-10.  -h side runs forward A->B, +h side backward B'->A'. */
static int emit_join(ctx_t* c, const so_style* st, v2f Vf, v2f T0, v2f Wf, v2f T1, float h) {
    v2d V = {Vf.x, Vf.y}, W = {Wf.x, Wf.y};
    float cr = crossf(T0, T1), dt = dotf(T0, T1);
    int outer_minus = (cr > 0.0f) || (cr == 0.0f && dt < 0.0f);
    v2d A = offset_point(V, T0, -h), B = offset_point(W, T1, -h);
    v2d Bp = offset_point(W, T1, h), Ap = offset_point(V, T0, h);
    float phi = fabsf(atan2_r(cr, dt));
    float opd = 1.0f + dt;
    int miter_ok = (opd > 1e-6f) && (2.0f / opd <= st->miter_limit * st->miter_limit); /* 1/sin(beta/2) <= limit */
    for (int side = 0; side < 2; side++) {
        v2d s0 = side == 0 ? A : Bp, s1 = side == 0 ? B : Ap;
        int sb = side == 0 ? 0 : K_PLUS;
        int outer = side == 0 ? outer_minus : !outer_minus;
        c->out->stats[ST_REC_JOIN]++;
        if (!outer) { /* inner join: through the vertex (strong correctness, L35) */
            if (push_rec(c, s0, V, 0, K_JOIN_INNER | sb) || push_rec(c, V, s1, 0, K_JOIN_INNER | sb)) return -1;
        } else if (st->join == JOIN_ROUND) {
            if (emit_round(c, V, s0, s1, phi, h, K_JOIN_OUTER | sb)) return -1;
        } else if (st->join == JOIN_MITER && miter_ok) {
            double sg = side == 0 ? -1.0 : 1.0; /* tip = V -/+ h (N0+N1)/(1+dt) */
            double nx = -(double)T0.y - (double)T1.y, ny = (double)T0.x + (double)T1.x;
            v2d tip = {V.x + sg * (double)h * nx / (double)opd, V.y + sg * (double)h * ny / (double)opd};
            if (push_rec(c, s0, tip, 0, K_JOIN_OUTER | sb) || push_rec(c, tip, s1, 0, K_JOIN_OUTER | sb)) return -1;
        } else {
            if (push_rec(c, s0, s1, 0, K_JOIN_OUTER | sb)) return -1;
        }
    }
    return 0;
}

/* cap at vertex V, outward direction T (the end tangent for an end cap, minus the start tangent for a
 * start cap); from V - hN(T) CCW to V + hN(T) (R-11). */
static int emit_cap(ctx_t* c, const so_style* st, v2f Vf, v2f T, float h, v2d from, v2d to) {
    v2d V = {Vf.x, Vf.y};
    c->out->stats[ST_REC_CAP]++;
    if (st->cap == CAP_ROUND) return emit_round(c, V, from, to, PI_F, h, K_CAP);
    if (st->cap == CAP_SQUARE) {
        v2d c1 = {from.x + (double)h * T.x, from.y + (double)h * T.y}, c2 = {to.x + (double)h * T.x, to.y + (double)h * T.y};
        if (push_rec(c, from, c1, 0, K_CAP) || push_rec(c, c1, c2, 0, K_CAP) || push_rec(c, c2, to, 0, K_CAP)) return -1;
        return 0;
    }
    return push_rec(c, from, to, 0, K_CAP);
}

/* ================================================================== the whole call */
void so_free(so_result* r) {
    free(r->xy); free(r->angle); free(r->kind); free(r->seg); free(r->seg_count); free(r->path_off);
    free(r->pt_off); free(r->path_idx); free(r->sp_first);
    memset(r, 0, sizeof(*r));
}

/* stroke_expand on the CPU.  All pointers host.  Returns 0 / -1 invalid arg or out of memory / -2 bad
 * stream.  Record order within segment i ("canonical order"): for every ES piece in
 * increasing t: [-h side, forward] [+h side, mirrored]; then the join [-h side][+h side], or, on the
 * last segment of an open subpath, [end cap][start cap] (the thread at the subpath end draws the start
 * cap, as the paper's marker thread does, L345). */
static int line_piece(ctx_t* c, const seg_t* s, float h) {   /* a straight segment as a piece of the dash walk */
    piece_t p;
    memset(&p, 0, sizeof(p));
    p.pa.x = s->P0.x; p.pa.y = s->P0.y; p.pb.x = s->P3.x; p.pb.y = s->P3.y;
    p.ua = s->ts; p.ub = s->te;
    p.ch = sub(s->P3, s->P0);
    p.chord = sqrtf(len2(p.ch));
    p.L = p.chord;
    return dash_piece(c, &p, h, 1);
}

static int expand_impl(const uint8_t* tags, uint64_t n_tags, const float* pts, uint64_t n_points, const so_style* styles,
                       uint64_t n_paths, const float* affine, float tolerance, int mode, const float* dash, int n_dash, float phase, so_result* out) {
    memset(out, 0, sizeof(*out));
    if (n_dash != 0 && (n_dash < 2 || n_dash > 8 || (n_dash & 1) || !dash || !(phase >= 0.0f) || !isfinite(phase))) return -1;
    for (int k = 0; k < n_dash; k++) if (!(dash[k] > 0.0f) || !isfinite(dash[k])) return -1;
    if (!(tolerance > 0) || (mode != MODE_LINE && mode != MODE_ARC && mode != MODE_LINE_REFINED)) return -1;
    float det = affine[0] * affine[3] - affine[1] * affine[2];
    if (!isfinite(det) || det == 0.0f) return -1;
    out->seg_count = (uint32_t*)calloc(n_tags + 1, sizeof(uint32_t));
    out->path_off = (uint64_t*)calloc(n_paths + 1, sizeof(uint64_t));
    out->pt_off = (uint32_t*)calloc(n_tags + 1, sizeof(uint32_t));
    out->path_idx = (uint32_t*)calloc(n_tags + 1, sizeof(uint32_t));
    out->sp_first = (uint32_t*)calloc(n_tags + 1, sizeof(uint32_t));
    int rc = so_tag_walk(tags, n_tags, n_points, n_paths, out->pt_off, out->path_idx, out->sp_first);
    if (rc) { so_free(out); return rc; }
    ctx_t c;
    memset(&c, 0, sizeof(c));
    c.out = out;
    c.mode = mode;
    c.tol_es = 0.1f * tolerance; /* R-13 */
    c.tol_fl = (mode == MODE_LINE_REFINED ? 0.9f : 0.8f) * tolerance;   /* R-22: the 6 % of f_approx (L145) no longer needs the margin */
    float scale = sqrtf(fabsf(det)); /* R-14 */
    c.nd = n_dash; c.period = 0; c.dashed = 0; c.measuring = 0; c.pos = 0; c.sp_total = 0;
    for (int k = 0; k < n_dash; k++) {
        c.dq[k] = (uint64_t)llrintf(dash[k] * 65536.0f);
        if (c.dq[k] == 0) c.dq[k] = 1;
        c.period += c.dq[k];
    }
    c.phase_q = n_dash ? (uint64_t)llrintf(phase * 65536.0f) : 0;
    uint64_t next_path = 0;
    for (uint64_t i = 0; i < n_tags; i++) {
        uint64_t before = out->n_rec;
        c.cur_seg = (uint32_t)i;
        uint32_t path = out->path_idx[i];
        while (next_path <= path) out->path_off[next_path++] = before;
        const so_style* st = &styles[path];
        float h = 0.5f * st->width * scale;
        c.fill = st->fill & 1;
        c.dashed = 0;   /* (set below for a dashed stroke: a filled path is never dashed) */
        if (c.fill) {
            /* Alg. 1: a filled path is flattened with offset 0; an open subpath is closed by a line from its last
             * point to its first (always emitted, possibly of zero length: counts stay a function of the tags) */
            seg_t s;
            load_segment(tags, pts, affine, out->pt_off, i, &s);
            v2d V0 = {s.P0.x, s.P0.y}, V3 = {s.P3.x, s.P3.y};
            if (s.kind == 1 || s.degenerate) {
                out->stats[ST_LINE_SEGS]++;
                if (push_rec(&c, V0, V3, 0, K_OFFSET)) goto oom;
            } else {
                out->stats[ST_CURVE_SEGS]++;
                if (flatten_cubic(&c, &s, 0.0f)) goto oom;
            }
            uint8_t tag = tags[i];
            if ((((tag >> 2) | (tag >> 4)) & 1) && !((tag >> 7) & 1)) {
                seg_t f;
                load_segment(tags, pts, affine, out->pt_off, out->sp_first[i], &f);
                v2d F0 = {f.P0.x, f.P0.y};
                if (push_rec(&c, V3, F0, 0, K_CLOSE)) goto oom;
            }
        } else if (h > 0.0f && isfinite(h)) { /* width <= 0 or non-finite: the path emits nothing */
            seg_t s;
            load_segment(tags, pts, affine, out->pt_off, i, &s);
            c.dashed = c.nd > 0 && (st->fill & 2);
            c.style = st;
            if (c.dashed && out->sp_first[i] == i) {
                /* the subpath's arc length: the same walk, measuring only (on the GPU: the prefix sum of L543) */
                c.measuring = 1; c.pos = 0;
                for (uint64_t j = i;; j++) {
                    seg_t m;
                    load_segment(tags, pts, affine, out->pt_off, j, &m);
                    if (m.kind == 1 || m.degenerate) { if (line_piece(&c, &m, h)) goto oom; }
                    else if (flatten_cubic(&c, &m, h)) goto oom;
                    if (((tags[j] >> 2) | (tags[j] >> 4)) & 1) break;
                }
                c.sp_total = c.pos; c.measuring = 0; c.pos = 0;
            }
            if (c.dashed) {
                if (s.kind == 1 || s.degenerate) { out->stats[ST_LINE_SEGS]++; if (line_piece(&c, &s, h)) goto oom; }
                else { out->stats[ST_CURVE_SEGS]++; if (flatten_cubic(&c, &s, h)) goto oom; }
                uint8_t tg = tags[i];
                if (!(((tg >> 2) | (tg >> 4)) & 1) && dash_covers(&c, c.pos)) {
                    seg_t n;
                    load_segment(tags, pts, affine, out->pt_off, i + 1, &n);
                    if (emit_join(&c, st, s.P3, s.te, n.P0, n.ts, h)) goto oom;
                }
                out->seg_count[i] = (uint32_t)(out->n_rec - before);
                continue;
            }
            if (s.kind == 1 || s.degenerate) {
                /* straight fast path (R-1b): the two offset lines are exact */
                v2d V0 = {s.P0.x, s.P0.y}, V3 = {s.P3.x, s.P3.y};
                out->stats[ST_LINE_SEGS]++;
                if (push_rec(&c, offset_point(V0, s.ts, -h), offset_point(V3, s.te, -h), 0, K_OFFSET)) goto oom;
                if (push_rec(&c, offset_point(V3, s.te, h), offset_point(V0, s.ts, h), 0, K_OFFSET | K_PLUS)) goto oom;
            } else {
                out->stats[ST_CURVE_SEGS]++;
                if (flatten_cubic(&c, &s, h)) goto oom;
            }
            uint8_t tag = tags[i];
            int sp_end = ((tag >> 2) | (tag >> 4)) & 1;
            int closed = (tag >> 7) & 1;
            if (!sp_end || closed) {
                uint64_t j = sp_end ? out->sp_first[i] : i + 1;
                seg_t n;
                load_segment(tags, pts, affine, out->pt_off, j, &n);
                if (emit_join(&c, st, s.P3, s.te, n.P0, n.ts, h)) goto oom;
            } else {
                seg_t f;
                load_segment(tags, pts, affine, out->pt_off, out->sp_first[i], &f);
                v2d V3 = {s.P3.x, s.P3.y}, V0 = {f.P0.x, f.P0.y};
                if (emit_cap(&c, st, s.P3, s.te, h, offset_point(V3, s.te, -h), offset_point(V3, s.te, h))) goto oom;
                if (emit_cap(&c, st, f.P0, v2(-f.ts.x, -f.ts.y), h, offset_point(V0, f.ts, h), offset_point(V0, f.ts, -h))) goto oom;
            }
        }
        out->seg_count[i] = (uint32_t)(out->n_rec - before);
    }
    while (next_path <= n_paths) out->path_off[next_path++] = out->n_rec;
    for (uint64_t r = 0; r < out->n_rec; r++) {
        int k = out->kind[r] & 7;
        if (k == K_OFFSET || k == K_OFFSET_REV) out->stats[ST_REC_OFFSET]++;
        else if (k == K_EVOLUTE) out->stats[ST_REC_EVOLUTE]++;
        else if (k == K_CONNECTOR) out->stats[ST_REC_CONNECTOR]++;
    }
    return 0;
oom:
    so_free(out);
    return -1;
}

int so_expand(const uint8_t* tags, uint64_t n_tags, const float* pts, uint64_t n_points, const so_style* styles,
              uint64_t n_paths, const float* affine, float tolerance, int mode, so_result* out) {
    return expand_impl(tags, n_tags, pts, n_points, styles, n_paths, affine, tolerance, mode, NULL, 0, 0.0f, out);
}
/* the same with a dash pattern (n_dash in {2, 4, 6, 8} positive lengths, phase >= 0, output px) for the paths whose style
 * has bit 1 of `fill` set: dash_piece above */
int so_expand_dashed(const uint8_t* tags, uint64_t n_tags, const float* pts, uint64_t n_points, const so_style* styles,
                     uint64_t n_paths, const float* affine, float tolerance, int mode, const float* dash, int n_dash, float phase, so_result* out) {
    return expand_impl(tags, n_tags, pts, n_points, styles, n_paths, affine, tolerance, mode, dash, n_dash, phase, out);
}

/* ------------------------------------------------------------------ thin exports used by the pins */
void so_fit_error_export(const float* u0, const float* u1, float q0mag, float q1mag, const float* ch, float dt, float* out4) {
    float th0, th1, chord;
    float e = so_fit_error(v2(u0[0], u0[1]), v2(u1[0], u1[1]), q0mag, q1mag, v2(ch[0], ch[1]), dt, &th0, &th1, &chord);
    out4[0] = th0; out4[1] = th1; out4[2] = chord; out4[3] = e;
}

/* One Euler-spiral piece given directly by its parameters (for the pins of sections 5 and 6, which measure the
 * emitted arcs / evolute chords against the exact spiral): unit-arc curvature kappa(s) = k0 + k1 s on [-1/2,1/2]
 * (R-1), arc length L px, starting at (x0, y0) with tangent angle dir0; both sides at half-width h, flatten
 * tolerance tol_fl (the TOL_FL of R-13, given directly), in canonical order.  Same code path as a piece accepted by
 * Alg. 2 from here on (piece_records). */
int so_piece_expand(float k0, float k1, float L, float x0, float y0, float dir0, float h, float tol_fl, int mode, so_result* out) {
    memset(out, 0, sizeof(*out));
    out->seg_count = (uint32_t*)calloc(2, sizeof(uint32_t));
    out->path_off = (uint64_t*)calloc(2, sizeof(uint64_t));
    out->pt_off = (uint32_t*)calloc(2, sizeof(uint32_t));
    out->path_idx = (uint32_t*)calloc(2, sizeof(uint32_t));
    out->sp_first = (uint32_t*)calloc(2, sizeof(uint32_t));
    ctx_t c;
    memset(&c, 0, sizeof(c));
    c.out = out; c.mode = mode; c.tol_es = 0; c.tol_fl = tol_fl; c.cur_seg = 0; c.fill = (h == 0.0f);   /* h = 0: the piece of a filled path */
    piece_t p;
    memset(&p, 0, sizeof(p));
    p.k0 = k0; p.k1 = k1; p.L = L;
    double zx, zy;
    so_es_integral(k0, k1, 1.0, &zx, &zy);
    double cd = cos((double)dir0), sd = sin((double)dir0);
    p.ua = v2((float)cd, (float)sd);
    p.ub = v2((float)cos((double)dir0 + (double)k0), (float)sin((double)dir0 + (double)k0)); /* phi(1) = k0 */
    p.ch = v2((float)((double)L * (cd * zx - sd * zy)), (float)((double)L * (sd * zx + cd * zy)));
    p.pa.x = x0; p.pa.y = y0;
    p.pb.x = (double)x0 + (double)p.ch.x; p.pb.y = (double)y0 + (double)p.ch.y;
    p.chord = sqrtf(len2(p.ch));
    if (piece_records(&c, &p, h)) { so_free(out); return -1; }
    out->seg_count[0] = (uint32_t)out->n_rec;
    out->path_off[1] = out->n_rec;
    return 0;
}
