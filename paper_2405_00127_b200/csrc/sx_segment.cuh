// sx_segment.cuh -- one input segment end to end (Alg. 1 L306-343 per thread, Alg. 2 L351-438 inside).
//
// The pieces the kernels are made of: joins and caps (emit_join / emit_cap: the count pass with EMIT = false, the segment
// writer with EMIT = true), fit_next (Alg. 2 as a resumable generator) and process_segment, the thread-per-segment
// reference walk of everything a segment emits, in canonical order: the walk writer (k_write_walk) and the walk count of
// sx_count.cuh -- what a tile that does not fit the count pass's tables falls back to -- and the definition the
// node-parallel count pass and the table-driven writers reproduce bit for bit (tests/test_gpu_parity.py).  Counting and
// writing instantiate the same plan functions, so the counts agree by construction.
#pragma once
#include "sx_piece.cuh"

namespace sx {

// ---------------------------------------------------------------- record sink
// a 32-byte arc record in ONE 256-bit store (sm_100: STG.256; a full 32-byte sector instead of two half sectors) when the
// caller's buffer is 32-byte aligned, else as two 16-byte stores
SX_DEV void store_arc(float4* out, uint64_t rec, bool wide, float4 a, float4 b) {
    if (wide) {
        asm volatile("st.global.v8.f32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(out + 2 * rec), "f"(a.x), "f"(a.y), "f"(a.z), "f"(a.w),
                     "f"(b.x), "f"(b.y), "f"(b.z), "f"(b.w)
                     : "memory");
    } else {
        out[2 * rec] = a;
        out[2 * rec + 1] = b;
    }
}

struct Writer {
    float4* out;     // sx_line[] (1 float4 per record) or sx_arc[] (2 float4 per record)
    uint64_t base;   // index of the segment's first record
    uint32_t seg;
    int mode;
    bool wide;       // arc records by 256-bit stores (the buffer is 32-byte aligned)
    SX_DEV void put(uint32_t idx, V2 a, V2 b, float angle, uint32_t kind) const {
        uint64_t r = base + idx;
        if (mode != kModeArc) {
            out[r] = make_float4(a.x, a.y, b.x, b.y);
        } else {
            store_arc(out, r, wide, make_float4(a.x, a.y, b.x, b.y), make_float4(angle, u2f(seg), u2f(kind), 0.0f));
        }
    }
};

// one side's record in forward-t order; the +h side is the mirror image of its forward list (reverse
// order, end points swapped, angle negated)
struct SideSink {
    const Writer* w;
    uint32_t first;  // index (within the segment) of the side's first record
    uint32_t total;
    bool mirror;
    SX_DEV void put(uint32_t idx, V2 a, V2 b, float angle, uint32_t kind) const {
        if (mirror) w->put(first + (total - 1u - idx), b, a, 0.0f - angle, kind | kPlus);  // never a negative zero
        else w->put(first + idx, a, b, angle + 0.0f, kind);
    }
};

// ---------------------------------------------------------------- one side of one piece
template <bool EMIT>
SX_DEV uint32_t piece_side(const Piece& p, const Spiral& z, float eta, bool mirror, const Params& P, const Writer* w, uint32_t first) {
    SidePlan s = side_plan(p, eta, P.mode, P.tol_fl);
    if (!EMIT) return (uint32_t)s.total;
    SideSink k;
    k.w = w; k.first = first; k.total = (uint32_t)s.total; k.mirror = mirror;
    const bool arc = P.mode == kModeArc;
    uint32_t idx = 0;
    for (int r = 0; r < s.nr; r++) {
        const OffPlan o = r == 0 ? s.off[0] : s.off[1];
        const bool sup = r == 0 ? s.sup[0] : s.sup[1];
        if (!sup) {
            V2 prev = es_offset(p, z, o.ta, eta);
            float tp = o.ta;
            for (int i = 1; i <= o.n; i++) {
                float t = i < o.n ? offset_t(p, o, eta, i) : o.tb;
                V2 cur = es_offset(p, z, t, eta);
                k.put(idx++, prev, cur, arc ? es_dphi(p, tp, t) : 0.0f, kOffset);
                prev = cur; tp = t;
            }
        } else {
            // evolute patch (section 6): the evolute meets the offset curve at the cusp
            V2 Oa = es_offset(p, z, o.ta, eta), Ob = es_offset(p, z, o.tb, eta);
            V2 Ea = s.cusp_a ? Oa : es_evolute(p, z, o.ta), Eb = s.cusp_b ? Ob : es_evolute(p, z, o.tb);
            if (!s.cusp_a) { k.put(idx, Oa, Ea, 0.0f, kConnector); k.put(idx + 1, Oa, Ea, 0.0f, kConnector); idx += 2; }  // "output twice", L197
            const int ne = s.evo.n;
            V2 pe = Ea;
            float te_prev = s.evo.ta;
            for (int i = 0; i < ne; i++) {
                const float te = (i == ne - 1) ? s.evo.tb : evolute_t(p, s.evo, i + 1);
                V2 b = (i == ne - 1) ? Eb : es_evolute(p, z, te);
                const float ang = arc ? es_dphi(p, te_prev, te) : 0.0f;   // the evolute's tangent is the spiral's normal
                k.put(idx + i, pe, b, ang, kEvolute);
                k.put(idx + ne + i, pe, b, ang, kEvolute);
                pe = b; te_prev = te;
            }
            idx += 2 * ne;
            V2 prev = Ob;  // reversed offset (L403, L191)
            float tp = o.tb;
            for (int i = o.n - 1; i >= 0; i--) {
                float t = i > 0 ? offset_t(p, o, eta, i) : o.ta;
                V2 cur = i > 0 ? es_offset(p, z, t, eta) : Oa;
                k.put(idx++, prev, cur, arc ? es_dphi(p, tp, t) : 0.0f, kOffsetRev);
                prev = cur; tp = t;
            }
            if (!s.cusp_b) { k.put(idx, Eb, Ob, 0.0f, kConnector); k.put(idx + 1, Eb, Ob, 0.0f, kConnector); idx += 2; }
        }
    }
    return (uint32_t)s.total;
}

// ---------------------------------------------------------------- round joins / caps (L65-69 exact arc metric; R-10)
__device__ __noinline__ int round_count(float phi, float h, int mode, float tol_fl) {
    if (mode == kModeArc) return (phi <= 0.5f * kPi) ? 1 : 2;
    float n_f = 1.0f;
    if (tol_fl < h) n_f = ceilf(phi / (2.0f * acosf(1.0f - tol_fl / h)));
    return count_clamp(n_f);
}
// centre V, from A = V + r sweeping CCW by phi to B, n records
SX_DEV void emit_round(const Writer* w, uint32_t first, int n, V2 V, V2 r, V2 A, V2 B, float phi, uint32_t kind, bool arc) {
    V2 prev = A;
    float ang = arc ? phi / (float)n : 0.0f;
    for (int i = 1; i <= n; i++) {
        V2 cur = B;
        if (i < n) {
            float a = phi * (float)i / (float)n, sa, ca;
            sx_sincos(a, &sa, &ca);
            cur.x = V.x + fmaf(ca, r.x, -sa * r.y);
            cur.y = V.y + fmaf(sa, r.x, ca * r.y);
        }
        w->put(first + (uint32_t)(i - 1), prev, cur, ang, kind);
        prev = cur;
    }
}

struct Style { float width, miter_limit; int join, cap; bool fill; };

// join between this segment (end point V, end tangent T0) and its partner (start point W, start
// tangent T1) -- R-10.  -h side runs forward A->B, +h side backward B'->A'.
template <bool EMIT>
SX_DEV uint32_t emit_join(const Params& P, const Style& st, V2 V, V2 T0, V2 W, V2 T1, float h, const Writer* w, uint32_t first) {
    // Written per ROLE (outer join, inner join), not per side: which side is the outer one depends on the turn, and
    // a warp whose lanes turn both ways would otherwise run the outer and the inner code twice each.
    const float cr = cross(T0, T1), dt = dot(T0, T1);
    const bool outer_minus = (cr > 0.0f) || (cr == 0.0f && dt < 0.0f);
    const float opd = 1.0f + dt;
    const bool miter = st.join == kJoinMiter && (opd > 1e-6f) && (2.0f / opd <= st.miter_limit * st.miter_limit);
    const bool round = st.join == kJoinRound;
    const bool arc = P.mode == kModeArc;
    float phi = 0.0f;
    uint32_t n_outer = miter ? 2u : 1u;
    if (round) { phi = fabsf(atan2_r(cr, dt)); n_outer = (uint32_t)round_count(phi, h, P.mode, P.tol_fl); }
    if (EMIT) {
        // side 0 (-h, forward V -> W) comes first, then side 1 (+h, backward W -> V)
        const uint32_t first_outer = first + (outer_minus ? 0u : 2u), first_inner = first + (outer_minus ? n_outer : 0u);
        {   // outer side
            const bool plus = !outer_minus;
            const float hh = plus ? h : -h;
            const uint32_t kind = kJoinOuter | (plus ? (uint32_t)kPlus : 0u);
            const V2 s0 = offset_point(plus ? W : V, plus ? T1 : T0, hh), s1 = offset_point(plus ? V : W, plus ? T0 : T1, hh);
            if (round) {
                const V2 r = plus ? v2(fmaf(h, -T1.y, W.x - V.x), fmaf(h, T1.x, W.y - V.y)) : v2(h * T0.y, -h * T0.x);
                emit_round(w, first_outer, (int)n_outer, V, r, s0, s1, phi, kind, arc);
            } else if (miter) {
                const float k = hh / opd;  // tip = V -/+ h (N0+N1)/(1+dt)
                const V2 tip = v2(fmaf(k, -T0.y - T1.y, V.x), fmaf(k, T0.x + T1.x, V.y));
                w->put(first_outer, s0, tip, 0.0f, kind);
                w->put(first_outer + 1u, tip, s1, 0.0f, kind);
            } else {
                w->put(first_outer, s0, s1, 0.0f, kind);
            }
        }
        {   // inner side: through the vertex (strong correctness, L35)
            const bool plus = outer_minus;
            const float hh = plus ? h : -h;
            const uint32_t kind = kJoinInner | (plus ? (uint32_t)kPlus : 0u);
            const V2 s0 = offset_point(plus ? W : V, plus ? T1 : T0, hh), s1 = offset_point(plus ? V : W, plus ? T0 : T1, hh);
            w->put(first_inner, s0, V, 0.0f, kind);
            w->put(first_inner + 1u, V, s1, 0.0f, kind);
        }
    }
    return n_outer + 2u;
}

// cap at vertex V with outward direction T: from V - hN(T) counter-clockwise to V + hN(T) (R-11)
template <bool EMIT>
SX_DEV uint32_t emit_cap(const Params& P, const Style& st, V2 V, V2 T, float h, const Writer* w, uint32_t first) {
    if (st.cap == kCapRound) {
        int n = round_count(kPi, h, P.mode, P.tol_fl);
        if (EMIT) emit_round(w, first, n, V, v2(h * T.y, -h * T.x), offset_point(V, T, -h), offset_point(V, T, h), kPi, kCap, P.mode == kModeArc);
        return (uint32_t)n;
    }
    if (st.cap == kCapSquare) {
        if (EMIT) {
            V2 from = offset_point(V, T, -h), to = offset_point(V, T, h);
            V2 c1 = v2(fmaf(h, T.y + T.x, V.x), fmaf(h, T.y - T.x, V.y));
            V2 c2 = v2(fmaf(h, T.x - T.y, V.x), fmaf(h, T.x + T.y, V.y));
            w->put(first, from, c1, 0.0f, kCap);
            w->put(first + 1, c1, c2, 0.0f, kCap);
            w->put(first + 2, c2, to, 0.0f, kCap);
        }
        return 3;
    }
    if (EMIT) w->put(first, offset_point(V, T, -h), offset_point(V, T, h), 0.0f, kCap);
    return 1;
}

// ---------------------------------------------------------------- Alg. 2: cubic -> Euler spirals
// Iterative bisection with the two-word stack (t0_u, dt), pop by count-trailing-zeros (L444).  One pass
// serves both sides: the fit does not depend on the offset.  The loop is written as a resumable
// generator (fit_next returns one accepted piece per call): the walk count and the walk writer run the identical
// instruction sequence.
struct FitState {
    uint32_t t0_u;
    float dt;
    V2 last_p, last_u;
    float last_qmag;
};
SX_DEV FitState fit_begin(const Seg& s) {
    FitState f;
    f.t0_u = 0u; f.dt = 1.0f;
    f.last_p = v2(0.0f, 0.0f); f.last_u = s.ts;
    f.last_qmag = sqrtf(len2(s.c1));
    return f;
}
// advances Alg. 2 until the next accepted piece (true, piece in p) or the end of the segment (false)
SX_DEV bool fit_next(const Params& P, const Seg& s, FitState& f, Piece& p) {
    for (;;) {
        float t0 = (float)f.t0_u * f.dt;
        if (t0 == 1.0f) return false;
        float t1 = t0 + f.dt;
        V2 next_p, next_u;
        float next_qmag, th0, th1, chord;
        eval_cubic(s, t1, f.dt, &next_p, &next_qmag, &next_u);
        V2 ch = next_p - f.last_p;
        float err = node_error(f.last_u, next_u, f.last_qmag, next_qmag, ch, f.dt);
        if (err <= P.tol_es || f.dt <= kDtMin) {
            piece_angles(f.last_u, next_u, ch, &th0, &th1, &chord);
            p.base = s.P0; p.P3 = s.P3;
            p.la = f.last_p; p.lb = next_p;
            p.ua = f.last_u; p.ub = next_u;
            p.ch = ch;
            p.at0 = (t0 == 0.0f); p.at1 = (t1 == 1.0f);
            piece_params(p, th0, th1, chord);
            f.t0_u += 1u;
            int shift = ctz32(f.t0_u);
            f.t0_u >>= shift;
            f.dt *= (float)(1u << shift);
            f.last_p = next_p; f.last_u = next_u; f.last_qmag = next_qmag;
            return true;
        }
        f.t0_u *= 2u;
        f.dt *= 0.5f;
    }
}

// fill: "flatten_cubic(segment, 0)" (Alg. 1): h = 0 and the curve itself, once
template <bool EMIT>
SX_DEV uint32_t flatten_cubic(const Params& P, const Seg& s, float h, bool fill, const Writer* w) {
    uint32_t n = 0;
    FitState f = fit_begin(s);
    Piece p;
    Spiral z;
    while (fit_next(P, s, f, p)) {
        if (EMIT) es_prepare(p, z);
        n += piece_side<EMIT>(p, z, -h, false, P, w, n);             // -h side, forward
        if (!fill) n += piece_side<EMIT>(p, z, h, true, P, w, n);    // +h side, mirrored
    }
    return n;
}

// ---------------------------------------------------------------- Alg. 1: the whole segment
SX_DEV bool load_style(const Params& P, uint32_t path, Style* st, float* h) {
    uint4 raw = __ldg(reinterpret_cast<const uint4*>(P.styles) + path);
    st->width = u2f(raw.x);
    st->miter_limit = u2f(raw.y);
    st->join = (int)(raw.z & 0xffu);
    st->cap = (int)((raw.z >> 8) & 0xffu);
    st->fill = ((raw.z >> 16) & 1u) != 0u;   // Alg. 1: the path is filled: offset 0, one side
    *h = st->fill ? 0.0f : 0.5f * st->width * P.scale;
    return st->fill || (*h > 0.0f && *h < INFINITY);  // a stroke of width <= 0 or non-finite: the path emits nothing
}

// what follows the offset curves of segment i (Alg. 1): the join with its partner, or, on the last
// segment of an open subpath, [end cap][start cap]
// tag_n, pt_n: tag and point offset of segment i + 1, first: sp_first[i] -- loaded by the caller together with the
// segment's own scan results, so that the partner's points are one dependent load away, not two
// the tail with the partner's start point W and start tangent T1 given (the join partner, or the subpath's first segment
// for the caps and for the closing line of a fill)
template <bool EMIT>
SX_DEV uint32_t segment_tail_given(const Params& P, uint32_t tag, const Seg& s, const Style& st, float h, V2 W, V2 T1, const Writer* w, uint32_t first) {
    const bool sp_end = ((tag >> 2) | (tag >> 4)) & 1u;
    const bool closed = (tag >> 7) & 1u;
    if (st.fill) {   // no joins, no caps: the line that closes an open subpath (always emitted: counts follow the tags)
        if (!sp_end || closed) return 0u;
        if (EMIT) w->put(first, s.P3, W, 0.0f, kClose);
        return 1u;
    }
    if (!sp_end || closed) return emit_join<EMIT>(P, st, s.P3, s.te, W, T1, h, w, first);
    uint32_t n = emit_cap<EMIT>(P, st, s.P3, s.te, h, w, first);
    n += emit_cap<EMIT>(P, st, W, v2(-T1.x, -T1.y), h, w, first + n);
    return n;
}
template <bool EMIT>
SX_DEV uint32_t segment_tail(const Params& P, uint32_t tag, const Seg& s, const Style& st, float h, uint32_t first_seg, uint32_t tag_n,
                             uint32_t pt_n, const Writer* w, uint32_t first) {
    const bool sp_end = ((tag >> 2) | (tag >> 4)) & 1u;
    const bool closed = (tag >> 7) & 1u;
    V2 W = v2(0.0f, 0.0f), T1 = v2(1.0f, 0.0f);
    if (!sp_end) load_segment_start_at(P, pt_n, tag_n, &W, &T1);
    else if (!st.fill || !closed) load_segment_start(P, first_seg, &W, &T1);
    return segment_tail_given<EMIT>(P, tag, s, st, h, W, T1, w, first);
}
template <bool EMIT>
SX_DEV uint32_t segment_tail(const Params& P, uint32_t i, uint32_t tag, const Seg& s, const Style& st, float h, const Writer* w, uint32_t first) {
    const uint32_t jn = i + 1u < P.n_tags ? i + 1u : i;
    return segment_tail<EMIT>(P, tag, s, st, h, P.sp_first[i], P.tags[jn], P.pt_off[jn], w, first);
}

// straight fast path (R-1b): the two offset lines of a line (or fully degenerate) segment are exact
SX_DEV uint32_t emit_straight(const Seg& s, float h, bool fill, const Writer* w) {
    if (fill) { w->put(0, s.P0, s.P3, 0.0f, kOffset); return 1u; }   // the segment itself
    w->put(0, offset_point(s.P0, s.ts, -h), offset_point(s.P3, s.te, -h), 0.0f, kOffset);
    w->put(1, offset_point(s.P3, s.te, h), offset_point(s.P0, s.ts, h), 0.0f, kOffset | kPlus);
    return 2u;
}

// thread-per-segment reference path: everything segment i emits, in canonical order
template <bool EMIT>
SX_DEV uint32_t process_segment(const Params& P, uint32_t i, Writer* w, uint32_t* tail_out = nullptr) {
    uint32_t tag = P.tags[i];
    Style st;
    float h;
    if (tail_out) *tail_out = 0u;
    if (!load_style(P, P.path_idx[i], &st, &h)) return 0;
    Seg s = load_segment(P, i, tag);
    uint32_t n;
    if (s.kind == 1 || s.degenerate) {
        if (EMIT) emit_straight(s, h, st.fill, w);
        n = st.fill ? 1u : 2u;
    } else {
        n = flatten_cubic<EMIT>(P, s, h, st.fill, w);
    }
    const uint32_t tail = segment_tail<EMIT>(P, i, tag, s, st, h, w, n);
    if (tail_out) *tail_out = tail;
    return n + tail;
}

}  // namespace sx
