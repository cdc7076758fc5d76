// sx_dash.cuh -- dashing on the GPU ("the core algorithm is prefix sum applied to
// segment length, and the Euler spiral representation is particularly well suited"; L589: "Given its parameterization by arc
// length, we believe the Euler spiral representation lends itself well to an approach based on parallel prefix sums of segment
// arc lengths").  The paper dashes on the CPU; reading R-23 of DESIGN.md fixes the definition.
//
// Definition (R-23).  The call's pattern -- nd in {2, 4, 6, 8} positive lengths (on, off, ...) and a phase >= 0, output px --
// applies to every stroked path whose style has bit 1 of `fill` set and restarts at every subpath.  Lengths are INTEGERS in
// units of 2^-16 px (llrintf(x * 65536)): sums are exact and independent of the order of addition, so the parallel prefix
// sum below reproduces a sequential walk bit for bit.  The arc length of a curve is that of its Euler-spiral pieces (L = chord
// / c, App. A) in the order of Alg. 2, of a line the distance of its end points.  The part of a dash [a, b) inside a piece
// [S, S + L) is the sub-range ta = (a - S) / L .. tb = (b - S) / L of the piece: an Euler-spiral piece again (k0' = (tb - ta)
// (k0 + k1 ((ta + tb) / 2 - 1/2)), k1' = k1 (tb - ta)^2, L' = L (tb - ta)) that goes through the SAME flattening as an
// undashed piece (side plans, cusps, evolutes: piece_side of sx_segment.cuh).  A dash begins where its pattern entry begins or
// at arc length 0 (start cap) and ends where the entry ends or at the subpath's total length (end cap); the join after a
// segment is emitted iff a dash covers the junction strictly inside.  A closed subpath is dashed like an open one.  Record order
// within a segment: per piece in increasing t, per dash in increasing arc length [start cap][-h side][+h side][end cap]; then
// the join.
//
// Pipeline (all launched by the host side in place of the count pass / the writers when a pattern is set):
//   k_dash_len     thread per segment: the segment's arc length in units (Alg. 2 once, summing the pieces' lengths)
//   (prefix sum)   the allocation scan of sx_scan.cuh over the lengths: 64-bit positions
//   k_dash_totals  thread per segment: the last segment of a subpath stores the subpath's total length at its first segment
//   k_dash_count   thread per segment: Alg. 2 again, pieces cut by the pattern, records counted (plans only)
//   (allocation scan, as in every call)
//   k_dash_write   thread per segment: the same walk, writing
// Thread per segment, as the paper's own kernel (L21) and this library's walk: dashing has not been moved onto the tiled,
// node-parallel count pass.  Every vertex of a dash is offset_point(V, T, r) of a global fp32 point V and a unit tangent T that
// the neighbouring piece, the cap and the join compute from the same bits: dashes are watertight outlines.
#pragma once
#include "sx_segment.cuh"
#include "sx_scan.cuh"   // (the error flags)

namespace sx {

constexpr int kDashThreads = 128;
constexpr float kDashUnit = 65536.0f;   // units per px

struct DashArgs {
    Params P;
    uint32_t nd;
    unsigned long long dq[8], period, phase_q;
    uint32_t* seg_len;                       // [n] the segments' arc lengths (units; 32 bits: < 65536 px per segment)
    const unsigned long long* seg_pos;       // [n] exclusive prefix sum of seg_len over the whole call
    unsigned long long* sp_total;            // [n] at a subpath's first segment: its total length
    uint32_t* seg_count;
    const uint64_t* seg_off;
    float4* out;
    uint64_t cap_records;
    uint32_t* err;
    uint32_t wide;
};

SX_DEV bool style_dashed(const Params& P, uint32_t path) {
    const uint4 raw = __ldg(reinterpret_cast<const uint4*>(P.styles) + path);
    return ((raw.z >> 17) & 1u) != 0u && ((raw.z >> 16) & 1u) == 0u;   // bit 1 of `fill`, and not a fill
}
SX_DEV unsigned long long dash_units(float L) { return (unsigned long long)__float2ll_rn(L * kDashUnit); }

// a straight segment as a piece of the dash walk (k0 = k1 = 0, L = its length)
SX_DEV Piece line_piece(const Seg& s) {
    Piece p;
    p.base = s.P0; p.P3 = s.P3;
    p.la = v2(0.0f, 0.0f); p.lb = s.P3 - s.P0;
    p.ua = s.ts; p.ub = s.te;
    p.ch = p.lb;
    p.k0 = 0.0f; p.k1 = 0.0f;
    p.L = sqrtf(len2(p.ch));
    p.at0 = p.at1 = true;
    return p;
}

// ---------------------------------------------------------------- arc length of a segment
__global__ void __launch_bounds__(kDashThreads)
k_dash_len(const DashArgs A) {
    const Params& P = A.P;
    const uint32_t i = blockIdx.x * (uint32_t)kDashThreads + threadIdx.x;
    if (i >= P.n_tags) return;
    uint32_t len = 0u;
    Style st;
    float h;
    if ((*A.err & kErrBadStream) == 0u && style_dashed(P, P.path_idx[i]) && load_style(P, P.path_idx[i], &st, &h)) {
        const Seg s = load_segment(P, i, P.tags[i]);
        unsigned long long sum = 0ull;
        if (s.kind == 1 || s.degenerate) {
            sum = dash_units(line_piece(s).L);
        } else {
            FitState f = fit_begin(s);
            Piece p;
            while (fit_next(P, s, f, p)) sum += dash_units(p.L);
        }
        if (sum > 0xffffffffull) { atomicOr(A.err, kErrBadStream); sum = 0ull; }   // a dashed segment of 65536 px or more: refused
        len = (uint32_t)sum;
    }
    A.seg_len[i] = len;
}

__global__ void __launch_bounds__(kDashThreads)
k_dash_totals(const DashArgs A) {
    const Params& P = A.P;
    const uint32_t i = blockIdx.x * (uint32_t)kDashThreads + threadIdx.x;
    if (i >= P.n_tags) return;
    const uint32_t tag = P.tags[i];
    if (((tag >> 2) | (tag >> 4)) & 1u) {
        const uint32_t f = P.sp_first[i];
        A.sp_total[f] = A.seg_pos[i] + A.seg_len[i] - A.seg_pos[f];
    }
}

// ---------------------------------------------------------------- the walk
struct DashState {
    unsigned long long S;       // arc position of the next piece's start within the subpath
    unsigned long long total;   // the subpath's length
};

// the sub-range [ta, tb] of piece p as a piece of its own, every end a global vertex (at0 = at1 = true)
template <bool EMIT>
SX_DEV Piece dash_sub_piece(const Piece& p, const Spiral& z, float ta, float tb, bool line) {
    Piece q = p;
    if (!line && (ta != 0.0f || tb != 1.0f)) {
        const float dt = tb - ta, tm = 0.5f * (ta + tb) - 0.5f;
        q.k0 = dt * (p.k0 + p.k1 * tm);
        q.k1 = p.k1 * dt * dt;
        q.L = p.L * dt;
        if (!(q.L > 1e-12f)) q.L = 1e-12f;
    }
    if (EMIT) {
        V2 Va = p.at0 ? p.base : v2(p.base.x + p.la.x, p.base.y + p.la.y), Vb = p.at1 ? p.P3 : v2(p.base.x + p.lb.x, p.base.y + p.lb.y);
        if (line) {
            if (ta != 0.0f) Va = v2(fmaf(ta, p.ch.x, p.base.x), fmaf(ta, p.ch.y, p.base.y));
            if (tb != 1.0f) Vb = v2(fmaf(tb, p.ch.x, p.base.x), fmaf(tb, p.ch.y, p.base.y));
        } else {
            V2 l, T;
            if (ta != 0.0f) { es_eval(p, z, ta, &l, &T); Va = v2(p.base.x + l.x, p.base.y + l.y); q.ua = T; }
            if (tb != 1.0f) { es_eval(p, z, tb, &l, &T); Vb = v2(p.base.x + l.x, p.base.y + l.y); q.ub = T; }
        }
        q.base = Va; q.P3 = Vb;
        q.la = v2(0.0f, 0.0f); q.lb = Vb - Va; q.ch = q.lb;
        q.at0 = q.at1 = true;
    }
    return q;
}

// one piece under the pattern: the records of the dashes that cross it, starting at index `first` of the segment
template <bool EMIT>
SX_DEV uint32_t dash_piece(const DashArgs& A, const Piece& p, bool line, DashState& d, const Style& st, float h, const Writer* w, uint32_t first) {
    const Params& P = A.P;
    const unsigned long long Lq = dash_units(p.L), S = d.S, E = S + Lq;
    d.S = E;
    if (Lq == 0ull) return 0u;   // a piece without length carries no part of a dash
    unsigned long long u = (S + A.phase_q) % A.period;
    uint32_t j = 0;
    while (u >= A.dq[j]) { u -= A.dq[j]; j++; }
    Spiral z, zq;
    bool z_ready = false;
    uint32_t n = 0;
    unsigned long long s = S;
    while (s < E) {
        const unsigned long long e = s + (A.dq[j] - u);
        if ((j & 1u) == 0u) {
            const unsigned long long b = e < E ? e : E;
            const bool starts = u == 0ull || s == 0ull, ends = e <= E || E == d.total;
            const float ta = s == S ? 0.0f : (float)(s - S) / (float)Lq;
            const float tb = b == E ? 1.0f : (float)(b - S) / (float)Lq;
            if (EMIT && !line && !z_ready && (ta != 0.0f || tb != 1.0f)) { es_prepare(p, z); z_ready = true; }
            const Piece q = dash_sub_piece<EMIT>(p, z, ta, tb, line);
            if (starts) n += emit_cap<EMIT>(P, st, q.base, v2(-q.ua.x, -q.ua.y), h, w, first + n);
            if (line) {
                if (EMIT) {
                    w->put(first + n, offset_point(q.base, q.ua, -h), offset_point(q.P3, q.ub, -h), 0.0f, kOffset);
                    w->put(first + n + 1u, offset_point(q.P3, q.ub, h), offset_point(q.base, q.ua, h), 0.0f, kOffset | kPlus);
                }
                n += 2u;
            } else {
                if (EMIT) es_prepare(q, zq);
                n += piece_side<EMIT>(q, zq, -h, false, P, w, first + n);
                n += piece_side<EMIT>(q, zq, h, true, P, w, first + n);
            }
            if (ends) n += emit_cap<EMIT>(P, st, EMIT ? q.P3 : q.base, q.ub, h, w, first + n);
        }
        s = e; u = 0ull; j = j + 1u == A.nd ? 0u : j + 1u;
    }
    return n;
}

// does a dash cover arc position s strictly inside?
SX_DEV bool dash_covers(const DashArgs& A, unsigned long long s, unsigned long long total) {
    if (s == 0ull || s >= total) return false;
    unsigned long long u = (s + A.phase_q) % A.period;
    uint32_t j = 0;
    while (u >= A.dq[j]) { u -= A.dq[j]; j++; }
    return (j & 1u) == 0u && u > 0ull;
}

// everything segment i emits (a path that is not dashed: the plain walk of sx_segment.cuh)
template <bool EMIT>
SX_DEV uint32_t dash_segment(const DashArgs& A, uint32_t i, const Writer* w) {
    const Params& P = A.P;
    const uint32_t path = P.path_idx[i];
    if (!style_dashed(P, path)) {
        Writer w2;
        if (EMIT) w2 = *w;
        return process_segment<EMIT>(P, i, &w2);
    }
    Style st;
    float h;
    if (!load_style(P, path, &st, &h)) return 0u;
    const uint32_t tag = P.tags[i], f0 = P.sp_first[i];
    const Seg s = load_segment(P, i, tag);
    DashState d;
    d.S = A.seg_pos[i] - A.seg_pos[f0];
    d.total = A.sp_total[f0];
    uint32_t n = 0;
    if (s.kind == 1 || s.degenerate) {
        n += dash_piece<EMIT>(A, line_piece(s), true, d, st, h, w, n);
    } else {
        FitState f = fit_begin(s);
        Piece p;
        while (fit_next(P, s, f, p)) n += dash_piece<EMIT>(A, p, false, d, st, h, w, n);
    }
    const bool sp_end = ((tag >> 2) | (tag >> 4)) & 1u;
    if (!sp_end && dash_covers(A, d.S, d.total)) {
        V2 W, T1;
        load_segment_start(P, i + 1u, &W, &T1);
        n += emit_join<EMIT>(P, st, s.P3, s.te, W, T1, h, w, n);
    }
    return n;
}

__global__ void __launch_bounds__(kDashThreads)
k_dash_count(const DashArgs A) {
    const uint32_t i = blockIdx.x * (uint32_t)kDashThreads + threadIdx.x;
    if (i >= A.P.n_tags) return;
    uint32_t n = 0u;
    if ((*A.err & kErrBadStream) == 0u) n = dash_segment<false>(A, i, nullptr);
    A.seg_count[i] = n;
}

__global__ void __launch_bounds__(kDashThreads)
k_dash_write(const DashArgs A) {
    const uint32_t i = blockIdx.x * (uint32_t)kDashThreads + threadIdx.x;
    if (i >= A.P.n_tags) return;
    const uint32_t count = A.seg_count[i];
    if (count == 0u) return;
    const uint64_t base = A.seg_off[i];
    if (base + count > A.cap_records) { atomicOr(A.err, kErrCapacity); return; }   // nothing of the segment is written
    Writer w;
    w.out = A.out; w.base = base; w.seg = i; w.mode = A.P.mode; w.wide = A.wide != 0u;
    dash_segment<true>(A, i, &w);
}

}  // namespace sx
