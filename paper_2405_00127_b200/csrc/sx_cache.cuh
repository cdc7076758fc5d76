// sx_cache.cuh -- the piece cache between the count kernel (b) and the write kernel (d), and the
// record-indexed evaluation of one side of one Euler-spiral piece.
//
// The count kernel runs Alg. 2 once per curve segment and stores every accepted
// Euler-spiral piece as an 80-byte descriptor; the write kernel never repeats the cubic -> spiral fit.
// It maps one thread to one OUTPUT RECORD (the per-output-point balance the paper leaves as future
// work, L585): a block stages a tile of descriptors in shared memory, rebuilds the two side plans of
// each piece (same device functions as the count kernel, hence the same counts), scans the plan totals
// and lets every thread locate its record by binary search.
#pragma once
#include "sx_segment.cuh"

namespace sx {

constexpr uint32_t kInvalidSeg = 0xffffffffu;
constexpr uint32_t kRelMask = 0x3fffffffu, kAt0Bit = 1u << 30, kAt1Bit = 1u << 31;
constexpr int kDescQuads = 5;   // 5 x 16 B
constexpr int kChunk = 32;      // descriptor slots a warp reserves per atomic

SX_DEV float f_of_u(uint32_t u) { return __uint_as_float(u); }
SX_DEV uint32_t u_of_f(float f) { return __float_as_uint(f); }

// q0: P0 P3 | q1: la lb | q2: ua ub | q3: k0 k1 L h | q4: seg, rel|flags, n_minus, n_plus
SX_DEV void piece_store(float4* slot, const Piece& p, float h, uint32_t seg, uint32_t rel, uint32_t n_minus, uint32_t n_plus) {
    slot[0] = make_float4(p.base.x, p.base.y, p.P3.x, p.P3.y);
    slot[1] = make_float4(p.la.x, p.la.y, p.lb.x, p.lb.y);
    slot[2] = make_float4(p.ua.x, p.ua.y, p.ub.x, p.ub.y);
    slot[3] = make_float4(p.k0, p.k1, p.L, h);
    uint32_t r = (rel & kRelMask) | (p.at0 ? kAt0Bit : 0u) | (p.at1 ? kAt1Bit : 0u);
    slot[4] = make_float4(f_of_u(seg), f_of_u(r), f_of_u(n_minus), f_of_u(n_plus));
}
SX_DEV void piece_invalidate(float4* slot) { slot[4] = make_float4(f_of_u(kInvalidSeg), 0.0f, 0.0f, 0.0f); }

struct PieceHead { uint32_t seg, rel, n_minus, n_plus; bool at0, at1; };
SX_DEV PieceHead piece_head(const float4* slot) {
    float4 q = __ldg(slot + 4);
    PieceHead hd;
    hd.seg = u_of_f(q.x);
    uint32_t r = u_of_f(q.y);
    hd.rel = r & kRelMask; hd.at0 = (r & kAt0Bit) != 0u; hd.at1 = (r & kAt1Bit) != 0u;
    hd.n_minus = u_of_f(q.z); hd.n_plus = u_of_f(q.w);
    return hd;
}
SX_DEV void piece_load(const float4* slot, const PieceHead& hd, Piece& p, float* h) {
    float4 a = __ldg(slot), b = __ldg(slot + 1), c = __ldg(slot + 2), d = __ldg(slot + 3);
    p.base = v2(a.x, a.y); p.P3 = v2(a.z, a.w);
    p.la = v2(b.x, b.y); p.lb = v2(b.z, b.w);
    p.ua = v2(c.x, c.y); p.ub = v2(c.z, c.w);
    p.ch = p.lb - p.la;  // the same subtraction fit_next performed
    p.k0 = d.x; p.k1 = d.y; p.L = d.z; *h = d.w;
    p.at0 = hd.at0; p.at1 = hd.at1;
}

// ---------------------------------------------------------------- record j (forward-t order) of one side
// Same vertices, in the same order, as piece_side<true> (sx_segment.cuh) walks sequentially.  The record
// index is first DECODED into two vertex specifications (cheap integer logic, where the threads of a warp
// may diverge); the expensive part -- subdivision parameter, Euler-spiral integral, normal offset -- then
// runs once per end point in a single code path that every thread of the warp executes together.
struct VertexSpec {
    float t;      // parameter when src == 0
    int i;        // subdivision index when src != 0
    int src;      // 0: t given, 1: offset_t(i), 2: evolute_t(i)
    bool evo;     // point on the evolute (r = 1/kappa) instead of the parallel curve (r = eta)
};
SX_DEV VertexSpec vs_fixed(float t, bool evo) { VertexSpec v; v.t = t; v.i = 0; v.src = 0; v.evo = evo; return v; }
SX_DEV VertexSpec vs_offset(const OffPlan& o, uint32_t i) {
    VertexSpec v; v.evo = false; v.i = (int)i; v.t = i == 0u ? o.ta : o.tb; v.src = (i == 0u || i == (uint32_t)o.n) ? 0 : 1; return v;
}
SX_DEV VertexSpec vs_evolute(const SidePlan& s, const OffPlan& o, uint32_t i) {
    const uint32_t ne = (uint32_t)s.evo.n;
    if (i == 0u) return vs_fixed(o.ta, !s.cusp_a);   // the evolute meets the offset curve at the cusp
    if (i == ne) return vs_fixed(o.tb, !s.cusp_b);
    VertexSpec v; v.evo = true; v.i = (int)i; v.t = 0.0f; v.src = 2; return v;
}

SX_DEV void side_record(const Piece& p, const Spiral& z, const SidePlan& s, float eta, bool arc, uint32_t j, V2* a, V2* b, float* angle, uint32_t* kind) {
    VertexSpec va = vs_fixed(0.0f, false), vb = va;
    OffPlan o = s.off[0];
    bool want_angle = false;
    *kind = kOffset;
#pragma unroll
    for (int r = 0; r < 2; r++) {
        if (r >= s.nr) break;
        const OffPlan oo = r == 0 ? s.off[0] : s.off[1];
        const bool sup = r == 0 ? s.sup[0] : s.sup[1];
        const uint32_t n = (uint32_t)oo.n;
        if (!sup) {
            if (j < n) {
                o = oo; va = vs_offset(oo, j); vb = vs_offset(oo, j + 1u); want_angle = arc; *kind = kOffset;
                break;
            }
            j -= n;
        } else {
            // evolute patch (section 6): connectors x2, evolute x2, reversed offset, connectors x2
            const uint32_t nca = s.cusp_a ? 0u : 2u, ncb = s.cusp_b ? 0u : 2u, ne = (uint32_t)s.evo.n;
            const uint32_t tot = nca + 2u * ne + n + ncb;
            if (j < tot) {
                o = oo;
                if (j < nca) {
                    va = vs_fixed(oo.ta, false); vb = vs_fixed(oo.ta, true); *kind = kConnector;
                } else if (j < nca + 2u * ne) {
                    uint32_t i = j - nca;
                    if (i >= ne) i -= ne;
                    va = vs_evolute(s, oo, i); vb = vs_evolute(s, oo, i + 1u); *kind = kEvolute;
                } else if (j < nca + 2u * ne + n) {
                    uint32_t hi = n - (j - (nca + 2u * ne));  // reversed offset (L403, L191): vertex hi -> vertex hi-1
                    va = vs_offset(oo, hi); vb = vs_offset(oo, hi - 1u); want_angle = arc; *kind = kOffsetRev;
                } else {
                    va = vs_fixed(oo.tb, true); vb = vs_fixed(oo.tb, false); *kind = kConnector;
                }
                break;
            }
            j -= tot;
        }
    }
    // ---- the convergent part
    float t0 = 0.0f, t1 = 0.0f;
    V2 p0 = v2(0.0f, 0.0f), p1 = p0;
#pragma unroll 1
    for (int e = 0; e < 2; e++) {
        const VertexSpec v = e == 0 ? va : vb;
        float t = v.t;
        if (v.src == 1) t = offset_t(p, o, eta, v.i);
        else if (v.src == 2) t = evolute_t(p, s.evo, v.i);
        const float r = v.evo ? 1.0f / es_kappa(p, t) : eta;
        const V2 g = normal_point(p, z, t, r);
        if (e == 0) { t0 = t; p0 = g; } else { t1 = t; p1 = g; }
    }
    *a = p0; *b = p1;
    *angle = want_angle ? es_dphi(p, t0, t1) : 0.0f;
}

}  // namespace sx
