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
    p.zready = false;
}

// ---------------------------------------------------------------- record j (forward-t order) of one side
// Same vertices, in the same order, as piece_side<true> (sx_segment.cuh) walks sequentially.
SX_DEV void side_record(Piece& p, const SidePlan& s, float eta, bool arc, uint32_t j, V2* a, V2* b, float* angle, uint32_t* kind) {
    *angle = 0.0f;
#pragma unroll
    for (int r = 0; r < 2; r++) {
        if (r >= s.nr) break;
        const OffPlan o = r == 0 ? s.off[0] : s.off[1];
        const bool sup = r == 0 ? s.sup[0] : s.sup[1];
        const uint32_t n = (uint32_t)o.n;
        if (!sup) {
            if (j < n) {
                float t0 = j == 0u ? o.ta : offset_t(p, o, eta, (int)j);
                float t1 = j + 1u == n ? o.tb : offset_t(p, o, eta, (int)j + 1);
                *a = es_offset(p, t0, eta);
                *b = es_offset(p, t1, eta);
                if (arc) *angle = es_dphi(p, t0, t1);
                *kind = kOffset;
                return;
            }
            j -= n;
        } else {
            // evolute patch (section 6): connectors x2, evolute x2, reversed offset, connectors x2
            const uint32_t nca = s.cusp_a ? 0u : 2u, ncb = s.cusp_b ? 0u : 2u, ne = (uint32_t)s.evo.n;
            const uint32_t tot = nca + 2u * ne + n + ncb;
            if (j < tot) {
                if (j < nca) {
                    *a = es_offset(p, o.ta, eta); *b = es_evolute(p, o.ta); *kind = kConnector;
                } else if (j < nca + 2u * ne) {
                    uint32_t i = j - nca;
                    if (i >= ne) i -= ne;
                    *a = i == 0u ? (s.cusp_a ? es_offset(p, o.ta, eta) : es_evolute(p, o.ta)) : es_evolute(p, evolute_t(p, s.evo, (int)i));
                    *b = i + 1u == ne ? (s.cusp_b ? es_offset(p, o.tb, eta) : es_evolute(p, o.tb)) : es_evolute(p, evolute_t(p, s.evo, (int)i + 1));
                    *kind = kEvolute;
                } else if (j < nca + 2u * ne + n) {
                    uint32_t hi = n - (j - (nca + 2u * ne)), lo = hi - 1u;  // reversed offset (L403, L191): vertex hi -> vertex lo
                    float t1 = hi == n ? o.tb : offset_t(p, o, eta, (int)hi);
                    float t0 = lo == 0u ? o.ta : offset_t(p, o, eta, (int)lo);
                    *a = es_offset(p, t1, eta);
                    *b = es_offset(p, t0, eta);
                    if (arc) *angle = es_dphi(p, t1, t0);
                    *kind = kOffsetRev;
                } else {
                    *a = es_evolute(p, o.tb); *b = es_offset(p, o.tb, eta); *kind = kConnector;
                }
                return;
            }
            j -= tot;
        }
    }
    *a = *b = v2(0.0f, 0.0f);
    *kind = kOffset;
}

}  // namespace sx
