// sx_cache.cuh -- the record-indexed evaluation of one side of one Euler-spiral piece: packed side plans and PART tables.
//
// The general writer (k_write_general, sx_write.cuh) maps one thread to one OUTPUT RECORD (the per-output-point balance
// the paper leaves as future work, L585): a warp stages 16 pieces in shared memory, builds the two side plans of
// each (same device functions as the count pass, hence the same counts), turns them into a table of PARTS (below)
// and lets every thread locate its record by binary search over the parts.
#pragma once
#include "sx_segment.cuh"

namespace sx {

SX_DEV float f_of_u(uint32_t u) { return __uint_as_float(u); }
SX_DEV uint32_t u_of_f(float f) { return __float_as_uint(f); }

// ---------------------------------------------------------------- the side plan as the writer keeps it in shared memory
// 52 bytes instead of sizeof(SidePlan) = 100: range bounds are implied by the cusp parameter (range 0 = [0, tc],
// range 1 = [tc, 1]; the super-critical range is range 0 iff sup0), counts fit 16 bits.
struct PlanLite {
    float eta, tc;
    uint32_t seg, total;
    uint16_t n0, n1, ne;
    uint8_t flags;   // bit 0 two ranges, 1 sup0, 2 sup1, 3 refined f (mode 2), 5 uniform evolute, 6 evolute parameters by cubing (arc mode)
    uint8_t rules;   // spacing rule (kRule*) of range 0 | of range 1 << 2
    float ua0, ub0, ua1, ub1, wa, wb, skp;
};
SX_DEV PlanLite plan_pack(const SidePlan& s) {
    PlanLite q;
    q.eta = s.eta; q.tc = s.off[0].tb; q.seg = s.seg; q.total = (uint32_t)s.total;
    q.n0 = (uint16_t)s.off[0].n; q.n1 = (uint16_t)s.off[1].n; q.ne = (uint16_t)s.evo.n;
    q.flags = (uint8_t)((s.nr == 2 ? 1u : 0u) | (s.sup[0] ? 2u : 0u) | (s.sup[1] ? 4u : 0u) | (SX_OFF_REFINED(s.off[0]) ? 8u : 0u) | (s.evo.uniform ? 32u : 0u) | (s.evo.cube ? 64u : 0u));
    q.rules = (uint8_t)((uint32_t)s.off[0].rule | ((uint32_t)s.off[1].rule << 2));
    q.ua0 = s.off[0].ua; q.ub0 = s.off[0].ub; q.ua1 = s.off[1].ua; q.ub1 = s.off[1].ub;
    q.wa = s.evo.wa; q.wb = s.evo.wb; q.skp = s.evo.skp;
    return q;
}
SX_DEV OffPlan plan_off(const PlanLite& q, bool second) {
    OffPlan o;
    o.n = second ? q.n1 : q.n0;
    o.rule = (int)((q.rules >> (second ? 2 : 0)) & 3u);
    o.ta = second ? q.tc : 0.0f; o.tb = second ? 1.0f : q.tc;
    o.ua = second ? q.ua1 : q.ua0; o.ub = second ? q.ub1 : q.ub0;
#if SX_REFINED
    o.refined = (q.flags & 8u) != 0u;
#endif
    return o;
}
SX_DEV EvoPlan plan_evo(const PlanLite& q) {
    EvoPlan e;
    const bool second = (q.flags & 1u) && !(q.flags & 2u);  // two ranges and the first one regular
    e.n = q.ne; e.uniform = (q.flags & 32u) != 0u; e.cube = (q.flags & 64u) != 0u;
    e.ta = second ? q.tc : 0.0f; e.tb = second ? 1.0f : q.tc;
    e.wa = q.wa; e.wb = q.wb; e.skp = q.skp;
    return e;
}

// ---------------------------------------------------------------- parts
// The records of one side of one piece, in OUTPUT order, are a short list of PARTS (at most 8): chains of n
// records over n+1 vertices.  Vertex m of a part is either one of the part's two END vertices -- a piece end
// (t = 0 or t = 1, on the parallel curve or on the evolute) or the side's cusp point -- or the interior
// subdivision vertex of index i0 +- m of an offset range (sections 4, 5) or of the evolute (section 6).  This
// is piece_side<true> (sx_segment.cuh) turned into data: the writer's threads do not branch on what kind of
// record they own.  The mirror image of the +h side (reverse order, end points swapped) is folded into the
// table when it is built.
enum : uint32_t { kEndT0 = 0u, kEndT1 = 1u, kEndCusp = 2u, kEndEvo = 4u };  // end-vertex code: which point | evolute flag
struct __align__(16) Part {
    uint64_t base;   // output index of the part's first record
    uint16_t n;      // records (a single subdivision count is clamped to 65535)
    uint16_t i0;     // vertex m has subdivision index i0 + dir * m
    uint32_t info;   // 0-6 side slot, 7 dir < 0, 8-9 src (0 none, 1 offset range, 2 evolute), 10 range, 11 arc angle wanted,
                     // 12-15 record kind, 16-18 end code of vertex 0, 19-21 end code of vertex n
};  // 16 bytes
SX_DEV uint32_t end_code(float t) { return t == 0.0f ? kEndT0 : (t == 1.0f ? kEndT1 : kEndCusp); }

// number of parts of a side
SX_DEV uint32_t side_part_count(const SidePlan& s) {
    uint32_t c = (uint32_t)s.nr;  // one offset part per range
    if (s.sup[0] || (s.nr == 2 && s.sup[1])) c += 2u + (s.cusp_a ? 0u : 2u) + (s.cusp_b ? 0u : 2u);
    return c;
}

// part k (OUTPUT order) of the `count` parts of a side, and the number of the side's records before it: piece_side<true>
// (sx_segment.cuh) turned into data, one part at a time -- the general writer builds its table with one lane per PART (a
// lane per side spent 22 % of the kernel's instructions at 4 of 32 lanes on config 5, where a third of the pieces carry an
// evolute patch of 7 parts).  Forward order of a side with a super-critical range [ta, tb] (section 6):
// [regular range 0] [connector x2 unless the range starts at the cusp] [evolute x2] [reversed offset, L403 / L191]
// [connector x2 unless it ends at the cusp] [regular range 1]; the mirror image of the +h side reverses the list and each chain.
SX_DEV Part side_part_at(const PlanLite& q, uint32_t k, uint32_t count, uint32_t side_slot, bool mirror, bool arc, uint64_t side_base, uint32_t* before_out) {
    const uint32_t idx = mirror ? count - 1u - k : k;
    const bool two = (q.flags & 1u) != 0u, sup0 = (q.flags & 2u) != 0u, sup1 = two && (q.flags & 4u) != 0u;
    const uint32_t n0 = q.n0, n1 = q.n1, ne = q.ne;
    const float tc = q.tc;   // range 0 = [0, tc], range 1 = [tc, 1]; tc = 1 when there is one range
    uint32_t n = 0, src = 1u, ri = 0u, kind = kOffset, f0 = 0u, f1 = 0u, fwd = 0u;
    int32_t i0 = 0;
    bool dirneg = false, angle = true;
    if (!(sup0 || sup1)) {   // regular ranges only
        ri = idx;
        n = idx ? n1 : n0;
        f0 = end_code(idx ? tc : 0.0f); f1 = end_code(idx ? 1.0f : tc);
        fwd = idx ? n0 : 0u;
    } else {
        const uint32_t sr = sup0 ? 0u : 1u, nsr = sr ? n1 : n0;   // the super-critical range and its offset count
        const float ta = sr ? tc : 0.0f, tb = sr ? 1.0f : tc;
        const uint32_t ca = end_code(ta), cb = end_code(tb);
        const bool cusp_a = ta != 0.0f, cusp_b = tb != 1.0f;
        const uint32_t ea = cusp_a ? (uint32_t)kEndCusp : (ca | kEndEvo), eb = cusp_b ? (uint32_t)kEndCusp : (cb | kEndEvo);
        const uint32_t nca = cusp_a ? 0u : 2u, ncb = cusp_b ? 0u : 2u;
        uint32_t i = idx;
        if (i < sr) {   // the regular range 0 before the patch
            n = n0; f0 = end_code(0.0f); f1 = end_code(tc);
        } else {
            i -= sr; fwd = sr ? n0 : 0u;
            if (i < nca) { n = 1u; src = 0u; angle = false; kind = kConnector; f0 = ca; f1 = ea; fwd += i; }
            else {
                i -= nca; fwd += nca;
                if (i < 2u) { n = ne; src = 2u; kind = kEvolute; f0 = ea; f1 = eb; fwd += i * ne; }   // (arc mode: the evolute turns with the spiral)
                else {
                    fwd += 2u * ne;
                    if (i == 2u) { n = nsr; i0 = (int32_t)nsr; dirneg = true; ri = sr; kind = kOffsetRev; f0 = cb; f1 = ca; }
                    else {
                        i -= 3u; fwd += nsr;
                        if (i < ncb) { n = 1u; src = 0u; angle = false; kind = kConnector; f0 = eb; f1 = cb; fwd += i; }
                        else { fwd += ncb; n = n1; ri = 1u; f0 = end_code(tc); f1 = end_code(1.0f); }   // the regular range 1 after the patch
                    }
                }
            }
        }
    }
    uint32_t before = fwd;
    if (mirror) {   // reverse the list, reverse each chain
        before = q.total - fwd - n;
        i0 = dirneg ? i0 - (int32_t)n : i0 + (int32_t)n; dirneg = !dirneg;
        const uint32_t t = f0; f0 = f1; f1 = t;
        kind |= kPlus;
    }
    Part r;
    r.base = side_base + before; r.n = (uint16_t)n; r.i0 = (uint16_t)i0;
    r.info = side_slot | (dirneg ? 128u : 0u) | (src << 8) | (ri << 10) | ((angle && arc) ? 2048u : 0u) | (kind << 12) | (f0 << 16) | (f1 << 19);
    *before_out = before;
    return r;
}

// an END vertex of a part: same arithmetic as normal_point at t = 0 / t = 1; the cusp point is evaluated once per
// side (normal_point at the cusp parameter) and shared by the parts that meet there
SX_DEV V2 end_vertex(const Piece& p, uint32_t code, float eta, float4 cusp, float* t_out) {
    const uint32_t which = code & 3u;
    const bool e1 = which == kEndT1;
    const float t = e1 ? 1.0f : 0.0f;
    const V2 l = e1 ? p.lb : p.la, T = e1 ? p.ub : p.ua;
    const float r = (code & kEndEvo) ? es_radius(p, t) : eta;
    V2 g = v2(p.base.x + fmaf(r, -T.y, l.x), p.base.y + fmaf(r, T.x, l.y));
    if (e1 ? p.at1 : p.at0) g = offset_point(e1 ? p.P3 : p.base, T, r);
    *t_out = t;
    if (which == kEndCusp) { g = v2(cusp.x, cusp.y); *t_out = cusp.z; }
    return g;
}

}  // namespace sx
