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
SX_DEV EvoPlan plan_evo(const PlanLite& q);
// the fields of the SidePlan that the part table is built from
SX_DEV SidePlan plan_unpack(const PlanLite& q) {
    SidePlan s;
    s.eta = q.eta; s.seg = q.seg; s.total = (int)q.total;
    s.nr = (q.flags & 1u) ? 2 : 1;
    s.sup[0] = (q.flags & 2u) != 0u; s.sup[1] = (q.flags & 4u) != 0u;
    s.off[0] = plan_off(q, false); s.off[1] = plan_off(q, true);
    s.evo = plan_evo(q);
    s.cusp_a = s.evo.ta != 0.0f; s.cusp_b = s.evo.tb != 1.0f;
    return s;
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

// writes the parts of a side (output order) to dst[0..count), and their tile-relative record prefixes to pref[]
SX_DEV void side_parts(const SidePlan& s, uint32_t side_slot, bool mirror, bool arc, uint64_t side_base, uint32_t tile_prefix,
                       uint32_t count, Part* dst, uint32_t* pref) {
    uint32_t idx = 0, fwd = 0;  // forward part index, records before the part in forward order
    const uint32_t total = (uint32_t)s.total;
    auto push = [&](uint32_t n, int32_t i0, bool dirneg, uint32_t src, uint32_t ri, bool angle, uint32_t kind, uint32_t f0, uint32_t f1) {
        Part q;
        uint32_t pos = idx, before = fwd;
        if (mirror) {  // reverse the list, reverse each chain
            pos = count - 1u - idx; before = total - fwd - n;
            i0 = dirneg ? i0 - (int32_t)n : i0 + (int32_t)n; dirneg = !dirneg;
            uint32_t t = f0; f0 = f1; f1 = t;
            kind |= kPlus;
        }
        q.base = side_base + before; q.n = (uint16_t)n; q.i0 = (uint16_t)i0;
        q.info = side_slot | (dirneg ? 128u : 0u) | (src << 8) | (ri << 10) | ((angle && arc) ? 2048u : 0u) | (kind << 12) | (f0 << 16) | (f1 << 19);
        dst[pos] = q;
        pref[pos] = tile_prefix + before;
        idx++; fwd += n;
    };
#pragma unroll 1
    for (int r = 0; r < s.nr; r++) {
        const OffPlan o = r == 0 ? s.off[0] : s.off[1];
        const bool sup = r == 0 ? s.sup[0] : s.sup[1];
        const uint32_t ca = end_code(o.ta), cb = end_code(o.tb);
        if (!sup) {
            push((uint32_t)o.n, 0, false, 1u, (uint32_t)r, true, kOffset, ca, cb);
        } else {
            // evolute patch (section 6): connectors x2, evolute x2, reversed offset, connectors x2;
            // the evolute meets the offset curve at the cusp.  (Loops, not copies: code size.)
            const uint32_t ea = s.cusp_a ? (uint32_t)kEndCusp : (ca | kEndEvo), eb = s.cusp_b ? (uint32_t)kEndCusp : (cb | kEndEvo);
#pragma unroll 1
            for (int c = 0; c < (s.cusp_a ? 0 : 2); c++) push(1u, 0, false, 0u, 0u, false, kConnector, ca, ea);
#pragma unroll 1
            for (int c = 0; c < 2; c++) push((uint32_t)s.evo.n, 0, false, 2u, 0u, true, kEvolute, ea, eb);   // (arc mode: the evolute turns with the spiral)
            push((uint32_t)o.n, o.n, true, 1u, (uint32_t)r, true, kOffsetRev, cb, ca);  // L403, L191
#pragma unroll 1
            for (int c = 0; c < (s.cusp_b ? 0 : 2); c++) push(1u, 0, false, 0u, 0u, false, kConnector, eb, cb);
        }
    }
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
