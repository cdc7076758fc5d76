// sx_write.cuh -- (d) the write pass: four small kernels, each with one job, all reading what the count pass left
// (seg_count, seg_tail, the allocation scan's seg_off, the 32-byte leaf records) and none repeating the fit.
//
//   k_write_segments   thread per input segment: the two exact offset lines of a straight segment (R-1b), the join with
//                      the next segment or the caps (Alg. 1; sx_segment.cuh).
//   k_write_simple     thread per leaf over the SIMPLE leaves (both sides one regular range of at most
//                      kDirectMax records): end points from the cubic, interior vertices from the spiral, no tables.
//   k_write_general    warp per 16 leaves over the other leaves, thread per output record: side plans, spiral anchors and
//                      the part tables of sx_cache.cuh staged in shared memory, 32 records per iteration, interior
//                      vertices evaluated densely into a ring just ahead of the records (evolute patches, cusps, long
//                      sides: everything the per-thread writer would diverge on).
//   k_write_walk       thread per segment of the walk list (what did not fit the count pass's tables or the leaf
//                      buffer): the thread-per-segment walk of sx_segment.cuh.
// Every vertex is a pure function of (segment, dyadic parameter, side): pieces that meet share bits, and so do the
// writers (watertight outlines).
#pragma once
#include "sx_count.cuh"
#include "sx_cache.cuh"

namespace sx {

constexpr int kExParts = 64;                         // part table of a stage (8 sides x 8 parts always fit)
constexpr int kRing = 64;                            // interior vertices kept ahead of the records (>= 2 x 32)
constexpr int kWrThreads = 128;

struct WriteArgs {
    Params P;
    const uint32_t* seg_count;
    const uint32_t* seg_tail;
    const uint64_t* seg_off;
    const LeafRec* leaves;
    uint32_t leaf_cap;
    const unsigned long long* leaf_counter;
    const uint32_t* leaf_end_inv;
    const uint32_t* walk_list;
    const uint32_t* walk_count;
    float4* out;
    uint64_t cap_records;
    uint32_t* err;
    uint32_t wide;   // the output buffer is 32-byte aligned: arc records go out as 256-bit stores
};

SX_DEV uint32_t n_simple_leaves(const WriteArgs& A) {
    const uint32_t reserved = (uint32_t)(*A.leaf_counter & 0xffffffffull), valid = ~A.leaf_end_inv[0];
    return reserved < valid ? reserved : valid;
}
SX_DEV uint32_t n_other_leaves(const WriteArgs& A) {
    const uint32_t reserved = (uint32_t)(*A.leaf_counter >> 32), valid = ~A.leaf_end_inv[1];
    return reserved < valid ? reserved : valid;
}
SX_DEV LeafRec load_leaf(const LeafRec* p) {
    // (one 256-bit load, sm_100)
    uint4 a, b;
    asm volatile("ld.global.nc.v8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];" : "=r"(a.x), "=r"(a.y), "=r"(a.z), "=r"(a.w), "=r"(b.x), "=r"(b.y), "=r"(b.z), "=r"(b.w) : "l"(p));
    LeafRec r;
    r.seg = a.x; r.key = a.y; r.n = a.z; r.rel = a.w;
    r.k0 = __uint_as_float(b.x); r.k1 = __uint_as_float(b.y); r.L = __uint_as_float(b.z); r.h = __uint_as_float(b.w);
    return r;
}

// the piece of a leaf record: the segment's control points (transform, degree elevation: the same load_segment_at the
// count pass used), the end points and tangents at the two dyadic parameters (the same cubic_point), the stored k0, k1, L
SX_DEV void leaf_piece(const Params& P, const LeafRec& r, Piece& p) {
    const Seg s = load_segment_at(P, P.pt_off[r.seg], P.tags[r.seg]);
    const uint32_t t0_u = r.key & 0xffffu, level = (r.key >> 16) & 31u;
    const float dt = __uint_as_float((127u - level) << 23);
    p.base = s.P0; p.P3 = s.P3;
    p.at0 = t0_u == 0u; p.at1 = t0_u + 1u == (1u << level);
    float qm, q2;
    float4 a = cubic_point(s, (float)t0_u * dt, &qm, &q2), b = cubic_point(s, (float)(t0_u + 1u) * dt, &qm, &q2);
    if (p.at0) a = make_float4(0.0f, 0.0f, s.ts.x, s.ts.y);
    if (p.at1) b = make_float4(s.c3.x, s.c3.y, s.te.x, s.te.y);
    p.la = v2(a.x, a.y); p.ua = v2(a.z, a.w);
    p.lb = v2(b.x, b.y); p.ub = v2(b.z, b.w);
    p.ch = p.lb - p.la;
    p.k0 = r.k0; p.k1 = r.k1; p.L = r.L;
}

SX_DEV void put_record(float4* out, bool arc, bool wide, uint64_t rec, V2 a, V2 b, float angle, uint32_t seg, uint32_t kind) {
    if (!arc) out[rec] = make_float4(a.x, a.y, b.x, b.y);
    else store_arc(out, rec, wide, make_float4(a.x, a.y, b.x, b.y), make_float4(angle, f_of_u(seg), f_of_u(kind), 0.0f));
}

// ---------------------------------------------------------------- straight segments, joins, caps
__global__ void __launch_bounds__(kWrThreads)
k_write_segments(const WriteArgs A) {
    const Params& P = A.P;
    const uint32_t i = blockIdx.x * (uint32_t)kWrThreads + threadIdx.x;
    const bool in = i < P.n_tags;
    const uint32_t ii = in ? i : P.n_tags - 1u;
    // first level of loads in one batch (the kernel is bound by the latency of its dependent loads)
    const uint32_t count = in ? A.seg_count[ii] : 0u, tail = A.seg_tail[ii], tag = P.tags[ii], pt = P.pt_off[ii], path = P.path_idx[ii], first_seg = P.sp_first[ii];
    const uint64_t base = A.seg_off[ii];
    Style st;
    float h;
    load_style(P, path, &st, &h);
    const Seg s = load_segment_at(P, pt, tag);
    // the join partner of a segment that does not end its subpath is the next segment: the next lane's start point and start
    // tangent (the same load_segment_at, hence the bits the partner itself uses); only the warp's last lane and the segments
    // that close a subpath or carry the caps load theirs
    const int lane = threadIdx.x & 31;
    V2 W, T1;
    W.x = __shfl_down_sync(kFull, s.P0.x, 1); W.y = __shfl_down_sync(kFull, s.P0.y, 1);
    T1.x = __shfl_down_sync(kFull, s.ts.x, 1); T1.y = __shfl_down_sync(kFull, s.ts.y, 1);
    if (count == 0u) return;   // width <= 0, a malformed stream, or beyond the end
    if (base + count > A.cap_records) { atomicOr(A.err, kErrCapacity); return; }   // nothing of the segment is written
    const bool sp_end = ((tag >> 2) | (tag >> 4)) & 1u;
    if (sp_end) { if (!st.fill || !((tag >> 7) & 1u)) load_segment_start(P, first_seg, &W, &T1); }
    else if (lane == 31) load_segment_start(P, i + 1u, &W, &T1);
    Writer w;
    w.out = A.out; w.base = base; w.seg = i; w.mode = P.mode; w.wide = A.wide != 0u;
    uint32_t first = count - tail;
    if (s.kind == 1 || s.degenerate) first = emit_straight(s, h, st.fill, &w);
    segment_tail_given<true>(P, tag, s, st, h, W, T1, &w, first);
}

// ---------------------------------------------------------------- simple leaves: thread per leaf
// control points of a curve segment (quadratic or cubic) without its tangents: what load_segment_at computes, branch-free
// (the same expressions, hence the same bits); l* / e*: the legs pick_tangent chooses the start / end tangent from
struct Ctrl { V2 P0, P3, c1, c2, c3, l1, l2, l3, e1, e2, e3; };
SX_DEV Ctrl load_ctrl(const Params& P, uint32_t pt, uint32_t tag) {
    const bool cubic = (tag & 3u) == 3u;
    const float* p = P.pts + 2 * (uint64_t)pt;
    const float2 a0 = ldg2(p), a1 = ldg2(p + 2), a2 = ldg2(p + 4), a3 = ldg2(p + (cubic ? 6 : 4));
    const V2 q0 = xform(P.A, a0.x, a0.y), q1 = xform(P.A, a1.x, a1.y), q2 = xform(P.A, a2.x, a2.y), q3 = xform(P.A, a3.x, a3.y);
    Ctrl c;
    c.P0 = q0; c.P3 = q3;
    const V2 a = q1 - q0, b = q2 - q0, d = q3 - q0;
    // quadratic (L349): c1 = 2/3 a, c2 = b + 2/3 (a - b), c3 = b; cubic: the control points themselves
    const V2 e1q = v2(a.x * (2.0f / 3.0f), a.y * (2.0f / 3.0f));
    const V2 e2q = v2(b.x + (a.x - b.x) * (2.0f / 3.0f), b.y + (a.y - b.y) * (2.0f / 3.0f));
    c.c1 = cubic ? a : e1q; c.c2 = cubic ? b : e2q; c.c3 = cubic ? d : b;
    c.l1 = a; c.l2 = b; c.l3 = cubic ? d : b;
    c.e1 = cubic ? d - b : b - a; c.e2 = cubic ? d - a : b; c.e3 = cubic ? d : b;
    return c;
}

__global__ void __launch_bounds__(kWrThreads, 6)
k_write_simple(const WriteArgs A) {
    const Params& P = A.P;
    const bool arc = P.mode == kModeArc;
    const uint64_t n_leaves = n_simple_leaves(A);
    // thread per LEAF: the segment's control points and the piece's two end points once, then its two sides (their records
    // are neighbours in the output: [-h side][+h side]).  The count pass stores a tile's one-record leaves first, so the
    // warps here are (mostly) of one kind.
    for (uint64_t idx = (uint64_t)blockIdx.x * kWrThreads + threadIdx.x; idx < n_leaves; idx += (uint64_t)gridDim.x * kWrThreads) {
        const LeafRec r = load_leaf(A.leaves + idx);
        const uint32_t n_minus = r.n & 0xffffu, n_plus = r.n >> 16;
        const uint64_t leaf_base = A.seg_off[r.seg] + r.rel;
        const Ctrl c = load_ctrl(P, P.pt_off[r.seg], P.tags[r.seg]);
        // the piece's end points: at an end of the segment the cubic's own point and limit tangent (R-5), inside it
        // cubic_point() as in the count pass
        const uint32_t t0_u = r.key & 0xffffu, level = (r.key >> 16) & 31u;
        const float dt = __uint_as_float((127u - level) << 23);
        Seg s;
        s.kind = 3; s.degenerate = false; s.P0 = c.P0; s.P3 = c.P3; s.c1 = c.c1; s.c2 = c.c2; s.c3 = c.c3;
        s.ts = s.te = v2(0.0f, 0.0f);
        Piece p;
        p.base = c.P0; p.P3 = c.P3; p.at0 = t0_u == 0u; p.at1 = t0_u + 1u == (1u << level);
        float4 pa = make_float4(0.0f, 0.0f, 0.0f, 0.0f), pb = pa;
#pragma unroll 1
        for (int k = 0; k < 2; k++) {
            float4 q;
            if (k ? p.at1 : p.at0) {
                bool dg;
                const V2 u = pick_tangent(k ? c.e1 : c.l1, k ? c.e2 : c.l2, k ? c.e3 : c.l3, &dg);
                q = k ? make_float4(c.c3.x, c.c3.y, u.x, u.y) : make_float4(0.0f, 0.0f, u.x, u.y);
            } else {
                float qm, q2;
                q = cubic_point(s, (float)(t0_u + (uint32_t)k) * dt, &qm, &q2);
            }
            if (k) pb = q; else pa = q;
        }
        p.la = v2(pa.x, pa.y); p.ua = v2(pa.z, pa.w);
        p.lb = v2(pb.x, pb.y); p.ub = v2(pb.z, pb.w);
        p.ch = p.lb - p.la;
        p.k0 = r.k0; p.k1 = r.k1; p.L = r.L;
        const float4 nocusp = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        Spiral z;
        if (n_minus > 1u || n_plus > 1u) es_prepare(p, z);
#pragma unroll 1
        for (int side = 0; side < 2; side++) {
            const uint32_t nrec = side ? n_plus : n_minus;
            const uint64_t base = leaf_base + (side ? n_minus : 0u);
            if (base + nrec > A.cap_records) { atomicOr(A.err, kErrCapacity); continue; }   // the side is not written
            const float eta = side ? r.h : -r.h;
            const uint32_t kind = side ? (uint32_t)(kOffset | kPlus) : (uint32_t)kOffset;
            OffPlan o;
            o.n = (int)nrec; o.rule = kRuleUniform; o.ta = 0.0f; o.tb = 1.0f; o.ua = o.ub = 0.0f;
#if SX_REFINED
            o.refined = false;
#endif
            if (nrec > 1u && !arc) o = offset_plan_call(p.k0, p.k1, p.L, eta, 0.0f, 1.0f, P.mode, P.tol_fl);   // (same call, same count as in the count pass)
            float tp;
            V2 prev = end_vertex(p, kEndT0, eta, nocusp, &tp);
            for (uint32_t i = 1; i <= nrec; i++) {
                float t;
                V2 cur;
                if (i < nrec) { t = offset_t(p, o, eta, (int)i); cur = normal_point(p, z, t, eta); }
                else cur = end_vertex(p, kEndT1, eta, nocusp, &t);
                const uint64_t rec = base + (side ? nrec - i : i - 1u);
                put_record(A.out, arc, A.wide != 0u, rec, side ? cur : prev, side ? prev : cur, (side ? es_dphi(p, t, tp) : es_dphi(p, tp, t)) + 0.0f, r.seg, kind);
                prev = cur; tp = t;
            }
        }
    }
}

// ---------------------------------------------------------------- the other leaves: thread per record
struct PieceLite {   // what a record needs of its piece (Piece without the derived chord)
    float bx, by, p3x, p3y, lax, lay, lbx, lby, uax, uay, ubx, uby, k0, k1, L;
    uint32_t flags;  // bit 0 at0, 1 at1
};
SX_DEV void piece_of(const PieceLite& q, Piece& p) {
    p.base = v2(q.bx, q.by); p.P3 = v2(q.p3x, q.p3y);
    p.la = v2(q.lax, q.lay); p.lb = v2(q.lbx, q.lby);
    p.ua = v2(q.uax, q.uay); p.ub = v2(q.ubx, q.uby);
    p.ch = p.lb - p.la;
    p.k0 = q.k0; p.k1 = q.k1; p.L = q.L;
    p.at0 = (q.flags & 1u) != 0u; p.at1 = (q.flags & 2u) != 0u;
}
struct WarpStage {
    float4 cusp[32];
    float4 ring[kRing];
    Part part[kExParts];
    Spiral spiral[16];
    PlanLite plan[32];
    PieceLite piece[16];
    uint32_t ppref[kExParts + 1];
    uint32_t pad[3];
};

__global__ void __launch_bounds__(kWrThreads)
k_write_general(const WriteArgs A) {
    __shared__ WarpStage stage[kWrThreads / 32];
    const Params& P = A.P;
    const int lane = threadIdx.x & 31;
    WarpStage& W = stage[threadIdx.x >> 5];
    const bool arc = P.mode == kModeArc;
    const int side = lane & 1;
    float4* const out = A.out;
    const uint32_t n_leaf = n_other_leaves(A);
    const uint32_t warps = gridDim.x * (uint32_t)(kWrThreads / 32), warp_id = blockIdx.x * (uint32_t)(kWrThreads / 32) + (threadIdx.x >> 5);
    for (uint32_t chunk = warp_id; (uint64_t)chunk * 16u < n_leaf; chunk += warps) {
        // ---- stage: lane = (leaf, side)
        const uint32_t li = chunk * 16u + (uint32_t)(lane >> 1);
        const bool live = li < n_leaf;
        Piece p;
        p.k0 = 0.0f; p.k1 = 0.0f; p.L = 1.0f;
        p.la = p.lb = p.ua = p.ub = p.ch = p.base = p.P3 = v2(0.0f, 0.0f);
        p.at0 = p.at1 = false;
        float h = 0.0f;
        uint32_t seg = 0, nrec = 0;
        uint64_t base = 0;
        if (live) {
            const LeafRec r = load_leaf(A.leaves + (A.leaf_cap - 1u - li));
            leaf_piece(P, r, p);
            h = r.h; seg = r.seg;
            const uint32_t n_minus = r.n & 0xffffu;
            nrec = side ? r.n >> 16 : n_minus;
            base = A.seg_off[r.seg] + r.rel + (side ? n_minus : 0u);
            if (base + nrec > A.cap_records) { atomicOr(A.err, kErrCapacity); nrec = 0; }   // the side is not written
            if (side == 0) {
                PieceLite q;
                q.bx = p.base.x; q.by = p.base.y; q.p3x = p.P3.x; q.p3y = p.P3.y;
                q.lax = p.la.x; q.lay = p.la.y; q.lbx = p.lb.x; q.lby = p.lb.y;
                q.uax = p.ua.x; q.uay = p.ua.y; q.ubx = p.ub.x; q.uby = p.ub.y;
                q.k0 = p.k0; q.k1 = p.k1; q.L = p.L;
                q.flags = (p.at0 ? 1u : 0u) | (p.at1 ? 2u : 0u);
                W.piece[lane >> 1] = q;
            }
        }
        const float eta = side ? h : -h;
        uint32_t nparts = 0;
        bool two_ranges = false;
        float tc = 0.0f;
        if (live) {
            SidePlan sp = side_plan(p, eta, P.mode, P.tol_fl);
            if (nrec) nparts = side_part_count(sp);
            two_ranges = sp.nr == 2;
            tc = sp.off[0].tb;
            sp.seg = seg;
            W.plan[lane] = plan_pack(sp);
        }
        {   // anchor table: each lane of a pair integrates one half
            const int K = es_intervals(p.k0, p.k1);
            float hx[kAnchors / 2], hy[kAnchors / 2], tx, ty;
            const int cnt = es_anchor_half<false>(p, K, side, hx, hy, &tx, &ty);
            const float ox = __shfl_xor_sync(kFull, tx, 1), oy = __shfl_xor_sync(kFull, ty, 1);
            if (live) es_anchor_store(W.spiral[lane >> 1], K, side, cnt, hx, hy, tx, ty, ox, oy);
        }
        __syncwarp();
        if (live && two_ranges) {
            const V2 c = normal_point(p, W.spiral[lane >> 1], tc, eta);
            W.cusp[lane] = make_float4(c.x, c.y, tc, 0.0f);
        }
        if (!nparts) nrec = 0;
        // ---- table + write, in one pass, or in halves / quarters of the warp's sides when the parts do not fit
        const uint32_t all_parts = __reduce_add_sync(kFull, nparts);
        if (all_parts == 0u) { __syncwarp(); continue; }
        const uint32_t low_parts = __reduce_add_sync(kFull, lane < 16 ? nparts : 0u);
        const int n_pass = all_parts <= (uint32_t)kExParts ? 1 : ((low_parts <= (uint32_t)kExParts && all_parts - low_parts <= (uint32_t)kExParts) ? 2 : 4);
        const int pass_shift = n_pass == 2 ? 4 : 3;
        for (int pass = 0; pass < n_pass; pass++) {
            const bool mine = n_pass == 1 || (lane >> pass_shift) == pass;
            const uint32_t np_ = mine ? nparts : 0u, nr_ = mine ? nrec : 0u;
            uint32_t ip = np_, ir = nr_;
#pragma unroll
            for (int dd = 1; dd < 32; dd <<= 1) {
                const uint32_t a2 = __shfl_up_sync(kFull, ip, dd), b2 = __shfl_up_sync(kFull, ir, dd);
                if (lane >= dd) { ip += a2; ir += b2; }
            }
            const uint32_t tparts = __shfl_sync(kFull, ip, 31), trecs = __shfl_sync(kFull, ir, 31);
            // the part table, lane per PART: the owning side is the last lane whose first part is <= j (binary search by
            // shuffles over the non-decreasing prefix), its plan is in shared memory, the part a closed form of its index
            {
                const uint32_t p_first = ip - np_, r_first = ir - nr_;
                const uint32_t base_lo = (uint32_t)base, base_hi = (uint32_t)(base >> 32);
                for (uint32_t j0 = 0; j0 < tparts; j0 += 32u) {
                    const uint32_t j = j0 + (uint32_t)lane;
                    uint32_t own = 0;
#pragma unroll
                    for (uint32_t step = 16u; step > 0u; step >>= 1) {
                        const uint32_t cand = own + step;
                        const uint32_t pc = __shfl_sync(kFull, p_first, (int)(cand & 31u));
                        if (cand < 32u && pc <= j) own = cand;
                    }
                    const uint32_t o_first = __shfl_sync(kFull, p_first, (int)own), o_np = __shfl_sync(kFull, np_, (int)own), o_rec = __shfl_sync(kFull, r_first, (int)own);
                    const uint64_t o_base = (uint64_t)__shfl_sync(kFull, base_lo, (int)own) | ((uint64_t)__shfl_sync(kFull, base_hi, (int)own) << 32);
                    if (j < tparts) {
                        uint32_t before;
                        W.part[j] = side_part_at(W.plan[own], j - o_first, o_np, own, (own & 1u) != 0u, arc, o_base, &before);
                        W.ppref[j] = o_rec + before;
                    }
                }
            }
            if (lane == 0) W.ppref[tparts] = trecs;
            __syncwarp();
            const uint32_t tverts = trecs - tparts;
            uint32_t v_done = 0;
            for (uint32_t r0 = 0; r0 < trecs; r0 += 32u) {
                const uint32_t r = r0 + (uint32_t)lane;
                const bool act = r < trecs;
                uint32_t lo = 0;
                Part pt;
                pt.base = 0; pt.n = 1; pt.i0 = 0; pt.info = 0;
                uint32_t m = 0;
                if (act) {
                    uint32_t hi = tparts;
#pragma unroll 1
                    while (hi - lo > 1u) {
                        const uint32_t mid = (lo + hi) >> 1;
                        if (W.ppref[mid] <= r) lo = mid; else hi = mid;
                    }
                    pt = W.part[lo];
                    m = r - W.ppref[lo];
                }
                const bool s_int = act && m >= 1u, e_int = act && m + 1u < (uint32_t)pt.n;
                const int v_end = (int)(r - lo);
                const int need = e_int ? v_end : (s_int ? v_end - 1 : -1);
                const int need_max = __reduce_max_sync(kFull, need);
                while ((int)v_done <= need_max) {
                    const uint32_t v = v_done + (uint32_t)lane;
                    if (v < tverts) {
                        uint32_t l2 = 0, h2 = tparts;
#pragma unroll 1
                        while (h2 - l2 > 1u) {
                            const uint32_t mid = (l2 + h2) >> 1;
                            if (W.ppref[mid] - mid <= v) l2 = mid; else h2 = mid;
                        }
                        const Part pj = W.part[l2];
                        const uint32_t mm = v - (W.ppref[l2] - l2) + 1u;
                        const uint32_t ss = pj.info & 127u;
                        Piece pc;
                        piece_of(W.piece[ss >> 1], pc);
                        const PlanLite& sp = W.plan[ss];
                        const int idx = (pj.info & 128u) ? (int)pj.i0 - (int)mm : (int)pj.i0 + (int)mm;
                        const bool evo = ((pj.info >> 8) & 3u) == 2u;
                        const float t = evo ? evolute_t(pc, plan_evo(sp), idx) : offset_t(pc, plan_off(sp, (pj.info & 1024u) != 0u), sp.eta, idx);
                        const V2 g = normal_point(pc, W.spiral[ss >> 1], t, evo ? es_radius(pc, t) : sp.eta);
                        W.ring[v & (uint32_t)(kRing - 1)] = make_float4(g.x, g.y, t, 0.0f);
                    }
                    v_done += 32u;
                    __syncwarp();
                }
                if (act) {
                    const uint32_t ss = pt.info & 127u;
                    Piece pc;
                    piece_of(W.piece[ss >> 1], pc);
                    const PlanLite& sp = W.plan[ss];
                    const float4 cusp = W.cusp[ss];
                    V2 Av, Bv;
                    float tA, tB;
                    if (s_int) { const float4 q = W.ring[(uint32_t)(v_end - 1) & (uint32_t)(kRing - 1)]; Av = v2(q.x, q.y); tA = q.z; }
                    else Av = end_vertex(pc, (pt.info >> 16) & 7u, sp.eta, cusp, &tA);
                    if (e_int) { const float4 q = W.ring[(uint32_t)v_end & (uint32_t)(kRing - 1)]; Bv = v2(q.x, q.y); tB = q.z; }
                    else Bv = end_vertex(pc, (pt.info >> 19) & 7u, sp.eta, cusp, &tB);
                    put_record(out, arc, A.wide != 0u, pt.base + m, Av, Bv, (pt.info & 2048u) ? es_dphi(pc, tA, tB) + 0.0f : 0.0f, sp.seg, (pt.info >> 12) & 15u);
                }
                __syncwarp();
            }
            __syncwarp();
        }
    }
}

// ---------------------------------------------------------------- the walk list: thread per segment
__global__ void __launch_bounds__(kWrThreads)
k_write_walk(const WriteArgs A) {
    const Params& P = A.P;
    const uint32_t n = *A.walk_count;
    for (uint32_t k = blockIdx.x * (uint32_t)kWrThreads + threadIdx.x; k < n; k += gridDim.x * (uint32_t)kWrThreads) {
        const uint32_t i = A.walk_list[k];
        const uint32_t count = A.seg_count[i];
        const uint64_t base = A.seg_off[i];
        if (count == 0u) continue;
        if (base + count > A.cap_records) { atomicOr(A.err, kErrCapacity); continue; }
        Style st;
        float h;
        load_style(P, P.path_idx[i], &st, &h);
        const Seg s = load_segment(P, i, P.tags[i]);
        Writer w;
        w.out = A.out; w.base = base; w.seg = i; w.mode = P.mode; w.wide = A.wide != 0u;
        flatten_cubic<true>(P, s, h, st.fill, &w);
    }
}

}  // namespace sx
