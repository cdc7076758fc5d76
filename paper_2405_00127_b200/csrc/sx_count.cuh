// sx_count.cuh -- (b) k_count: the count pass, and the cubic -> Euler-spiral fit it keeps for the writers.
//
// Every WARP is on its own (one-warp blocks, a persistent grid, no block barrier): it takes a TILE of T = 32, 16 or 8
// consecutive input segments from an atomic ticket and runs, with every intermediate result in its own 12 KB of shared
// memory:
//   A  segments    lane per segment: transform + degree elevation, end tangents (L251), the
//                  number of join / cap records (Alg. 1); straight segments are finished here (2 + tail).
//   B  fit         Alg. 2 (L351-438) NODE-PARALLEL: a warp-wide FIFO of nodes (curve, t0_u, level); every lane
//                  evaluates one node per round -- the accept/split test of a node depends only on its own two end
//                  points and dt = 2^-level, so the accepted set is exactly the one the two-word stack of L444
//                  visits -- a rejected node evaluates its mid point once and pushes its two children, an accepted
//                  node becomes a LEAF (one Euler-spiral piece).  The bisection tree is kept (parent links).  Queue
//                  positions come from warp ballots: no atomics.
//   C  pieces      lane per leaf: end-tangent angles (reading R-17), App. A parameters (L628-653), and per side
//                  the cusp split (L380-386) and the subdivision counts (sections 4, 5, 6).
//   D  counts      subtree sums over the bisection tree give every leaf the number of records that precede it in
//                  its segment (canonical order = increasing t) and every segment its count.
// Output: seg_count[i], seg_tail[i] (join / cap records) and one 32-byte LEAF RECORD per Euler-spiral piece -- segment,
// dyadic parameter range, k0, k1, L, half width, the two sides' counts, the piece's offset within its segment -- so the
// writers never repeat the fit: they rebuild a piece's end points from the segment's control points and the parameter
// range with the same cubic_point() this kernel used, hence the same bits.  Leaves whose two sides are single short
// regular ranges (one thread can write them) are stored from the FRONT of the leaf buffer, all others from the BACK
// (one 64-bit atomic reserves both for a tile): the two kinds have their own writer.
//
// A tile whose nodes, points or leaves do not fit the tables is redone in SUB-TILES of 8 segments, a sub-tile that still
// does not fit is halved (8 -> 4 -> 2 -> 1).  What does not fit even alone, what meets a zero derivative at an interior
// subdivision point (the perturbation rule of L251 then depends on the visiting order), and what finds no room for its
// leaves in the leaf buffer takes the thread-per-segment
// walk of sx_segment.cuh: its curve segments go to the WALK LIST, which the walk writer serves.  Same records, slower.
// The tile size of a call comes from the context's hint word, which the last warp of every launch adapts to the
// scene (pieces per segment seen) for the calls that follow.
#pragma once
#include "sx_scan.cuh"
#include "sx_segment.cuh"

namespace sx {

constexpr int kCtTile = 32;                          // segments per tile at most (a warp: lane per segment)
constexpr int kCtSub = 8;                            // segments per sub-tile of a tile that overflowed (halved again when that overflows)
constexpr int kCtTileMin = 4;                        // the smallest tile of a call
constexpr int kCtSplitCap = 112;                     // splits of Alg. 2 per tile
constexpr int kCtLeafCap = kCtTile + kCtSplitCap;    // Euler-spiral pieces per tile (leaves = curves + splits)
constexpr int kCtPointCap = 2 * kCtTile + kCtSplitCap;   // the end points of every segment + 1 per split
constexpr int kCtTreeCap = kCtTile + 2 * kCtSplitCap;    // roots + 2 per split (<= 256: parent links are bytes)
constexpr int kCtQueueCap = 128;                     // pending nodes (power of two)
constexpr int kLevelMax = 16;                        // dt = 2^-16 = kDtMin: accepted unconditionally
constexpr int kDirectMax = 6;                        // records of a side that one thread writes (the simple writer)
constexpr int kCtWarpsPerSM = 16;
constexpr uint32_t kFull = 0xffffffffu;

enum : uint32_t { kForceWalk = 1u, kForceSub = 2u };   // CountArgs::force (test knob); 4 .. 32 fix the tile size
enum : int { kStDirect = 0, kStSub = 1, kStWalk = 2, kStLeaves = 3, kStSegs = 4, kStDone = 5, kStWords = 8 };

// one Euler-spiral piece as the count pass hands it to the writers
struct __align__(16) LeafRec {
    uint32_t seg;        // input segment
    uint32_t key;        // t0_u (bits 0-15) | level << 16: the piece is C([t0_u, t0_u + 1] * 2^-level)
    uint32_t n;          // records of the -h side | of the +h side << 16
    uint32_t rel;        // records of the segment that precede this piece
    float k0, k1, L, h;  // App. A parameters, arc length; half width of the stroke
};

struct CountArgs {
    Params P;
    uint32_t n_paths;
    uint32_t* ticket;
    uint32_t* err;
    uint32_t* seg_count;            // [n_tags] records of every segment
    uint32_t* seg_tail;             // [n_tags] of which join / cap records
    LeafRec* leaves;                // [leaf_cap]: simple leaves from the front, the others from the back
    uint32_t leaf_cap;
    unsigned long long* leaf_counter;   // others << 32 | simple: what the tiles reserved
    uint32_t* leaf_end_inv;         // [2] ~(end of the valid simple leaves), ~(end of the valid others): set by the first
                                    // reservation that found no room (0 = every reservation fitted)
    uint32_t* walk_list;            // [n_tags] curve segments the walk writer serves
    uint32_t* walk_count;
    uint32_t* stats;                // kSt*
    uint32_t* hint;                 // [0] tile size of this call, [1] tile size the launch proposes for the next call
    uint32_t force;                 // test knob: 0 adaptive; 8, 16, 32 fixed tile size; kForceWalk; kForceSub
};

// position and unit tangent of the cubic at an interior parameter t (0 < t < 1), |q| in *qmag.  The count pass and the
// writers both call this, with the same dyadic t, and so agree bit for bit.
SX_DEV float4 cubic_point(const Seg& s, float t, float* qmag, float* q2_out) {
    const V2 q = cubic_q(s, t);
    const float q2 = len2(q), m = sqrtf(q2);
    const V2 pos = cubic_pos(s, t);
    *qmag = m; *q2_out = q2;
    return make_float4(pos.x, pos.y, q.x / m, q.y / m);
}

// ---------------------------------------------------------------- shared memory of a warp
struct __align__(16) CtSeg {
    float c1x, c1y, c2x, c2y, c3x, c3y;              // control points local to P0
    float tsx, tsy, tex, tey;                        // unit start / end tangents
    float h;
    uint32_t pad;
};
struct CtLeaf {
    uint32_t w;          // bytes: [0] point a, [1] point b (phases B, C1) -> simple flags of the two sides (C1, C2) -> rank within the
                         // class, class (C3, D); [2] segment (tile-local); [3] tree slot
    uint32_t key;
    float k0, k1, L;
    uint16_t n[2];       // n_minus, n_plus
};
struct CtWarp {
    CtSeg seg[kCtTile];
    float4 pts[kCtPointCap];       // x, y local position; z, w unit tangent
    float qmag[kCtPointCap];
    uint32_t qx[kCtQueueCap];      // t0_u | level << 20
    uint32_t qy[kCtQueueCap];      // bytes: point a, point b, segment (tile-local), tree slot
    uint32_t acc[kCtTreeCap];
    uint8_t parent[kCtTreeCap];
    CtLeaf leaf[kCtLeafCap];
};

SX_DEV Seg seg_of(const CtSeg& r) {
    Seg s;
    s.kind = 3; s.degenerate = false;
    s.P0 = v2(0.0f, 0.0f); s.P3 = v2(0.0f, 0.0f);
    s.c1 = v2(r.c1x, r.c1y); s.c2 = v2(r.c2x, r.c2y); s.c3 = v2(r.c3x, r.c3y);
    s.ts = v2(r.tsx, r.tsy); s.te = v2(r.tex, r.tey);
    return s;
}

// number of join / cap records that follow the offset curves of segment i (Alg. 1); the partner's start tangent
// comes from the tile when the partner is in it
SX_DEV uint32_t count_tail(const CtWarp& S, const Params& P, uint32_t s0, uint32_t sn, uint32_t i, uint32_t tag, V2 te, const Style& st, float h,
                           uint32_t first_seg) {
    const bool sp_end = ((tag >> 2) | (tag >> 4)) & 1u;
    const bool closed = (tag >> 7) & 1u;
    if (st.fill) return (sp_end && !closed) ? 1u : 0u;   // a filled path: the closing line of an open subpath (Alg. 1)
    const uint32_t j = (!sp_end) ? i + 1u : first_seg;   // join partner, or the owner of the start cap
    V2 W, T1;
    if (j >= s0 && j - s0 < sn) { const CtSeg& r = S.seg[j - s0]; T1 = v2(r.tsx, r.tsy); W = v2(0.0f, 0.0f); }
    else load_segment_start(P, j, &W, &T1);
    const V2 Z = v2(0.0f, 0.0f);
    if (!sp_end || closed) return emit_join<false>(P, st, Z, te, Z, T1, h, nullptr, 0);
    return emit_cap<false>(P, st, Z, te, h, nullptr, 0) + emit_cap<false>(P, st, Z, v2(-T1.x, -T1.y), h, nullptr, 0);
}

// the thread-per-segment walk of a sub-tile that does not fit the tables: out of line (rarely executed, large)
__device__ __noinline__ uint32_t slow_count(const Params& P, uint32_t i, uint32_t* tail) { return process_segment<false>(P, i, nullptr, tail); }

// One leaf of the bisection, straight-line: the end-tangent angles of the accepted piece (L211-213: th0 from the start
// tangent to the chord, th1 from the chord to the end tangent; reading R-17; a zero chord is accepted at the deepest level
// only: th0 = th1 = atan2(0, 1) = 0, as in fit_error), the App. A parameters, and per side either the count of the one
// offset range of a side that is regular throughout -- decided from approximate cusp factors 1 - kappa eta at both ends,
// positive by a wide margin, so that side_plan's own exactly rounded ones have the same signs; the count is offset_plan's,
// the call the writers repeat -- or the request for the full plan.
struct LeafEval { float k0, k1, L; uint32_t n[2]; bool full[2]; };
// (one copy of each: the count pass's working set has to stay inside the instruction cache -- 16 unsynchronised warps per SM)
__device__ __noinline__ float atan2_r_core_call(float y, float x) { return atan2_r_core(y, x); }
SX_DEV uint32_t offset_count(float k0, float k1, float L, float eta, int mode, float tol_fl) {
    return (uint32_t)offset_plan_call(k0, k1, L, eta, 0.0f, 1.0f, mode, tol_fl).n;
}
SX_DEV LeafEval leaf_eval(float4 pa, float4 pb, float h, int mode, float tol_fl) {
    LeafEval e;
    const V2 ch = v2(pb.x, pb.y) - v2(pa.x, pa.y);
    const float chord2 = len2(ch), chord = sqrtf(chord2);
    const V2 uc = v2(ch.x / chord, ch.y / chord);
    const bool flat = !(chord2 >= kEpsQ2);
    float th[2];
#pragma unroll 1
    for (int k = 0; k < 2; k++) {
        const V2 f0 = k ? uc : v2(pa.z, pa.w), f1 = k ? v2(pb.z, pb.w) : uc;
        th[k] = atan2_r_core_call(flat ? 0.0f : cross(f0, f1), flat ? 1.0f : dot(f0, f1));
    }
    Piece p;
    piece_params(p, th[0], th[1], chord);
    e.k0 = p.k0; e.k1 = p.k1; e.L = p.L;
    const float il = rcp_fast(p.L), ka = (p.k0 - 0.5f * p.k1) * il, kb = (p.k0 + 0.5f * p.k1) * il;
    // (arc mode: the count of a regular side does not depend on the sign of eta -- "same arc approximation ... both sides", L181)
    const uint32_t n_arc = mode == kModeArc ? offset_count(p.k0, p.k1, p.L, h, kModeArc, tol_fl) : 0u;
#pragma unroll 1
    for (int side = 0; side < 2; side++) {
        const float eta = side ? h : -h;
        e.full[side] = !(fmaf(-ka, eta, 1.0f) > 1e-3f && fmaf(-kb, eta, 1.0f) > 1e-3f);
        e.n[side] = n_arc;
        if (mode != kModeArc && !e.full[side]) e.n[side] = offset_count(p.k0, p.k1, p.L, eta, mode, tol_fl);
        if (e.full[side]) e.n[side] = 0xffffu;   // (not simple until the full plan says so)
    }
    if (h == 0.0f) { e.n[1] = 0u; e.full[1] = false; }   // a filled path (Alg. 1): offset 0, the curve once
    return e;
}

// ---------------------------------------------------------------- the kernel
__global__ void __launch_bounds__(32, kCtWarpsPerSM)
k_count(const CountArgs A) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    CtWarp& S = *reinterpret_cast<CtWarp*>(smem_raw);
    const Params& P = A.P;
    const int lane = threadIdx.x & 31;
    const uint32_t lt = (1u << lane) - 1u;
    const bool ok = (*A.err & kErrBadStream) == 0u;   // a malformed stream silences every segment
    uint32_t T = A.force >= (uint32_t)kCtTileMin ? A.force : *reinterpret_cast<volatile uint32_t*>(A.hint);
    T = T >= 32u ? 32u : (T >= (uint32_t)kCtTileMin ? T : (uint32_t)kCtTileMin);   // any size from kCtTileMin to a warp's 32 lanes
    uint32_t st_direct = 0, st_sub = 0, st_walk = 0, st_leaves = 0, st_segs = 0;

    for (;;) {
        uint32_t tile = 0;
        if (lane == 0) tile = atomicAdd(A.ticket, 1u);
        tile = __shfl_sync(kFull, tile, 0);
        if ((uint64_t)tile * T >= (uint64_t)P.n_tags) break;
        const uint32_t tile0 = tile * T, tile_n = min(T, P.n_tags - tile0), tile_end = tile0 + tile_n;
        uint32_t s0 = tile0, sn = tile_n;
        bool sub = false;   // the tile is being redone in sub-tiles
        uint32_t sub_size = (uint32_t)kCtSub;
        if (A.force == kForceSub && tile_n > (uint32_t)kCtSub) { sub = true; sn = (uint32_t)kCtSub; st_sub++; }

        for (;;) {
            __syncwarp();
            // ================================================================ A: segments
            uint32_t my_tag = 0, my_first = 0, my_path = 0, my_tail = 0;
            bool my_valid = false, my_curve = false;
            if (lane < (int)sn) {
                const uint32_t i = s0 + (uint32_t)lane;
                my_tag = P.tags[i];
                my_path = P.path_idx[i];
                my_first = P.sp_first[i];
                const uint32_t pt = P.pt_off[i];
                Style st;
                float h;
                my_valid = load_style(P, my_path, &st, &h) && ok;
                const Seg s = load_segment_at(P, pt, my_tag);
                my_curve = my_valid && s.kind != 1 && !s.degenerate;
                CtSeg r;
                r.c1x = s.c1.x; r.c1y = s.c1.y; r.c2x = s.c2.x; r.c2y = s.c2.y; r.c3x = s.c3.x; r.c3y = s.c3.y;
                r.tsx = s.ts.x; r.tsy = s.ts.y; r.tex = s.te.x; r.tey = s.te.y;
                r.h = h; r.pad = 0;
                S.seg[lane] = r;
                // the two end points of a curve are points 2 lane and 2 lane + 1 of the table; its root node is tree slot lane
                if (my_curve) {
                    float qm;
                    V2 pos, u;
                    S.pts[2 * lane] = make_float4(0.0f, 0.0f, s.ts.x, s.ts.y);
                    S.qmag[2 * lane] = sqrtf(len2(s.c1));
                    eval_cubic(s, 1.0f, 1.0f, &pos, &qm, &u);
                    S.pts[2 * lane + 1] = make_float4(pos.x, pos.y, u.x, u.y);
                    S.qmag[2 * lane + 1] = qm;
                }
                S.acc[lane] = 0u;
            }
            // roots into the queue, in segment order
            const uint32_t root_mask = __ballot_sync(kFull, my_curve);
            const uint32_t n_roots = __popc(root_mask);
            if (my_curve) {
                const uint32_t q = __popc(root_mask & lt);
                S.qx[q] = 0u;
                S.qy[q] = (uint32_t)(2 * lane) | ((uint32_t)(2 * lane + 1) << 8) | ((uint32_t)lane << 16) | ((uint32_t)lane << 24);
            }
            __syncwarp();
            // join / cap record counts (partners from the tile's records)
            if (lane < (int)sn && my_valid) {
                const CtSeg& r = S.seg[lane];
                Style st;
                float h;
                load_style(P, my_path, &st, &h);
                my_tail = count_tail(S, P, s0, sn, s0 + (uint32_t)lane, my_tag, v2(r.tex, r.tey), st, h, my_first);
            }

            // ================================================================ B: Alg. 2, node-parallel
            uint32_t q_head = 0, q_tail = n_roots, n_leaf = 0, n_split = 0;
            bool overflow = A.force == kForceWalk;
            while (q_head != q_tail && !overflow) {
                const uint32_t n_round = min(q_tail - q_head, 32u);
                bool accept = false, push = false, bad = false;
                uint32_t qx = 0, qy = 0;
                float4 mid = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                float mid_q = 0.0f;
                if ((uint32_t)lane < n_round) {
                    const uint32_t qi = (q_head + (uint32_t)lane) & (uint32_t)(kCtQueueCap - 1);
                    qx = S.qx[qi]; qy = S.qy[qi];
                    const uint32_t t0_u = qx & 0xfffffu, level = qx >> 20;
                    const uint32_t pa_i = qy & 0xffu, pb_i = (qy >> 8) & 0xffu;
                    const float4 a = S.pts[pa_i], b = S.pts[pb_i];
                    const float dt = __uint_as_float((127u - level) << 23);
                    const float err = node_error(v2(a.z, a.w), v2(b.z, b.w), S.qmag[pa_i], S.qmag[pb_i], v2(b.x, b.y) - v2(a.x, a.y), dt);
                    if (err <= P.tol_es || level >= (uint32_t)kLevelMax) {
                        accept = true;
                    } else {
                        // split: the mid point is evaluated once, for both children (Alg. 2 L369 with the rule of L251)
                        push = true;
                        float q2;
                        mid = cubic_point(seg_of(S.seg[(qy >> 16) & 0xffu]), (float)t0_u * dt + 0.5f * dt, &mid_q, &q2);
                        bad = q2 < kEpsQ2;   // zero derivative inside the curve: the visiting order matters (L251)
                    }
                }
                const uint32_t m_acc = __ballot_sync(kFull, accept), m_push = __ballot_sync(kFull, push);
                const uint32_t n_acc = __popc(m_acc), n_push = __popc(m_push);
                // the tables, and the ring from this round's first entry to the new tail, must hold everything
                if (__any_sync(kFull, bad) || n_leaf + n_acc > (uint32_t)kCtLeafCap || n_split + n_push > (uint32_t)kCtSplitCap ||
                    q_tail + 2u * n_push - q_head > (uint32_t)kCtQueueCap) { overflow = true; break; }
                if (accept) {
                    CtLeaf& lf = S.leaf[n_leaf + __popc(m_acc & lt)];
                    lf.w = qy; lf.key = (qx & 0xffffu) | ((qx >> 20) << 16);
                }
                if (push) {
                    // children: one point, two tree slots, two queue entries per split
                    const uint32_t rank = __popc(m_push & lt);
                    const uint32_t k = n_split + rank;
                    const uint32_t pm = 2u * (uint32_t)kCtTile + k, ts = (uint32_t)kCtTile + 2u * k;
                    const uint32_t slot = qy >> 24;
                    S.pts[pm] = mid;
                    S.qmag[pm] = mid_q;
                    S.parent[ts] = (uint8_t)slot; S.parent[ts + 1u] = (uint8_t)slot;
                    S.acc[ts] = 0u; S.acc[ts + 1u] = 0u;
                    const uint32_t q = (q_tail + 2u * rank) & (uint32_t)(kCtQueueCap - 1), q1 = (q + 1u) & (uint32_t)(kCtQueueCap - 1);
                    const uint32_t t0_u = qx & 0xfffffu, lv = ((qx >> 20) + 1u) << 20;
                    S.qx[q] = (2u * t0_u) | lv;       S.qy[q] = (qy & 0x00ff00ffu) | (pm << 8) | (ts << 24);
                    S.qx[q1] = (2u * t0_u + 1u) | lv; S.qy[q1] = (qy & 0x00ffff00u) | pm | ((ts + 1u) << 24);
                }
                q_head += n_round; q_tail += 2u * n_push; n_leaf += n_acc; n_split += n_push;
                __syncwarp();
            }
            __syncwarp();

            // ================================================================ C: pieces (lane per leaf)
            uint32_t n_triv = 0, n_multi = 0, n_other = 0;
            if (!overflow) {
                // C1, lane per leaf: angles, App. A parameters, and the counts of the sides that are regular throughout by a wide
                // margin (the usual case)
                uint16_t* const full_list = reinterpret_cast<uint16_t*>(S.qx);   // (the queue is dead: qx, qy = 512 entries)
                uint32_t n_full = 0;
                for (uint32_t l0 = 0; l0 < n_leaf; l0 += 32u) {
                    const uint32_t li = l0 + (uint32_t)lane;
                    const bool live = li < n_leaf;
                    const uint32_t lw = live ? S.leaf[li].w : 0u;
                    const LeafEval ev = leaf_eval(S.pts[lw & 0xffu], S.pts[(lw >> 8) & 0xffu], S.seg[(lw >> 16) & 0xffu].h, P.mode, P.tol_fl);
                    const bool f0 = live && ev.full[0], f1 = live && ev.full[1];
                    const uint32_t m0 = __ballot_sync(kFull, f0), m1 = __ballot_sync(kFull, f1);
                    if (live) {
                        CtLeaf& lf = S.leaf[li];
                        lf.k0 = ev.k0; lf.k1 = ev.k1; lf.L = ev.L;
                        lf.n[0] = (uint16_t)ev.n[0]; lf.n[1] = (uint16_t)ev.n[1];
                        lf.w = (lw & 0xffff0000u) | (ev.n[0] <= (uint32_t)kDirectMax ? 1u : 0u) | (ev.n[1] <= (uint32_t)kDirectMax ? 0x100u : 0u);   // simple flags of the two sides (bytes 0, 1)
                    }
                    if (f0) full_list[n_full + __popc(m0 & lt)] = (uint16_t)(2u * li);
                    n_full += __popc(m0);
                    if (f1) full_list[n_full + __popc(m1 & lt)] = (uint16_t)(2u * li + 1u);
                    n_full += __popc(m1);
                }
                __syncwarp();
                // C2, lane per side that has a cusp or a super-critical range: the full plan (cusp split L380-386, evolute L195)
                bool too_long = false;
                for (uint32_t e0 = 0; e0 < n_full; e0 += 32u) {
                    if (e0 + (uint32_t)lane < n_full) {
                        const uint32_t e = full_list[e0 + (uint32_t)lane], l = e >> 1, side = e & 1u;
                        CtLeaf& lf = S.leaf[l];
                        Piece p;
                        p.k0 = lf.k0; p.k1 = lf.k1; p.L = lf.L;
                        const float h = S.seg[(lf.w >> 16) & 0xffu].h;
                        const SidePlan sp = side_plan(p, side ? h : -h, P.mode, P.tol_fl);
                        too_long |= (uint32_t)sp.total > 0xffffu;   // a side of more than 65535 records: the walk
                        lf.n[side] = (uint16_t)sp.total;
                        reinterpret_cast<uint8_t*>(&lf.w)[side] = (sp.nr == 1 && !sp.sup[0] && sp.total <= kDirectMax) ? 1 : 0;
                    }
                }
                __syncwarp();
                if (__any_sync(kFull, too_long)) overflow = true;
                // C3, lane per leaf: class, rank within the class, subtree sums
                for (uint32_t l0 = 0; l0 < n_leaf; l0 += 32u) {
                    const uint32_t l = l0 + (uint32_t)lane;
                    const bool live = l < n_leaf;
                    uint32_t n = 0, no = 0, fl = 0, slot = 0;
                    if (live) { const CtLeaf& lf = S.leaf[l]; n = lf.n[0]; no = lf.n[1]; fl = lf.w; slot = fl >> 24; }
                    // classes: 1 both sides one record (the simple writer's straight path), 2 both sides simple, 0 the others
                    const bool both = live && (fl & 0x101u) == 0x101u;
                    const bool triv = both && n == 1u && no == 1u;
                    const uint32_t m_triv = __ballot_sync(kFull, triv), m_multi = __ballot_sync(kFull, both && !triv), m_other = __ballot_sync(kFull, live && !both);
                    if (live) {
                        S.leaf[l].w = (fl & 0xffff0000u) | (triv ? ((n_triv + __popc(m_triv & lt)) | 0x100u) : (both ? ((n_multi + __popc(m_multi & lt)) | 0x200u) : (n_other + __popc(m_other & lt))));
                        // subtree sums: the leaf's records are added to itself and to all its ancestors
                        const uint32_t c = n + no;
                        uint32_t cur = slot;
                        for (;;) {
                            atomicAdd(&S.acc[cur], c);
                            if (cur < (uint32_t)kCtTile) break;
                            cur = S.parent[cur];
                        }
                    }
                    n_triv += __popc(m_triv); n_multi += __popc(m_multi); n_other += __popc(m_other);
                }
            }
            __syncwarp();
            if (overflow && !sub && sn > (uint32_t)kCtSub) {   // redo the tile in sub-tiles
                sub = true; s0 = tile0; sn = (uint32_t)kCtSub; st_sub++;
                continue;
            }
            if (overflow && sn > 1u && A.force != kForceWalk) {   // a (sub-)tile that still does not fit: halve it, down to one segment
                if (!sub) { sub = true; st_sub++; }
                sub_size = sn >> 1;
                sn = sub_size;
                continue;
            }

            // ================================================================ D: counts, leaf records
            bool walk = overflow;
            const uint32_t n_simple = n_triv + n_multi;
            if (!walk && n_leaf) {
                // room in the leaf buffer for the (sub-)tile: one atomic for both ends
                unsigned long long got = 0;
                if (lane == 0) got = atomicAdd(A.leaf_counter, ((unsigned long long)n_other << 32) | (unsigned long long)n_simple);
                got = __shfl_sync(kFull, got, 0);
                const uint32_t base_simple = (uint32_t)(got & 0xffffffffull), base_other = (uint32_t)(got >> 32);
                if ((unsigned long long)base_simple + n_simple + (unsigned long long)base_other + n_other > (unsigned long long)A.leaf_cap) {
                    // (the reservation stays: the counter keeps telling how much room the scene needs; reservations are
                    // totally ordered and both ends only grow, so every later one fails too: the valid leaves are a prefix)
                    walk = true;
                    if (lane == 0) { atomicMax(A.leaf_end_inv, ~base_simple); atomicMax(A.leaf_end_inv + 1, ~base_other); }
                } else {
                    for (uint32_t li = (uint32_t)lane; li < n_leaf; li += 32u) {
                        const CtLeaf lf = S.leaf[li];
                        // records that precede the leaf in its segment: over the path to the root, the left siblings' subtree sums
                        uint32_t cur = lf.w >> 24, rel = 0;
                        while (cur >= (uint32_t)kCtTile) {
                            if ((cur - (uint32_t)kCtTile) & 1u) rel += S.acc[cur - 1u];
                            cur = S.parent[cur];
                        }
                        const uint32_t sl = (lf.w >> 16) & 0xffu;
                        LeafRec r;
                        r.seg = s0 + sl; r.key = lf.key; r.n = (uint32_t)lf.n[0] | ((uint32_t)lf.n[1] << 16); r.rel = rel;
                        r.k0 = lf.k0; r.k1 = lf.k1; r.L = lf.L; r.h = S.seg[sl].h;
                        // the tile's simple leaves: the one-record ones from the front of its block, the others from its back,
                        // so that the warps of the simple writer see (mostly) one kind
                        const uint32_t rank = lf.w & 0xffu, cls = (lf.w >> 8) & 0xffu;
                        const uint32_t pos = cls == 1u ? base_simple + rank : (cls == 2u ? base_simple + n_simple - 1u - rank : A.leaf_cap - 1u - (base_other + rank));
                        // (one 256-bit store: a full 32-byte sector; the leaf buffer is the context's own, aligned allocation)
                        asm volatile("st.global.v8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(A.leaves + pos), "r"(r.seg), "r"(r.key), "r"(r.n), "r"(r.rel),
                                     "r"(__float_as_uint(r.k0)), "r"(__float_as_uint(r.k1)), "r"(__float_as_uint(r.L)), "r"(__float_as_uint(r.h))
                                     : "memory");
                    }
                }
            }
            if (lane < (int)sn) {
                const uint32_t i = s0 + (uint32_t)lane;
                uint32_t count = 0, tail = my_tail;
                if (!overflow) { if (my_valid) count = (my_curve ? S.acc[lane] : (S.seg[lane].h == 0.0f ? 1u : 2u)) + my_tail; }   // (h == 0: a fill)
                else if (ok) count = slow_count(P, i, &tail);
                A.seg_count[i] = count;
                A.seg_tail[i] = tail;
            }
            if (walk) {   // the curve segments of the (sub-)tile go to the walk writer
                const uint32_t m = __ballot_sync(kFull, my_curve);
                if (m) {
                    uint32_t base = 0;
                    if (lane == 0) base = atomicAdd(A.walk_count, (uint32_t)__popc(m));
                    base = __shfl_sync(kFull, base, 0);
                    if (my_curve) A.walk_list[base + __popc(m & lt)] = s0 + (uint32_t)lane;
                }
                st_walk += sn;
            } else {
                st_leaves += n_leaf;
            }
            if (!sub) { st_direct++; break; }
            s0 += sn;
            if (s0 >= tile_end) break;
            sn = min(sub_size, tile_end - s0);
        }
        st_segs += tile_n;
    }

    // ---- statistics; the last warp adapts the tile size for the calls that follow: the largest tile whose expected
    // number of pieces stays below 65 % of the table (pieces per segment as seen by this launch)
    if (lane == 0) {
        if (st_direct) atomicAdd(A.stats + kStDirect, st_direct);
        if (st_sub) atomicAdd(A.stats + kStSub, st_sub);
        if (st_walk) atomicAdd(A.stats + kStWalk, st_walk);
        if (st_leaves) atomicAdd(A.stats + kStLeaves, st_leaves);
        if (st_segs) atomicAdd(A.stats + kStSegs, st_segs);
        __threadfence();
        if (atomicAdd(A.stats + kStDone, 1u) == gridDim.x - 1u) {
            __threadfence();
            const uint32_t leaves = *reinterpret_cast<volatile uint32_t*>(A.stats + kStLeaves);
            const uint32_t segs = *reinterpret_cast<volatile uint32_t*>(A.stats + kStSegs);
            const uint32_t walked = *reinterpret_cast<volatile uint32_t*>(A.stats + kStWalk);
            if (segs >= 256u) {   // (a handful of segments says nothing about the scene)
                const float per_seg = (float)leaves / (float)max(segs - walked, 1u);
                const float room = 0.65f * (float)kCtLeafCap, room12 = 0.72f * (float)kCtLeafCap;   // (12: config 5, 8.5 pieces per segment, count pass - 17 % against 8)
                uint32_t next = per_seg * 32.0f <= room ? 32u : (per_seg * 16.0f <= room ? 16u : (per_seg * 12.0f <= room12 ? 12u : (per_seg * 8.0f <= room ? 8u : (uint32_t)kCtTileMin)));
                if (walked * 4u >= segs) next = (uint32_t)kCtTileMin;   // a launch that mostly walked: its pieces were not counted
                A.hint[1] = next;
            }
        }
    }
}

}  // namespace sx
