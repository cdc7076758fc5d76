// sx_expand.cuh -- k_expand: count (b), allocation scan (c) and write (d) of the stroke-expansion path in ONE pass.
//
// A block takes a TILE of kExTile consecutive input segments (tile ids from an atomic ticket) and runs, with every
// intermediate result in shared memory:
//   A  segments    thread per segment: transform + degree elevation, end tangents (L251), the
//                  number of join / cap records (Alg. 1); straight segments are finished here (2 + tail).
//   B  fit         Alg. 2 (L351-438) NODE-PARALLEL: a block-wide FIFO of nodes (curve, t0_u, level); every thread
//                  evaluates one node per round -- the accept/split test of a node depends only on its own two end
//                  points and dt = 2^-level, so the accepted set is exactly the one the two-word stack of L444
//                  visits -- a rejected node evaluates its mid point once and pushes its two children, an accepted
//                  node becomes a LEAF (one Euler-spiral piece).  The bisection tree is kept (parent links).
//   C  pieces      lane pair per leaf: end-tangent angles (reading R-17), App. A parameters (L628-653), and per side
//                  the cusp split (L380-386) and the subdivision counts (sections 4, 5, 6).
//   D  allocation  subtree sums over the bisection tree give every leaf the number of records that precede it in
//                  its segment (canonical order = increasing t); a block scan over the segments' counts and a
//                  decoupled look-back over the tiles' totals (replaces the atomic bump allocation of L448) give
//                  every segment, and every path, its offset in the output.
//   E  write       (WRITE only) thread per segment: the exact offset lines of straight segments, joins, caps;
//                  thread per output record for the pieces: per warp, tiles of 16 leaves are staged (side plans,
//                  spiral anchors, part tables: sx_cache.cuh) and written 32 records at a time.
// Nothing between the input streams and the output records touches HBM except the look-back words (and, when the
// caller asks for them, the per-segment counts / offsets).  WRITE = false is the count-only pass behind sx_count.
//
// A tile whose nodes, points or leaves do not fit the shared-memory tables, or that meets a zero derivative at an
// interior subdivision point (the perturbation rule of L251 then depends on the visiting order), takes the
// thread-per-segment walk of sx_segment.cuh instead (count, look-back, write): same records, slower.
#pragma once
#include "sx_scan.cuh"
#include "sx_cache.cuh"

namespace sx {

constexpr int kExThreads = 256;
constexpr int kExWarps = kExThreads / 32;
constexpr int kExRange = 128;                        // segments per block
constexpr int kExSlot = 32;                          // segments per look-back word; a block works on its range as 1, 2 or 4 tiles
constexpr int kExSlotsPerRange = kExRange / kExSlot;
constexpr int kExSplitCap = 1024;                    // splits of Alg. 2 per tile
constexpr int kExLeafCap = kExRange + kExSplitCap;   // Euler-spiral pieces per tile (leaves = curves + splits)
constexpr int kExPointCap = 2 * kExRange + kExSplitCap;  // the end points of every segment + 1 per split
constexpr int kExTreeCap = kExRange + 2 * kExSplitCap;   // roots + 2 per split
constexpr int kExQueueCap = 1024;                    // pending nodes (power of two)
constexpr int kExLevelMax = 16;                      // dt = 2^-16 = kDtMin: accepted unconditionally
constexpr int kExDirectMax = 6;                      // records of a side its own staging lane writes
constexpr int kExParts = 64;                         // part table of a warp's stage (8 sides x 8 parts always fit)
constexpr int kRing = 64;                            // interior vertices kept ahead of the records (>= 2 x 32)

struct ExArgs {
    Params P;
    uint32_t n_paths;
    uint64_t* states;          // look-back words of the tiles: status (2 bits) | inclusive or aggregate count
    uint32_t* ticket;
    uint32_t* err;
    uint64_t* path_off;        // [n_paths + 1]
    uint64_t* d_total;
    uint32_t* seg_count;       // optional (nullptr: not kept)
    uint64_t* seg_off;         // optional
    float4* out;
    uint64_t cap_records;
    uint32_t* stats;           // [0] tiles on the fast path, [1] tiles on the thread-per-segment walk
    uint32_t* hint;            // tiles per range (1, 2, 4) the blocks start with; adapted on the device, kept across calls
    uint32_t force_tiles;      // test knob: 0 = adaptive; 1, 2, 4 = fixed; 8 = every tile takes the thread-per-segment walk
};

// ---------------------------------------------------------------- shared memory of a block
struct __align__(16) SegRec {
    float p0x, p0y, c1x, c1y, c2x, c2y, c3x, c3y;    // P0 global; control points local to P0
    float tsx, tsy, tex, tey;                        // unit start / end tangents
    float p3x, p3y;                                  // P3 global (the canonical end vertex, shared with the join)
    float h;
    uint32_t info;                                   // bit 0 valid (width > 0), 1 curve (goes through Alg. 2), 8-15 tag
    uint32_t n_tail;                                 // records of the join / caps
    uint32_t off;                                    // phase D: offset of the segment's first record within the tile
    uint32_t pad[2];
};
struct Leaf {
    uint32_t ab;         // point indices a | b << 16
    uint32_t seg_slot;   // segment (tile-local) | tree slot << 8   (phase B-D);  segment | flags << 8 (phase E)
    float k0, k1, L;
    uint32_t n;          // n_minus | n_plus << 16
    uint32_t rel;        // records of the segment that precede this piece
};
constexpr uint32_t kLeafSimpleMinus = 1u << 8, kLeafSimplePlus = 1u << 9;

struct WarpStage {
    float4 cusp[32];
    float4 ring[kRing];
    Part part[kExParts];
    Spiral spiral[16];
    PlanLite plan[32];
    uint32_t ppref[kExParts + 1];
    uint32_t leaf[16];
    uint32_t pad[3];
};
struct FitArea {
    uint4 queue[kExQueueCap];      // x: t0_u | level << 20, y: a | b << 16, z: seg | slot << 8
    float qmag[kExPointCap];
    uint32_t acc[kExTreeCap];
    uint16_t parent[kExTreeCap];
};
union ExUnion {
    FitArea fit;
    WarpStage stage[kExWarps];
};
struct ExShared {
    SegRec seg[kExRange];
    float4 pts[kExPointCap];       // x, y local position; z, w unit tangent
    ExUnion u;
    Leaf leaf[kExLeafCap];
    uint16_t order[kExLeafCap];    // leaf indices: both sides simple from the front, the others from the back
    uint64_t tile_base;
    uint32_t warp_sum[kExWarps];
    uint32_t range, q_head, q_tail, n_leaf, overflow, n_simple, n_complex, chunk, n_tiles, fill_max;
};

// ---------------------------------------------------------------- helpers on the tile
SX_DEV Seg seg_of(const SegRec& r) {
    Seg s;
    s.kind = 3; s.degenerate = false;
    s.P0 = v2(r.p0x, r.p0y);
    s.c1 = v2(r.c1x, r.c1y); s.c2 = v2(r.c2x, r.c2y); s.c3 = v2(r.c3x, r.c3y);
    s.P3 = v2(0.0f, 0.0f);
    s.ts = v2(r.tsx, r.tsy); s.te = v2(r.tex, r.tey);
    return s;
}

// the piece of a leaf: end points and tangents from the point table, the segment's base and end point from the
// segment record (the end point of the segment is P0 + c3 only up to rounding: at1 pieces use the stored point)
SX_DEV void leaf_piece(const ExShared& S, uint32_t tile0, const Leaf& lf, Piece& p, float* h, uint32_t* seg_global) {
    const uint32_t a = lf.ab & 0xffffu, b = lf.ab >> 16, sl = lf.seg_slot & 0xffu;
    const SegRec& r = S.seg[sl];
    const float4 pa = S.pts[a], pb = S.pts[b];
    p.base = v2(r.p0x, r.p0y);
    p.la = v2(pa.x, pa.y); p.lb = v2(pb.x, pb.y);
    p.ua = v2(pa.z, pa.w); p.ub = v2(pb.z, pb.w);
    p.ch = p.lb - p.la;
    p.k0 = lf.k0; p.k1 = lf.k1; p.L = lf.L;
    p.at0 = a == 2u * sl; p.at1 = b == 2u * sl + 1u;
    p.P3 = v2(r.p3x, r.p3y);
    *h = r.h;
    *seg_global = tile0 + sl;
}

// start point and start tangent of segment j (join partner / start-cap owner): from the tile when j is in it
SX_DEV void partner_start(const ExShared& S, const Params& P, uint32_t tile0, uint32_t n_in_tile, uint32_t j, V2* W, V2* T1) {
    if (j >= tile0 && j - tile0 < n_in_tile) {
        const SegRec& r = S.seg[j - tile0];
        *W = v2(r.p0x, r.p0y); *T1 = v2(r.tsx, r.tsy);
    } else {
        load_segment_start(P, j, W, T1);
    }
}

template <bool EMIT>
SX_DEV uint32_t tile_segment_tail(const ExShared& S, const Params& P, uint32_t tile0, uint32_t n_in_tile, uint32_t i, uint32_t tag, V2 P3, V2 te,
                                  const Style& st, float h, uint32_t first_seg, const Writer* w, uint32_t first) {
    const bool sp_end = ((tag >> 2) | (tag >> 4)) & 1u;
    const bool closed = (tag >> 7) & 1u;
    uint32_t n = 0;
    V2 W, T1;
    if (!sp_end || closed) {
        partner_start(S, P, tile0, n_in_tile, sp_end ? first_seg : i + 1u, &W, &T1);
        n += emit_join<EMIT>(P, st, P3, te, W, T1, h, w, first);
    } else {
        partner_start(S, P, tile0, n_in_tile, first_seg, &W, &T1);
        n += emit_cap<EMIT>(P, st, P3, te, h, w, first);
        n += emit_cap<EMIT>(P, st, W, v2(-T1.x, -T1.y), h, w, first + n);
    }
    return n;
}

// the thread-per-segment walk of a tile that does not fit the tables: out of line (rarely executed, large)
__device__ __noinline__ uint32_t slow_count(const Params& P, uint32_t i) { return process_segment<false>(P, i, nullptr); }
__device__ __noinline__ void slow_write(const Params& P, uint32_t i, Writer* w) { process_segment<true>(P, i, w); }

// block-wide exclusive scan of one value per thread (kExThreads threads); returns the exclusive prefix, *total the sum
SX_DEV uint32_t block_exclusive_scan(uint32_t v, uint32_t* warp_sum, uint32_t* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t o = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += o;
    }
    __syncthreads();
    if (lane == 31) warp_sum[warp] = incl;
    __syncthreads();
    uint32_t base = 0, tot = 0;
#pragma unroll
    for (int k = 0; k < kExWarps; k++) {
        if (k == warp) base = tot;
        tot += warp_sum[k];
    }
    *total = tot;
    return base + incl - v;
}

// Publishes the total of a tile in the look-back words and returns the number of records before the tile (called
// by warp 0).  A tile covers n_slots consecutive words (a block works on its range as 1, 2 or 4 tiles; the words have
// the granularity of the smallest tile): the first carries the tile's value, the others zero.  The block's first
// tile looks back over its predecessors (same protocol as k_alloc_scan: aggregate first, inclusive prefix after);
// its later tiles know their prefix and publish the inclusive value at once.
SX_DEV uint64_t tile_publish(uint64_t* states, uint32_t slot0, uint32_t n_slots, bool look_back, uint64_t known_prefix, uint64_t tile_agg) {
    const int lane = threadIdx.x & 31;
    uint64_t excl = known_prefix;
    if (look_back) {
        if ((uint32_t)lane < n_slots && slot0 > 0u)
            *reinterpret_cast<volatile uint64_t*>(states + slot0 + lane) = (1ull << 62) | (lane == 0 ? tile_agg : 0ull);
        excl = 0;
        int idx = (int)slot0 - 1;
        while (idx >= 0) {
            const int j = idx - lane;
            uint64_t word = 2ull << 62;
            if (j >= 0) { do { word = ld_volatile_u64(states + j); } while ((word >> 62) == 0ull); }
            const uint32_t m = __ballot_sync(0xffffffffu, (word >> 62) == 2ull);
            const int stop = __ffs((int)m) - 1;
            uint64_t v = (lane > stop && m) ? 0ull : (word & kValMask);
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
            excl += v;
            if (m) break;
            idx -= 32;
        }
    }
    // inclusive prefix: the tile's first word carries it; the tile's other words repeat it (a successor stops at the
    // first inclusive word it meets, scanning backwards)
    if ((uint32_t)lane < n_slots) *reinterpret_cast<volatile uint64_t*>(states + slot0 + lane) = (2ull << 62) | (excl + tile_agg);
    return excl;
}

// ---------------------------------------------------------------- phase E2: the records of the pieces
// Per warp: tiles of 16 leaves (lane = leaf, side), as in the two-pass writer this replaces: stage (side plan,
// anchor halves exchanged by shuffle, cusp vertex), part table by a warp scan, then 32 records per iteration with
// the interior vertices evaluated densely into a ring just ahead of the records.  Sides that are one short regular
// range are written by their own lane when (nearly) the whole warp is like that (the order[] list puts such leaves
// together).
template <int DUMMY = 0>
__device__ __noinline__ void write_pieces(ExShared& S, const ExArgs& A, uint32_t tile0, uint64_t tile_base, uint32_t n_leaf, uint32_t n_simple) {
    const Params& P = A.P;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpStage& W = S.u.stage[warp];
    const bool arc = P.mode == kModeArc;
    const int side = lane & 1;
    float4* const out = A.out;
    for (;;) {
        uint32_t chunk = 0;
        if (lane == 0) chunk = atomicAdd(&S.chunk, 1u);
        chunk = __shfl_sync(0xffffffffu, chunk, 0);
        if (chunk * 16u >= n_leaf) break;
        // ---- stage
        const uint32_t li = chunk * 16u + (uint32_t)(lane >> 1);
        const bool live = li < n_leaf;
        Piece p;
        p.k0 = 0.0f; p.k1 = 0.0f; p.L = 1.0f;
        p.la = p.lb = p.ua = p.ub = p.ch = p.base = p.P3 = v2(0.0f, 0.0f);
        p.at0 = p.at1 = false;
        float h = 0.0f;
        uint32_t seg = 0, lidx = 0, lflags = 0, ncnt = 0;
        uint64_t base = 0;
        if (live) {
            lidx = S.order[li < n_simple ? li : (uint32_t)kExLeafCap - 1u - (li - n_simple)];
            const Leaf lf = S.leaf[lidx];
            leaf_piece(S, tile0, lf, p, &h, &seg);
            lflags = lf.seg_slot; ncnt = lf.n;
            const uint32_t sl = lf.seg_slot & 0xffu;
            base = tile_base + S.seg[sl].off + lf.rel + (side ? (lf.n & 0xffffu) : 0u);
            if (side == 0) W.leaf[lane >> 1] = lidx;
        }
        const float eta = side ? h : -h;
        uint32_t nrec = live ? (side ? ncnt >> 16 : ncnt & 0xffffu) : 0u;
        const bool simple = live && (lflags & (side ? kLeafSimplePlus : kLeafSimpleMinus)) && nrec <= (uint32_t)kExDirectMax;
        const bool direct = __popc(__ballot_sync(0xffffffffu, simple || !live)) >= 28 && simple;
        uint32_t nparts = 0;
        bool two_ranges = false;
        float tc = 0.0f;
        // a direct side of one record needs neither plan nor spiral: its two vertices are piece end points
        const bool need_stage = live && !(direct && nrec == 1u);
        if (need_stage) {
            SidePlan sp = side_plan(p, eta, P.mode, P.tol_fl);
            if (!direct) nparts = side_part_count(sp);
            two_ranges = sp.nr == 2;
            tc = sp.off[0].tb;
            sp.seg = seg;
            W.plan[lane] = plan_pack(sp);
        }
        if (__any_sync(0xffffffffu, need_stage)) {   // anchor table: each lane of a pair integrates one half
            const int K = es_intervals(p.k0, p.k1);
            float hx[kAnchors / 2], hy[kAnchors / 2], tx, ty;
            const int cnt = es_anchor_half<false>(p, K, side, hx, hy, &tx, &ty);
            const float ox = __shfl_xor_sync(0xffffffffu, tx, 1), oy = __shfl_xor_sync(0xffffffffu, ty, 1);
            if (live) es_anchor_store(W.spiral[lane >> 1], K, side, cnt, hx, hy, tx, ty, ox, oy);
        }
        __syncwarp();
        if (live && two_ranges && !direct) {
            const V2 c = normal_point(p, W.spiral[lane >> 1], tc, eta);
            W.cusp[lane] = make_float4(c.x, c.y, tc, 0.0f);
        }
        if (direct) {
            const float4 nocusp = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            const uint32_t kind = side ? (uint32_t)(kOffset | kPlus) : (uint32_t)kOffset;
            OffPlan o;
            o.n = (int)nrec; o.rule = kRuleUniform; o.ta = 0.0f; o.tb = 1.0f; o.ua = o.ub = 0.0f;
            if (nrec > 1u) o = plan_off(W.plan[lane], false);
            float tp;
            V2 prev = end_vertex(p, kEndT0, eta, nocusp, &tp);
            for (uint32_t i = 1; i <= nrec; i++) {
                float t;
                V2 cur;
                if (i < nrec) { t = offset_t(p, o, eta, (int)i); cur = normal_point(p, W.spiral[lane >> 1], t, eta); }
                else cur = end_vertex(p, kEndT1, eta, nocusp, &t);
                const uint64_t rec = base + (side ? nrec - i : i - 1u);
                const V2 Av = side ? cur : prev, Bv = side ? prev : cur;
                if (!arc) {
                    out[rec] = make_float4(Av.x, Av.y, Bv.x, Bv.y);
                } else {
                    out[2 * rec] = make_float4(Av.x, Av.y, Bv.x, Bv.y);
                    out[2 * rec + 1] = make_float4((side ? es_dphi(p, t, tp) : es_dphi(p, tp, t)) + 0.0f, f_of_u(seg), f_of_u(kind), 0.0f);
                }
                prev = cur; tp = t;
            }
            nrec = 0;
        }
        if (!nparts) nrec = 0;
        // ---- table + write, in one pass, or in halves / quarters of the warp's sides when the parts do not fit
        const uint32_t all_parts = __reduce_add_sync(0xffffffffu, nparts);
        if (all_parts == 0u) { __syncwarp(); continue; }
        const uint32_t low_parts = __reduce_add_sync(0xffffffffu, lane < 16 ? nparts : 0u);
        const int n_pass = all_parts <= (uint32_t)kExParts ? 1 : ((low_parts <= (uint32_t)kExParts && all_parts - low_parts <= (uint32_t)kExParts) ? 2 : 4);
        const int pass_shift = n_pass == 2 ? 4 : 3;
        for (int pass = 0; pass < n_pass; pass++) {
            const bool mine = n_pass == 1 || (lane >> pass_shift) == pass;
            const uint32_t np_ = mine ? nparts : 0u, nr_ = mine ? nrec : 0u;
            uint32_t ip = np_, ir = nr_;
#pragma unroll
            for (int dd = 1; dd < 32; dd <<= 1) {
                const uint32_t a2 = __shfl_up_sync(0xffffffffu, ip, dd), b2 = __shfl_up_sync(0xffffffffu, ir, dd);
                if (lane >= dd) { ip += a2; ir += b2; }
            }
            const uint32_t tparts = __shfl_sync(0xffffffffu, ip, 31), trecs = __shfl_sync(0xffffffffu, ir, 31);
            if (np_) side_parts(plan_unpack(W.plan[lane]), (uint32_t)lane, side != 0, arc, base, ir - nr_, np_, &W.part[ip - np_], &W.ppref[ip - np_]);
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
                const int need_max = __reduce_max_sync(0xffffffffu, need);
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
                        float hh;
                        uint32_t sg;
                        leaf_piece(S, tile0, S.leaf[W.leaf[ss >> 1]], pc, &hh, &sg);
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
                    float hh;
                    uint32_t sg;
                    leaf_piece(S, tile0, S.leaf[W.leaf[ss >> 1]], pc, &hh, &sg);
                    const PlanLite& sp = W.plan[ss];
                    const float4 cusp = W.cusp[ss];
                    V2 Av, Bv;
                    float tA, tB;
                    if (s_int) { const float4 q = W.ring[(uint32_t)(v_end - 1) & (uint32_t)(kRing - 1)]; Av = v2(q.x, q.y); tA = q.z; }
                    else Av = end_vertex(pc, (pt.info >> 16) & 7u, sp.eta, cusp, &tA);
                    if (e_int) { const float4 q = W.ring[(uint32_t)v_end & (uint32_t)(kRing - 1)]; Bv = v2(q.x, q.y); tB = q.z; }
                    else Bv = end_vertex(pc, (pt.info >> 19) & 7u, sp.eta, cusp, &tB);
                    const uint64_t rec = pt.base + m;
                    if (!arc) {
                        out[rec] = make_float4(Av.x, Av.y, Bv.x, Bv.y);
                    } else {
                        out[2 * rec] = make_float4(Av.x, Av.y, Bv.x, Bv.y);
                        out[2 * rec + 1] = make_float4((pt.info & 2048u) ? es_dphi(pc, tA, tB) + 0.0f : 0.0f, f_of_u(sp.seg), f_of_u((pt.info >> 12) & 15u), 0.0f);
                    }
                }
                __syncwarp();
            }
            __syncwarp();
        }
    }
}

// ---------------------------------------------------------------- the kernel
template <bool WRITE>
__global__ void __launch_bounds__(kExThreads, 2)
k_expand(const ExArgs A) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    ExShared& S = *reinterpret_cast<ExShared*>(smem_raw);
    const Params& P = A.P;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) {
        S.range = atomicAdd(A.ticket, 1u);
        uint32_t nt = A.force_tiles ? A.force_tiles : *reinterpret_cast<volatile uint32_t*>(A.hint);
        S.n_tiles = nt >= 4u ? 4u : (nt >= 2u ? 2u : 1u);
        S.fill_max = 0;
    }
    __syncthreads();
    const uint32_t range = S.range, range0 = range * (uint32_t)kExRange;
    const uint32_t n_tiles = S.n_tiles, tile_segs = (uint32_t)kExRange / n_tiles, tile_slots = (uint32_t)kExSlotsPerRange / n_tiles;
    const bool ok = *A.err == 0u;
    bool cap_overflow = false;
    uint64_t running = 0;   // records before the current tile (known without a look-back from the block's second tile on)

    for (uint32_t t = 0; t < n_tiles; t++) {
        const uint32_t tile0 = range0 + t * tile_segs;
        if (tile0 >= P.n_tags) break;
        const uint32_t n_in_tile = min(tile_segs, P.n_tags - tile0);
        __syncthreads();   // the previous tile's writers are done with the shared tables
        if (tid == 0) {
            S.q_head = 0; S.q_tail = 0; S.n_leaf = 0; S.overflow = A.force_tiles == 8u ? 4u : 0u;
            S.n_simple = 0; S.n_complex = 0; S.chunk = 0;
        }

        // ================================================================ A: segments
        uint32_t my_tag = 0, my_first = 0, my_path = 0;
        bool my_valid = false, my_curve = false;
        if (tid < (int)n_in_tile) {
            const uint32_t i = tile0 + (uint32_t)tid;
            my_tag = P.tags[i];
            my_path = P.path_idx[i];
            my_first = P.sp_first[i];
            const uint32_t pt = P.pt_off[i];
            Style st;
            float h;
            my_valid = load_style(P, my_path, &st, &h) && ok;
            const Seg s = load_segment_at(P, pt, my_tag);
            my_curve = my_valid && s.kind != 1 && !s.degenerate;
            SegRec r;
            r.p0x = s.P0.x; r.p0y = s.P0.y;
            r.c1x = s.c1.x; r.c1y = s.c1.y; r.c2x = s.c2.x; r.c2y = s.c2.y; r.c3x = s.c3.x; r.c3y = s.c3.y;
            r.tsx = s.ts.x; r.tsy = s.ts.y; r.tex = s.te.x; r.tey = s.te.y;
            r.p3x = s.P3.x; r.p3y = s.P3.y;
            r.h = h;
            r.info = (my_valid ? 1u : 0u) | (my_curve ? 2u : 0u) | (my_tag << 8);
            r.n_tail = 0; r.off = 0; r.pad[0] = r.pad[1] = 0;
            S.seg[tid] = r;
            // the two end points of a curve are points 2 tid and 2 tid + 1 of the table; its root node is tree slot tid
            if (my_curve) {
                float qm;
                V2 pos, u;
                S.pts[2 * tid] = make_float4(0.0f, 0.0f, s.ts.x, s.ts.y);
                S.u.fit.qmag[2 * tid] = sqrtf(len2(s.c1));
                eval_cubic(s, 1.0f, 1.0f, &pos, &qm, &u);
                S.pts[2 * tid + 1] = make_float4(pos.x, pos.y, u.x, u.y);
                S.u.fit.qmag[2 * tid + 1] = qm;
            }
            S.u.fit.acc[tid] = 0u;
            S.u.fit.parent[tid] = 0xffffu;
        }
        uint32_t n_roots;
        {   // roots into the queue, in segment order
            const uint32_t ballot = __ballot_sync(0xffffffffu, my_curve);
            if (lane == 0) S.warp_sum[warp] = __popc(ballot);
            __syncthreads();
            uint32_t wbase = 0, tot = 0;
#pragma unroll
            for (int k = 0; k < kExWarps; k++) {
                if (k == warp) wbase = tot;
                tot += S.warp_sum[k];
            }
            n_roots = tot;
            if (my_curve) {
                const uint32_t q = wbase + __popc(ballot & ((1u << lane) - 1u));
                S.u.fit.queue[q] = make_uint4(0u, (uint32_t)(2 * tid) | ((uint32_t)(2 * tid + 1) << 16), (uint32_t)tid | ((uint32_t)tid << 8), 0u);
            }
            if (tid == 0) S.q_tail = tot;
        }
        // join / cap record counts (partners from the tile's records: S.seg is complete after the barrier above)
        if (tid < (int)n_in_tile && my_valid) {
            const SegRec& r = S.seg[tid];
            Style st;
            float h;
            load_style(P, my_path, &st, &h);
            S.seg[tid].n_tail = tile_segment_tail<false>(S, P, tile0, n_in_tile, tile0 + (uint32_t)tid, my_tag, v2(r.p3x, r.p3y), v2(r.tex, r.tey), st, h,
                                                         my_first, nullptr, 0);
        }

        // ================================================================ B: Alg. 2, node-parallel
        for (;;) {
            __syncthreads();
            const uint32_t head = S.q_head, tail = S.q_tail;
            const uint32_t avail = tail - head;
            const bool stop = avail == 0u || S.overflow != 0u;
            __syncthreads();
            if (stop) break;
            const uint32_t n_round = min(avail, (uint32_t)kExThreads);
            bool push = false;
            uint32_t slot = 0, sl = 0, level = 0, t0_u = 0, pa_i = 0, pb_i = 0;
            float4 mid = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            float mid_q = 0.0f;
            if ((uint32_t)tid < n_round) {
                const uint4 node = S.u.fit.queue[(head + (uint32_t)tid) & (uint32_t)(kExQueueCap - 1)];
                t0_u = node.x & 0xfffffu; level = node.x >> 20;
                pa_i = node.y & 0xffffu; pb_i = node.y >> 16;
                sl = node.z & 0xffu; slot = node.z >> 8;
                const float4 a = S.pts[pa_i], b = S.pts[pb_i];
                const float dt = __uint_as_float((127u - level) << 23);
                const float err = node_error(v2(a.z, a.w), v2(b.z, b.w), S.u.fit.qmag[pa_i], S.u.fit.qmag[pb_i], v2(b.x, b.y) - v2(a.x, a.y), dt);
                if (err <= P.tol_es || level >= (uint32_t)kExLevelMax) {
                    const uint32_t k = atomicAdd(&S.n_leaf, 1u);
                    if (k < (uint32_t)kExLeafCap) {
                        Leaf lf;
                        lf.ab = node.y; lf.seg_slot = node.z; lf.k0 = lf.k1 = lf.L = 0.0f; lf.n = 0; lf.rel = 0;
                        S.leaf[k] = lf;
                    } else S.overflow = 1u;
                } else {
                    // split: the mid point is evaluated once, for both children (Alg. 2 L369 with the rule of L251)
                    push = true;
                    const Seg s = seg_of(S.seg[sl]);
                    const float tm = (float)t0_u * dt + 0.5f * dt;
                    const V2 q = cubic_q(s, tm);
                    const float q2 = len2(q);
                    mid_q = sqrtf(q2);
                    const V2 pos = cubic_pos(s, tm);
                    if (q2 < kEpsQ2) S.overflow = 2u;   // zero derivative inside the curve: the visiting order matters (L251)
                    mid = make_float4(pos.x, pos.y, q.x / mid_q, q.y / mid_q);
                }
            }
            // children: one point, two tree slots, two queue entries per split (one shared-memory atomic per warp)
            const uint32_t pb = __ballot_sync(0xffffffffu, push);
            if (pb) {
                uint32_t base = 0;
                const uint32_t cnt = __popc(pb);
                const int leader = __ffs((int)pb) - 1;
                if (lane == leader) base = atomicAdd(&S.q_tail, 2u * cnt);
                base = __shfl_sync(0xffffffffu, base, leader);
                if (push) {
                    const uint32_t rank = __popc(pb & ((1u << lane) - 1u));
                    const uint32_t k = ((base - n_roots) >> 1) + rank;   // k-th split of the tile
                    const uint32_t pm = 2u * (uint32_t)kExRange + k, ts = (uint32_t)kExRange + 2u * k;
                    // the ring must hold everything from this round's first entry to the new tail
                    if (k >= (uint32_t)kExSplitCap || base + 2u * cnt - head > (uint32_t)kExQueueCap) S.overflow = 1u;
                    else {
                        S.pts[pm] = mid;
                        S.u.fit.qmag[pm] = mid_q;
                        S.u.fit.parent[ts] = (uint16_t)slot; S.u.fit.parent[ts + 1u] = (uint16_t)slot;
                        S.u.fit.acc[ts] = 0u; S.u.fit.acc[ts + 1u] = 0u;
                        const uint32_t q = (base + 2u * rank) & (uint32_t)(kExQueueCap - 1);
                        const uint32_t lv = (level + 1u) << 20;
                        S.u.fit.queue[q] = make_uint4((2u * t0_u) | lv, pa_i | (pm << 16), sl | (ts << 8), 0u);
                        S.u.fit.queue[(q + 1u) & (uint32_t)(kExQueueCap - 1)] = make_uint4((2u * t0_u + 1u) | lv, pm | (pb_i << 16), sl | ((ts + 1u) << 8), 0u);
                    }
                }
            }
            if (tid == 0) S.q_head = head + n_round;
        }
        // (the loop ends with a barrier: S.overflow, S.n_leaf and the tables are final)
        const bool slow_b = S.overflow != 0u;
        const uint32_t n_leaf = slow_b ? 0u : S.n_leaf;

        // ================================================================ C: pieces (lane pair per leaf)
        if (!slow_b) {
            for (uint32_t l0 = 0; l0 < n_leaf; l0 += (uint32_t)kExThreads / 2u) {
                const uint32_t li = l0 + (uint32_t)(tid >> 1);
                const int side = lane & 1;
                const bool live = li < n_leaf;
                Leaf lf;
                lf.ab = 0; lf.seg_slot = 0; lf.k0 = lf.k1 = lf.L = 0.0f; lf.n = 0; lf.rel = 0;
                if (live) lf = S.leaf[li];
                const uint32_t a = lf.ab & 0xffffu, b = lf.ab >> 16, sl = lf.seg_slot & 0xffu, slot = lf.seg_slot >> 8;
                const float4 pa = S.pts[a], pb = S.pts[b];
                const V2 ch = v2(pb.x, pb.y) - v2(pa.x, pa.y);
                const float chord2 = len2(ch), chord = sqrtf(chord2);
                float th = 0.0f;
                if (live && chord2 >= kEpsQ2) {   // (a zero chord is accepted at the deepest level only: th0 = th1 = 0, as in fit_error)
                    const V2 uc = v2(ch.x / chord, ch.y / chord);
                    const V2 u0 = v2(pa.z, pa.w), u1 = v2(pb.z, pb.w);
                    th = side ? atan2_r(cross(uc, u1), dot(uc, u1)) : atan2_r(cross(u0, uc), dot(u0, uc));
                }
                const float tho = __shfl_xor_sync(0xffffffffu, th, 1);
                Piece p;
                piece_params(p, side ? tho : th, side ? th : tho, chord);
                const float h = S.seg[sl].h;
                uint32_t n = 0;
                bool simple = false;
                if (live) {
                    const SidePlan sp = side_plan(p, side ? h : -h, P.mode, P.tol_fl);
                    n = (uint32_t)sp.total;
                    simple = sp.nr == 1 && !sp.sup[0];
                }
                const uint32_t no = __shfl_xor_sync(0xffffffffu, n, 1);
                const bool so = __shfl_xor_sync(0xffffffffu, simple ? 1 : 0, 1) != 0;
                if (live && side == 0) {
                    if (n > 0xffffu || no > 0xffffu) S.overflow = 1u;   // a side of more than 65535 records: the slow walk
                    lf.k0 = p.k0; lf.k1 = p.k1; lf.L = p.L;
                    lf.n = (n & 0xffffu) | (no << 16);
                    lf.rel = (simple ? kLeafSimpleMinus : 0u) | (so ? kLeafSimplePlus : 0u);   // parked here until phase D
                    S.leaf[li] = lf;
                    // subtree sums: the leaf's records are added to itself and to all its ancestors
                    const uint32_t c = n + no;
                    uint32_t cur = slot;
                    while (cur != 0xffffu) { atomicAdd(&S.u.fit.acc[cur], c); cur = S.u.fit.parent[cur]; }
                    // order[]: leaves whose two sides are short single ranges first (the direct writer), the others last
                    const bool both = simple && so && n <= (uint32_t)kExDirectMax && no <= (uint32_t)kExDirectMax;
                    if (both) S.order[atomicAdd(&S.n_simple, 1u)] = (uint16_t)li;
                    else S.order[(uint32_t)kExLeafCap - 1u - atomicAdd(&S.n_complex, 1u)] = (uint16_t)li;
                }
            }
        }
        __syncthreads();
        const bool slow = S.overflow != 0u;
        cap_overflow |= (S.overflow & 1u) != 0u;

        // ================================================================ D: allocation
        uint32_t my_count = 0;   // records of segment tid
        if (!slow) {
            // records that precede a leaf in its segment: over the path to the root, the left siblings' subtree sums
            for (uint32_t li = (uint32_t)tid; li < n_leaf; li += (uint32_t)kExThreads) {
                const uint32_t ss = S.leaf[li].seg_slot, flags = S.leaf[li].rel;
                uint32_t cur = ss >> 8, rel = 0;
                while (cur >= (uint32_t)kExRange) {
                    if ((cur - (uint32_t)kExRange) & 1u) rel += S.u.fit.acc[cur - 1u];
                    cur = S.u.fit.parent[cur];
                }
                S.leaf[li].rel = rel;
                S.leaf[li].seg_slot = (ss & 0xffu) | flags;
            }
            if (tid < (int)n_in_tile && my_valid) my_count = (my_curve ? S.u.fit.acc[tid] : 2u) + S.seg[tid].n_tail;
        } else if (tid < (int)n_in_tile && ok) {
            my_count = slow_count(P, tile0 + (uint32_t)tid);
        }
        uint32_t tile_total;
        const uint32_t my_off = block_exclusive_scan(my_count, S.warp_sum, &tile_total);
        if (tid < (int)n_in_tile) S.seg[tid].off = my_off;
        if (warp == 0) {
            const uint64_t excl = tile_publish(A.states, range * (uint32_t)kExSlotsPerRange + t * tile_slots, tile_slots, t == 0u, running, (uint64_t)tile_total);
            if (lane == 0) S.tile_base = excl;
        }
        __syncthreads();
        const uint64_t tile_base = S.tile_base;
        running = tile_base + tile_total;
        if (tid < (int)n_in_tile) {
            const uint32_t i = tile0 + (uint32_t)tid;
            const uint64_t off = tile_base + my_off;
            if (A.seg_count) { A.seg_count[i] = my_count; A.seg_off[i] = off; }
            if (ok && (i == 0u || (P.tags[i - 1u] & 16u)) && my_path < A.n_paths) A.path_off[my_path] = off;   // first segment of a path (Table 1)
            if (i == P.n_tags - 1u) { A.path_off[A.n_paths] = off + my_count; *A.d_total = off + my_count; }
        }
        if (tid == 0) {
            atomicAdd(A.stats + (slow ? 1 : 0), 1u);
            S.fill_max = max(S.fill_max, max(n_leaf * 100u / (uint32_t)kExLeafCap, (S.q_tail - n_roots) * 50u / (uint32_t)kExSplitCap));
        }
        if (!WRITE) continue;

        // ================================================================ E: write
        if (tile_base + tile_total > A.cap_records) {   // the tile does not fit the caller's buffer: nothing of it is written
            if (tid == 0) atomicOr(A.err, kErrCapacity);
            continue;
        }
        if (slow) {
            if (tid < (int)n_in_tile && my_count) {
                Writer w;
                w.out = A.out; w.base = tile_base + my_off; w.seg = tile0 + (uint32_t)tid; w.mode = P.mode;
                slow_write(P, tile0 + (uint32_t)tid, &w);
            }
            continue;
        }
        // E1: straight segments, joins, caps (thread per segment)
        if (tid < (int)n_in_tile && my_valid) {
            const SegRec& r = S.seg[tid];
            Style st;
            float h;
            load_style(P, my_path, &st, &h);
            Writer w;
            w.out = A.out; w.base = tile_base + my_off; w.seg = tile0 + (uint32_t)tid; w.mode = P.mode;
            const V2 P0 = v2(r.p0x, r.p0y), P3 = v2(r.p3x, r.p3y), ts = v2(r.tsx, r.tsy), te = v2(r.tex, r.tey);
            if (!my_curve) {
                w.put(0, offset_point(P0, ts, -h), offset_point(P3, te, -h), 0.0f, kOffset);
                w.put(1, offset_point(P3, te, h), offset_point(P0, ts, h), 0.0f, kOffset | kPlus);
            }
            tile_segment_tail<true>(S, P, tile0, n_in_tile, tile0 + (uint32_t)tid, my_tag, P3, te, st, h, my_first, &w, my_count - r.n_tail);
        }
        // E2: the pieces (the fit area is dead since the barrier after the look-back: it becomes the warps' stages)
        write_pieces(S, A, tile0, tile_base, n_leaf, S.n_simple);
    }
    // adapt the number of tiles per range for the blocks (and calls) that follow
    // (only full ranges vote for larger tiles: the stream's ragged last range says nothing about the scene)
    if (tid == 0 && A.force_tiles == 0u) {
        if (cap_overflow && n_tiles < 4u) atomicMax(A.hint, n_tiles * 2u);
        else if (!cap_overflow && n_tiles > 1u && S.fill_max < 30u && range0 + (uint32_t)kExRange <= P.n_tags) atomicMin(A.hint, n_tiles / 2u);
    }
}

}  // namespace sx
