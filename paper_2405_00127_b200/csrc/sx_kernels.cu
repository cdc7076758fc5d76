// sx_kernels.cu -- count kernel (b), the write kernels (d1 pieces, d2 segments, d3 fallback) and the C-ABI of
// include/stroke_expand.h.  The two scans (a), (c) are in sx_scan.cuh, the curve mathematics in sx_math.cuh /
// sx_piece.cuh, the thread-per-segment reference walk in sx_segment.cuh, the piece cache and part tables in sx_cache.cuh.
//
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -fmad=false -lineinfo -shared (see ../build.py).
// -fmad=false is part of the design: see the arithmetic discipline note in sx_math.cuh.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>

#include "../../include/stroke_expand.h"
#include "sx_scan.cuh"
#include "sx_cache.cuh"

namespace sx {

constexpr int kSegThreads = 128;           // thread-per-segment kernels (d2, d3)
constexpr int kCntThreads = 32;            // count kernel: curves (and segments) per block
constexpr int kWpThreads = 224;            // write kernel: threads per block (7 independent warps)
constexpr int kWpBlocksPerSM = 4;
constexpr int kShortSide = 2;               // records of a "short" side (scene statistic of the count kernel)
constexpr int kDirectMax = 6;               // DIRECT variant: records of a side its own staging thread writes

// (b) count pass: the number of records of every segment, and the piece cache.
// Part 1, one thread per segment of the block's tile: straight segments (2 exact offset lines + join / caps).
// Part 2, one thread per entry of the compact curve list built by the tag scan (so that a scene that mixes lines
// and curves still fills its warps with curves).  The block works in rounds: every thread advances its curve to
// its next accepted piece (fit_next, Alg. 2); the round's pieces are compacted through shared memory and
// their 2 x T side plans are spread over ALL threads of the block (a thread whose curve is finished still plans
// for its neighbours); one atomic per round reserves exactly T descriptor slots of the piece cache.
__global__ void __launch_bounds__(kCntThreads, 32)
k_count(Params P, uint32_t* __restrict__ seg_count, const uint32_t* __restrict__ curve_idx, const uint32_t* __restrict__ n_curves_p,
        float4* __restrict__ pieces, uint32_t piece_cap, uint32_t* piece_ctr, uint32_t* side_stats, const uint32_t* __restrict__ err) {
    __shared__ float4 s_q[kCntThreads];          // k0, k1, L, h of the round's pieces
    __shared__ uint32_t s_n[2 * kCntThreads];    // their side totals (-h, +h)
    __shared__ uint32_t s_wcnt[kCntThreads / 32];
    __shared__ uint32_t s_base;
    __shared__ uint32_t s_stat[2];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const bool ok = *err == 0u;
    {   // ---- part 1: straight segments of this block's tile
        const uint32_t i = blockIdx.x * (uint32_t)kCntThreads + (uint32_t)tid;
        if (i < P.n_tags) {
            const uint32_t tag = P.tags[i];
            if (!ok) seg_count[i] = 0u;
            else if ((tag & 3u) == 1u) {
                Style st;
                float h;
                uint32_t n = 0;
                if (load_style(P, P.path_idx[i], &st, &h)) {
                    Seg s = load_segment(P, i, tag);
                    n = 2u + segment_tail<false>(P, i, tag, s, st, h, nullptr, 0);
                }
                seg_count[i] = n;
            }
        }
    }
    // ---- part 2: curves
    const uint32_t n_curves = ok ? *n_curves_p : 0u;
    const uint32_t rank = blockIdx.x * (uint32_t)kCntThreads + (uint32_t)tid;
    if (blockIdx.x * (uint32_t)kCntThreads >= n_curves) return;
    if (tid < 2) s_stat[tid] = 0u;
    uint32_t st_all = 0, st_short = 0;  // sides planned by this thread / of which one short regular range
    bool active = false;
    uint32_t i = 0, n = 0, n_tail = 0;
    Seg s;
    FitState f;
    float h = 0.0f;
    if (rank < n_curves) {
        i = curve_idx[rank];
        const uint32_t tag = P.tags[i];
        Style st;
        if (!load_style(P, P.path_idx[i], &st, &h)) {
            seg_count[i] = 0u;
        } else {
            s = load_segment(P, i, tag);
            n_tail = segment_tail<false>(P, i, tag, s, st, h, nullptr, 0);
            if (s.degenerate) seg_count[i] = 2u + n_tail;  // all control points coincide: straight path (R-5)
            else { active = true; f = fit_begin(s); }
        }
    }
    for (;;) {
        bool have = false;
        Piece p;
        if (active) {
            have = fit_next(P, s, f, p);
            if (!have) { seg_count[i] = n + n_tail; active = false; }
        }
        const uint32_t ballot = __ballot_sync(0xffffffffu, have);
        if (lane == 0) s_wcnt[warp] = __popc(ballot);
        __syncthreads();
        uint32_t T = 0, wbase = 0;
#pragma unroll
        for (int k = 0; k < kCntThreads / 32; k++) {
            if (k == warp) wbase = T;
            T += s_wcnt[k];
        }
        if (T == 0u) break;  // fit_next yields a piece every round until the curve ends (block-uniform)
        const uint32_t idx = wbase + __popc(ballot & ((1u << lane) - 1u));
        if (have) s_q[idx] = make_float4(p.k0, p.k1, p.L, h);
        if (tid == 0) s_base = atomicAdd(piece_ctr, T);
        __syncthreads();
        for (uint32_t j = (uint32_t)tid; j < 2u * T; j += (uint32_t)kCntThreads) {
            const float4 q = s_q[j >> 1];
            Piece pp;
            pp.k0 = q.x; pp.k1 = q.y; pp.L = q.z;
            const SidePlan sp = side_plan(pp, (j & 1u) ? q.w : -q.w, P.mode, P.tol_fl);
            s_n[j] = (uint32_t)sp.total;
            st_all++;
            st_short += (sp.nr == 1 && !sp.sup[0] && sp.total <= kShortSide) ? 1u : 0u;
        }
        __syncthreads();
        if (have) {
            const uint32_t nm = s_n[2u * idx], np = s_n[2u * idx + 1u], slot = s_base + idx;
            if (slot < piece_cap) piece_store(pieces + (uint64_t)slot * kDescQuads, p, h, i, n, nm, np);
            n += nm + np;
        }
    }
    // scene statistic for the write kernel's choice of variant: how many sides are one short regular range
    st_all = __reduce_add_sync(0xffffffffu, st_all);
    st_short = __reduce_add_sync(0xffffffffu, st_short);
    if (lane == 0) { atomicAdd(&s_stat[0], st_all); atomicAdd(&s_stat[1], st_short); }
    __syncthreads();
    if (tid < 2 && s_stat[tid]) atomicAdd(side_stats + tid, s_stat[tid]);
}

// (d1) write pass over the piece cache: one thread per output record, no per-record branching, no block barriers.
// Every WARP works on its own tile of kWtPieces = 16 descriptors, staged in its own slice of shared memory; the
// warps of a block never wait for one another (a block-wide tile spent a quarter of its time at its three barriers).
//   stage   lane = (piece, side): rebuilds the side plan (same device function as the count kernel, hence the same
//           counts), integrates its half of the piece's anchor table (the lane pair exchanges totals by shuffle),
//           evaluates the side's cusp vertex;
//   table   a warp scan of (parts, records) places the side's PARTS (sx_cache.cuh) in the tile's part table;
//   write   the warp takes 31 consecutive records of the tile per iteration: lane k evaluates the START vertex of
//           record k (lane 31 that of the next record, for lane 30); the END vertex comes from the next lane by
//           shuffle, or is a part end (piece end point / cusp point: no integral).
// Records go out as 16-byte (line) or 2 x 16-byte (arc) stores to consecutive addresses within a part.  A tile whose
// sides have more than kWtParts parts in all (the worst case is 8 per side) is processed in two halves or four
// quarters of its sides.
constexpr int kWtPieces = 16;
constexpr int kWtSides = 32;
constexpr int kWtParts = 96;
constexpr int kRing = 64;                  // >= 2 x 32: see the write loop
constexpr int kWpWarps = kWpThreads / 32;
struct WarpTile {
    Piece piece[kWtPieces];
    Spiral spiral[kWtPieces];
    PlanLite plan[kWtSides];
    float4 cusp[kWtSides];          // x, y, t of the side's cusp vertex
    Part part[kWtParts];
    uint32_t ppref[kWtParts + 1];
    uint32_t pad[3];
    float4 ring[kRing];             // x, y, t of the interior vertices just ahead of the records being written
};

// Two variants, chosen on the DEVICE from the count kernel's scene statistic (both are launched, one exits at once):
// DIRECT = true when at least 80 % of the sides are one short regular range (CAD-like scenes: 2-3 records per
// side): such sides are then written by their own staging lane, without tables -- when (nearly) the whole warp is
// like that.  On evolute-heavy scenes the extra path only costs registers, hence the separate instantiation.
template <bool DIRECT>
__global__ void __launch_bounds__(kWpThreads, kWpBlocksPerSM)
k_write_pieces(Params P, const float4* __restrict__ pieces, uint32_t piece_cap, const uint32_t* __restrict__ piece_ctr,
               const uint32_t* __restrict__ side_stats, const uint64_t* __restrict__ seg_off, float4* __restrict__ out,
               uint64_t cap_records, uint32_t* err) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const uint32_t reserved = *piece_ctr;
    if (reserved > piece_cap) return;  // cache overflow: k_write_fallback takes the whole call
    if (((uint64_t)side_stats[1] * 10u >= (uint64_t)side_stats[0] * 8u) != DIRECT) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpTile& S = reinterpret_cast<WarpTile*>(smem_raw)[warp];
    const bool arc = P.mode == kModeArc;
    const uint32_t n_warps = gridDim.x * (uint32_t)kWpWarps;
    const int side = lane & 1;
    // The head of a descriptor (segment, relative offset, side totals) and the record offset of its segment are a chain
    // of two dependent loads at the start of every tile: they are fetched one tile ahead, into registers.
    float4 q4_next = make_float4(f_of_u(kInvalidSeg), 0.0f, 0.0f, 0.0f);
    uint64_t off_next = 0;
    {
        const uint64_t slot0 = (uint64_t)(blockIdx.x * (uint32_t)kWpWarps + (uint32_t)warp) * kWtPieces + (uint64_t)(lane >> 1);
        if (slot0 < reserved) { q4_next = __ldg(pieces + slot0 * kDescQuads + 4); off_next = seg_off[u_of_f(q4_next.x)]; }
    }
    for (uint32_t tile = blockIdx.x * (uint32_t)kWpWarps + (uint32_t)warp; (uint64_t)tile * kWtPieces < reserved; tile += n_warps) {
        // ---- stage
        const float4 q4 = q4_next;
        const uint64_t seg_base = off_next;
        {
            const uint64_t nslot = (uint64_t)(tile + n_warps) * kWtPieces + (uint64_t)(lane >> 1);
            q4_next = make_float4(f_of_u(kInvalidSeg), 0.0f, 0.0f, 0.0f);
            if (nslot < reserved) q4_next = __ldg(pieces + nslot * kDescQuads + 4);  // an L2 hit (prefetched below, a tile ago)
        }
        {   // pull the next tile's descriptors (16 x 80 B = ten 128-byte lines) into L2 while this tile is worked on
            const uint64_t nslot = (uint64_t)(tile + n_warps) * kWtPieces;
            if (lane < 10 && nslot < reserved)
                asm volatile("prefetch.global.L2 [%0];" ::"l"(reinterpret_cast<const char*>(pieces + nslot * kDescQuads) + 128 * lane));
        }
        const uint32_t slot = tile * (uint32_t)kWtPieces + (uint32_t)(lane >> 1);
        Piece p;
        p.k0 = 0.0f; p.k1 = 0.0f;
        float h = 0.0f;
        PieceHead hd;
        hd.seg = kInvalidSeg;
        if (slot < reserved) {
            const float4* d = pieces + (uint64_t)slot * kDescQuads;
            hd = piece_head(q4);
            piece_load(d, hd, p, &h);
        }
        const bool live = hd.seg != kInvalidSeg;
        const float eta = side ? h : -h;
        uint32_t nparts = 0, nrec = 0, ndirect = 0;
        uint64_t base = 0;
        bool simple = false, two_ranges = false;
        float tc = 0.0f;
        if (live) {
            SidePlan sp = side_plan(p, eta, P.mode, P.tol_fl);
            nrec = (uint32_t)sp.total;
            base = seg_base + hd.rel + (side ? hd.n_minus : 0u);
            if (base + nrec > cap_records) { atomicOr(err, kErrCapacity); nrec = 0; }
            else nparts = side_part_count(sp);
            simple = DIRECT && nparts == 1u && !sp.sup[0] && nrec <= (uint32_t)kDirectMax;
            two_ranges = sp.nr == 2;
            tc = sp.off[0].tb;
            sp.seg = hd.seg;
            S.plan[lane] = plan_pack(sp);
            if (side == 0) S.piece[lane >> 1] = p;
        }
        {   // anchor table: each of the two lanes of a piece integrates one half, then they exchange totals
            const int K = es_intervals(p.k0, p.k1);
            float hx[kAnchors / 2], hy[kAnchors / 2], tx, ty;
            const int cnt = es_anchor_half<DIRECT>(p, K, side, hx, hy, &tx, &ty);
            const float ox = __shfl_xor_sync(0xffffffffu, tx, 1), oy = __shfl_xor_sync(0xffffffffu, ty, 1);
            if (live) es_anchor_store(S.spiral[lane >> 1], K, side, cnt, hx, hy, tx, ty, ox, oy);
        }
        if (DIRECT) {  // a mixed warp would wait for its few direct writers: all or (nearly) nothing
            if (__popc(__ballot_sync(0xffffffffu, simple)) >= 28 && simple) { ndirect = nrec; nrec = 0; nparts = 0; }
        }
        __syncwarp();
        // the side's cusp vertex: the parallel curve at the cusp parameter (L380-386), evaluated once and shared by the
        // parts that meet there (a side has a cusp iff it has two ranges)
        if (live && two_ranges) {
            V2 c = normal_point_sel<DIRECT>(S.piece[lane >> 1], S.spiral[lane >> 1], tc, eta);
            S.cusp[lane] = make_float4(c.x, c.y, tc, 0.0f);
        }
        if (DIRECT && ndirect) {
            // vertices 0..n of the range in forward order, records stored mirrored for the +h side; the same vertex
            // functions as the table path, hence bit-identical records
            const OffPlan o = plan_off(S.plan[lane], false);
            const Spiral& z = S.spiral[lane >> 1];
            const float4 nocusp = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            const uint32_t kind = side ? (uint32_t)(kOffset | kPlus) : (uint32_t)kOffset;
            float tp;
            V2 prev = end_vertex(p, kEndT0, eta, nocusp, &tp);
            for (uint32_t i = 1; i <= ndirect; i++) {
                float t;
                V2 cur;
                if (i < ndirect) { t = offset_t(p, o, eta, (int)i); cur = normal_point_sel<DIRECT>(p, z, t, eta); }
                else cur = end_vertex(p, kEndT1, eta, nocusp, &t);
                const uint64_t rec = base + (side ? ndirect - i : i - 1u);
                const V2 A = side ? cur : prev, B = side ? prev : cur;
                if (!arc) {
                    out[rec] = make_float4(A.x, A.y, B.x, B.y);
                } else {
                    out[2 * rec] = make_float4(A.x, A.y, B.x, B.y);
                    out[2 * rec + 1] = make_float4((side ? es_dphi(p, t, tp) : es_dphi(p, tp, t)) + 0.0f, f_of_u(hd.seg), f_of_u(kind), 0.0f);
                }
                prev = cur; tp = t;
            }
        }
        off_next = u_of_f(q4_next.x) != kInvalidSeg ? seg_off[u_of_f(q4_next.x)] : 0u;  // consumed by the next tile
        // ---- table + write, in one pass, or in two halves of the warp's sides when the parts do not fit
        const uint32_t all_parts = __reduce_add_sync(0xffffffffu, nparts);
        const uint32_t low_parts = __reduce_add_sync(0xffffffffu, lane < 16 ? nparts : 0u);
        // 1 pass; or the two halves of the warp's sides; or its four quarters (8 sides x 8 parts always fit)
        const int n_pass = all_parts <= (uint32_t)kWtParts ? 1 : ((low_parts <= (uint32_t)kWtParts && all_parts - low_parts <= (uint32_t)kWtParts) ? 2 : 4);
        const int pass_shift = n_pass == 2 ? 4 : 3;
        for (int pass = 0; pass < n_pass; pass++) {
            const bool mine = n_pass == 1 || (lane >> pass_shift) == pass;
            const uint32_t np_ = mine ? nparts : 0u, nr_ = mine ? nrec : 0u;
            uint32_t ip = np_, ir = nr_;
#pragma unroll
            for (int dd = 1; dd < 32; dd <<= 1) {
                uint32_t a2 = __shfl_up_sync(0xffffffffu, ip, dd), b2 = __shfl_up_sync(0xffffffffu, ir, dd);
                if (lane >= dd) { ip += a2; ir += b2; }
            }
            const uint32_t tparts = __shfl_sync(0xffffffffu, ip, 31), trecs = __shfl_sync(0xffffffffu, ir, 31);
            if (np_) side_parts(plan_unpack(S.plan[lane]), (uint32_t)lane, side != 0, arc, base, ir - nr_, np_, &S.part[ip - np_], &S.ppref[ip - np_]);
            if (lane == 0) S.ppref[tparts] = trecs;
            __syncwarp();
            // ---- write: 32 records per iteration.  Record r of part i (its m-th) starts at the part's vertex m and ends
            // at vertex m + 1.  The INTERIOR vertices of all parts, in record order, have the running index
            // v = r - i - 1 (start) / r - i (end): they are evaluated densely, 32 at a time by all lanes, into a ring of
            // kRing entries just ahead of the records that use them (both neighbours read the same bits); part ends are
            // piece end points or the cusp point and cost no integral.
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
                    uint32_t hi = tparts;  // largest part with ppref <= r
#pragma unroll 1
                    while (hi - lo > 1u) {
                        uint32_t mid = (lo + hi) >> 1;
                        if (S.ppref[mid] <= r) lo = mid; else hi = mid;
                    }
                    pt = S.part[lo];
                    m = r - S.ppref[lo];
                }
                const bool s_int = act && m >= 1u, e_int = act && m + 1u < (uint32_t)pt.n;
                const int v_end = (int)(r - lo);  // index of the record's end vertex if interior; the start vertex is v_end - 1
                const int need = e_int ? v_end : (s_int ? v_end - 1 : -1);
                const int need_max = __reduce_max_sync(0xffffffffu, need);
                while ((int)v_done <= need_max) {
                    const uint32_t v = v_done + (uint32_t)lane;
                    if (v < tverts) {
                        uint32_t l2 = 0, h2 = tparts;  // largest part j with ppref[j] - j <= v: the part that owns vertex v
#pragma unroll 1
                        while (h2 - l2 > 1u) {
                            uint32_t mid = (l2 + h2) >> 1;
                            if (S.ppref[mid] - mid <= v) l2 = mid; else h2 = mid;
                        }
                        const Part pj = S.part[l2];
                        const uint32_t mm = v - (S.ppref[l2] - l2) + 1u;
                        const uint32_t ss = pj.info & 127u;
                        const Piece& pc = S.piece[ss >> 1];
                        const PlanLite& sp = S.plan[ss];
                        const int idx = (pj.info & 128u) ? (int)pj.i0 - (int)mm : (int)pj.i0 + (int)mm;
                        const bool evo = ((pj.info >> 8) & 3u) == 2u;
                        const float t = evo ? evolute_t(pc, plan_evo(sp), idx) : offset_t(pc, plan_off(sp, (pj.info & 1024u) != 0u), sp.eta, idx);
                        const V2 g = normal_point_sel<DIRECT>(pc, S.spiral[ss >> 1], t, evo ? es_radius(pc, t) : sp.eta);
                        S.ring[v & (uint32_t)(kRing - 1)] = make_float4(g.x, g.y, t, 0.0f);
                    }
                    v_done += 32u;
                    __syncwarp();
                }
                if (act) {
                    const uint32_t ss = pt.info & 127u;
                    const Piece& pc = S.piece[ss >> 1];
                    const PlanLite& sp = S.plan[ss];
                    const float4 cusp = S.cusp[ss];
                    V2 A, B;
                    float tA, tB;
                    if (s_int) { const float4 q = S.ring[(uint32_t)(v_end - 1) & (uint32_t)(kRing - 1)]; A = v2(q.x, q.y); tA = q.z; }
                    else A = end_vertex(pc, (pt.info >> 16) & 7u, sp.eta, cusp, &tA);
                    if (e_int) { const float4 q = S.ring[(uint32_t)v_end & (uint32_t)(kRing - 1)]; B = v2(q.x, q.y); tB = q.z; }
                    else B = end_vertex(pc, (pt.info >> 19) & 7u, sp.eta, cusp, &tB);
                    const uint64_t rec = pt.base + m;
                    if (!arc) {
                        out[rec] = make_float4(A.x, A.y, B.x, B.y);
                    } else {
                        out[2 * rec] = make_float4(A.x, A.y, B.x, B.y);
                        out[2 * rec + 1] = make_float4((pt.info & 2048u) ? es_dphi(pc, tA, tB) + 0.0f : 0.0f,  // + 0: no negative zero
                                                     f_of_u(sp.seg), f_of_u((pt.info >> 12) & 15u), 0.0f);
                    }
                }
                __syncwarp();
            }
            __syncwarp();
        }
    }
}

// (d2) write pass over the segments: the records that are not Euler-spiral pieces (the two exact offset
// lines of a straight segment, joins, caps).
__global__ void __launch_bounds__(kSegThreads)
k_write_segments(Params P, const uint32_t* __restrict__ seg_count, const uint64_t* __restrict__ seg_off, float4* __restrict__ out,
                 uint64_t cap_records, uint32_t piece_cap, const uint32_t* __restrict__ piece_ctr, uint32_t* err) {
    uint32_t i = blockIdx.x * (uint32_t)kSegThreads + threadIdx.x;
    if (i >= P.n_tags) return;
    // everything that can be loaded from i alone, in one batch (the kernel is bound by the latency of its dependent loads)
    const uint32_t jn = i + 1u < P.n_tags ? i + 1u : i;
    const uint32_t n = seg_count[i], tag = P.tags[i], path = P.path_idx[i], pt = P.pt_off[i], first_seg = P.sp_first[i];
    const uint32_t tag_n = P.tags[jn], pt_n = P.pt_off[jn];
    const uint64_t off = seg_off[i];
    if (n == 0u) return;
    if (off + n > cap_records) { atomicOr(err, kErrCapacity); return; }
    Writer w;
    w.out = out; w.base = off; w.seg = i; w.mode = P.mode;
    if (*piece_ctr > piece_cap) return;  // cache overflow: k_write_fallback takes the whole call
    Style st;
    float h;
    load_style(P, path, &st, &h);
    Seg s = load_segment_at(P, pt, tag);
    uint32_t first;
    if (s.kind == 1 || s.degenerate) { emit_straight(s, h, &w); first = 2u; }
    else first = n - segment_tail<false>(P, tag, s, st, h, first_seg, tag_n, pt_n, nullptr, 0);
    segment_tail<true>(P, tag, s, st, h, first_seg, tag_n, pt_n, &w, first);
}

// (d3) thread-per-segment writer for a call whose pieces did not fit the cache (sx_set_piece_cache_limit, or
// an asynchronous sx_count that outgrew the cache): repeats Alg. 2 per segment.  Exits at once otherwise.
__global__ void __launch_bounds__(kSegThreads)
k_write_fallback(Params P, const uint32_t* __restrict__ seg_count, const uint64_t* __restrict__ seg_off, float4* __restrict__ out,
                 uint64_t cap_records, uint32_t piece_cap, const uint32_t* __restrict__ piece_ctr, uint32_t* err) {
    if (*piece_ctr <= piece_cap) return;
    uint32_t i = blockIdx.x * (uint32_t)kSegThreads + threadIdx.x;
    if (i >= P.n_tags) return;
    uint32_t n = seg_count[i];
    if (n == 0u) return;
    uint64_t off = seg_off[i];
    if (off + n > cap_records) { atomicOr(err, kErrCapacity); return; }
    Writer w;
    w.out = out; w.base = off; w.seg = i; w.mode = P.mode;
    process_segment<true>(P, i, &w);
}

}  // namespace sx

// ====================================================================== host side
static thread_local cudaError_t g_last_cuda = cudaSuccess;

#define SX_CUDA(call)                                      \
    do {                                                   \
        cudaError_t e_ = (call);                           \
        if (e_ != cudaSuccess) { g_last_cuda = e_; return SX_E_CUDA; } \
    } while (0)

struct sx_ctx {
    int device;
    // scratch of the call in flight
    uint32_t *pt_off, *path_idx, *sp_first, *seg_count, *curve_idx;
    uint64_t* seg_off;
    uint64_t cap_segs;
    uint8_t* sync_area;   // [flags 64 B][d_total 64 B][alloc tile states][tag tile states]
    uint64_t sync_bytes;
    uint64_t* h_pinned;   // pinned: [0] total, [1] flags, [2] piece-cache slots reserved
    float4* pieces;       // piece cache (sx_cache.cuh), piece_cap descriptors
    uint64_t piece_cap;
    uint64_t piece_limit; // 0 = no limit (sx_set_piece_cache_limit)
    int sm_count;
    cudaStream_t side_stream;   // k_write_segments runs here, beside k_write_pieces on the caller's stream
    cudaEvent_t ev_fork, ev_join;
    // last sx_count
    sx::Params P;
    uint64_t n_paths;
    bool counted, total_known;
    bool cache_fits;      // known on the host (synchronous sx_count): every piece of the last count is cached
    uint64_t total;
    uint64_t launches;
    // staging for stroke_expand_host
    uint8_t* st_in;  uint64_t st_in_bytes;
    uint8_t* st_out; uint64_t st_out_bytes;
    uint64_t* st_path; uint64_t st_path_n;
};

static uint32_t* ctx_err(sx_ctx* c) { return reinterpret_cast<uint32_t*>(c->sync_area); }
static uint32_t* ctx_ticket(sx_ctx* c, int k) { return reinterpret_cast<uint32_t*>(c->sync_area) + 4 + 4 * k; }
static uint32_t* ctx_piece_ctr(sx_ctx* c) { return reinterpret_cast<uint32_t*>(c->sync_area) + 12; }
static uint32_t* ctx_side_stats(sx_ctx* c) { return reinterpret_cast<uint32_t*>(c->sync_area) + 14; }
static uint32_t* ctx_n_curves(sx_ctx* c) { return reinterpret_cast<uint32_t*>(c->sync_area) + 13; }
static uint64_t* ctx_total(sx_ctx* c) { return reinterpret_cast<uint64_t*>(c->sync_area + 64); }

static uint64_t round_up(uint64_t x, uint64_t m) { return (x + m - 1) / m * m; }

static sx_status ensure_scratch(sx_ctx* c, uint64_t n) {
    uint64_t n_alloc_tiles = (n + sx::kCntTile - 1) / sx::kCntTile + 1, n_tag_tiles = (n + sx::kTagTile - 1) / sx::kTagTile + 1;
    uint64_t need_sync = 128 + round_up(n_alloc_tiles * 8, 64) + n_tag_tiles * sizeof(sx::TagTileState);
    if (need_sync > c->sync_bytes) {
        if (c->sync_area) SX_CUDA(cudaFree(c->sync_area));
        c->sync_area = nullptr; c->sync_bytes = 0;
        uint64_t b = round_up(need_sync + need_sync / 4, 256);
        SX_CUDA(cudaMalloc(&c->sync_area, b));
        c->sync_bytes = b;
    }
    if (n > c->cap_segs) {
        if (c->pt_off) SX_CUDA(cudaFree(c->pt_off));
        c->pt_off = nullptr; c->cap_segs = 0;
        uint64_t cap = round_up(n + n / 8 + 64, 64);
        // one allocation: 5 u32 arrays then the u64 offsets (all 256-byte aligned since cap % 64 == 0)
        uint8_t* p;
        SX_CUDA(cudaMalloc(&p, cap * (6 * 4 + 8)));
        c->pt_off = reinterpret_cast<uint32_t*>(p);
        c->path_idx = c->pt_off + cap;
        c->sp_first = c->path_idx + cap;
        c->seg_count = c->sp_first + cap;
        c->curve_idx = c->seg_count + cap;
        c->seg_off = reinterpret_cast<uint64_t*>(c->curve_idx + 2 * cap);
        c->cap_segs = cap;
    }
    return SX_OK;
}

static sx_status ensure_pieces(sx_ctx* c, uint64_t need) {
    if (c->piece_limit && need > c->piece_limit) need = c->piece_limit;
    if (need <= c->piece_cap) return SX_OK;
    if (c->pieces) SX_CUDA(cudaFree(c->pieces));
    c->pieces = nullptr; c->piece_cap = 0;
    uint64_t cap = c->piece_limit ? need : round_up(need, 1024);
    if (cap > 0xfffffff0ull) cap = 0xfffffff0ull;
    SX_CUDA(cudaMalloc(&c->pieces, cap * sx::kDescQuads * sizeof(float4)));
    c->piece_cap = cap;
    return SX_OK;
}

// ====================================================================== C-ABI
extern "C" {

sx_status sx_create(sx_ctx** out, int32_t device) {
    if (!out) return SX_E_INVALID_ARG;
    *out = nullptr;
    int n_dev = 0;
    SX_CUDA(cudaGetDeviceCount(&n_dev));
    if (device < 0 || device >= n_dev) return SX_E_INVALID_ARG;
    SX_CUDA(cudaSetDevice(device));
    sx_ctx* c = static_cast<sx_ctx*>(calloc(1, sizeof(sx_ctx)));
    if (!c) return SX_E_INVALID_ARG;
    c->device = device;
    cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, device);
    if (c->sm_count <= 0) c->sm_count = 148;
    cudaError_t e = cudaMallocHost(reinterpret_cast<void**>(&c->h_pinned), 64);
    if (e != cudaSuccess) { g_last_cuda = e; free(c); return SX_E_CUDA; }
    e = cudaFuncSetAttribute(sx::k_write_pieces<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sx::kWpWarps * sizeof(sx::WarpTile)));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sx::k_write_pieces<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sx::kWpWarps * sizeof(sx::WarpTile)));
    if (e != cudaSuccess) { g_last_cuda = e; cudaFreeHost(c->h_pinned); free(c); return SX_E_CUDA; }
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->side_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming);
    if (e != cudaSuccess) { g_last_cuda = e; cudaFreeHost(c->h_pinned); free(c); return SX_E_CUDA; }
    *out = c;
    return SX_OK;
}

sx_status sx_destroy(sx_ctx* c) {
    if (!c) return SX_E_INVALID_ARG;
    cudaSetDevice(c->device);
    cudaDeviceSynchronize();
    cudaStreamDestroy(c->side_stream);
    cudaEventDestroy(c->ev_fork);
    cudaEventDestroy(c->ev_join);
    cudaFree(c->pt_off);
    cudaFree(c->pieces);
    cudaFree(c->sync_area);
    cudaFree(c->st_in);
    cudaFree(c->st_out);
    cudaFree(c->st_path);
    cudaFreeHost(c->h_pinned);
    free(c);
    return SX_OK;
}

sx_status sx_count(sx_ctx* c, const uint8_t* d_tags, uint64_t n_tags, const float* d_points_xy, uint64_t n_points,
                   const sx_style* d_styles, uint64_t n_paths, const float* h_affine, float tolerance, int32_t mode,
                   uint64_t* d_path_offsets, uint64_t* h_total, void* cuda_stream) {
    if (!c) return SX_E_INVALID_ARG;
    c->counted = false;
    if (!h_affine || !d_path_offsets) return SX_E_INVALID_ARG;
    if (!(tolerance > 0.0f) || !(tolerance < INFINITY)) return SX_E_INVALID_ARG;
    if (mode != SX_MODE_LINE && mode != SX_MODE_ARC) return SX_E_INVALID_ARG;
    if (n_tags >= (1ull << 32) - sx::kTagTile || n_points >= (1ull << 32) || n_paths > n_tags) return SX_E_INVALID_ARG;
    if (n_tags > 0 && (!d_tags || !d_points_xy || !d_styles)) return SX_E_INVALID_ARG;
    float det = h_affine[0] * h_affine[3] - h_affine[1] * h_affine[2];
    for (int k = 0; k < 6; k++)
        if (!(fabsf(h_affine[k]) < INFINITY)) return SX_E_INVALID_ARG;
    if (!(fabsf(det) < INFINITY) || det == 0.0f) return SX_E_INVALID_ARG;

    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    SX_CUDA(cudaSetDevice(c->device));
    sx_status rc = ensure_scratch(c, n_tags);
    if (rc != SX_OK) return rc;

    sx::Params& P = c->P;
    P.tags = d_tags; P.pts = d_points_xy; P.styles = reinterpret_cast<const uint8_t*>(d_styles);
    P.pt_off = c->pt_off; P.path_idx = c->path_idx; P.sp_first = c->sp_first;
    for (int k = 0; k < 6; k++) P.A[k] = h_affine[k];
    P.scale = sqrtf(fabsf(det));                 // R-14
    P.tol_es = 0.1f * tolerance;                 // R-13
    P.tol_fl = 0.8f * tolerance;
    P.mode = mode;
    P.n_tags = static_cast<uint32_t>(n_tags);
    c->n_paths = n_paths;
    c->total_known = false;
    c->cache_fits = false;
    c->total = 0;

    rc = ensure_pieces(c, 2 * n_tags + 4096);
    if (rc != SX_OK) return rc;
    for (int attempt = 0;; attempt++) {
        // reset the error flag, the tickets, the piece-cache counter, the total and the look-back states
        SX_CUDA(cudaMemsetAsync(c->sync_area, 0, c->sync_bytes, s));
        if (n_tags == 0) {
            SX_CUDA(cudaMemsetAsync(d_path_offsets, 0, 8, s));
        } else {
            uint32_t n = P.n_tags;
            uint32_t n_alloc_tiles = (n + sx::kCntTile - 1) / sx::kCntTile, n_tag_tiles = (n + sx::kTagTile - 1) / sx::kTagTile;
            uint64_t* alloc_states = reinterpret_cast<uint64_t*>(c->sync_area + 128);
            sx::TagTileState* tag_states = reinterpret_cast<sx::TagTileState*>(c->sync_area + 128 + round_up((uint64_t)(n_alloc_tiles + 1) * 8, 64));
            sx::k_tag_scan<<<n_tag_tiles, sx::kScanThreads, 0, s>>>(d_tags, n, (uint32_t)n_points, (uint32_t)n_paths, c->pt_off, c->path_idx,
                                                                   c->sp_first, c->curve_idx, ctx_n_curves(c), tag_states, ctx_ticket(c, 0), ctx_err(c));
            sx::k_count<<<(n + sx::kCntThreads - 1) / sx::kCntThreads, sx::kCntThreads, 0, s>>>(P, c->seg_count, c->curve_idx, ctx_n_curves(c), c->pieces, (uint32_t)c->piece_cap,
                                                                                              ctx_piece_ctr(c), ctx_side_stats(c), ctx_err(c));
            sx::k_alloc_scan<<<n_alloc_tiles, sx::kScanThreads, 0, s>>>(c->seg_count, n, d_tags, c->path_idx, (uint32_t)n_paths, c->seg_off,
                                                                      d_path_offsets, ctx_total(c), alloc_states, ctx_ticket(c, 1), ctx_err(c));
            c->launches += 3;
            SX_CUDA(cudaGetLastError());
        }
        c->counted = true;
        if (!h_total) break;  // asynchronous call: a cache overflow is handled on the device (k_write_segments)
        SX_CUDA(cudaMemcpyAsync(&c->h_pinned[0], ctx_total(c), 8, cudaMemcpyDeviceToHost, s));
        SX_CUDA(cudaMemcpyAsync(&c->h_pinned[1], ctx_err(c), 4, cudaMemcpyDeviceToHost, s));
        SX_CUDA(cudaMemcpyAsync(&c->h_pinned[2], ctx_piece_ctr(c), 4, cudaMemcpyDeviceToHost, s));
        SX_CUDA(cudaStreamSynchronize(s));
        uint32_t flags = static_cast<uint32_t>(c->h_pinned[1] & 0xffffffffu);
        uint64_t reserved = c->h_pinned[2] & 0xffffffffu;
        if (flags & sx::kErrBadStream) { c->counted = false; *h_total = 0; return SX_E_BAD_STREAM; }
        if (reserved > c->piece_cap && attempt == 0 && !(c->piece_limit && c->piece_cap >= c->piece_limit)) {
            // the piece cache was too small: size it from what this call needed and count again
            rc = ensure_pieces(c, reserved + reserved / 8 + 4096);
            if (rc != SX_OK) return rc;
            continue;
        }
        *h_total = c->h_pinned[0];
        c->total = c->h_pinned[0];
        c->total_known = true;
        c->cache_fits = reserved <= c->piece_cap;
        break;
    }
    return SX_OK;
}

sx_status sx_write(sx_ctx* c, void* d_out_records, uint64_t cap_records, void* cuda_stream) {
    if (!c) return SX_E_INVALID_ARG;
    if (!c->counted) return SX_E_STATE;
    if (c->total_known && c->total > cap_records) return SX_E_CAPACITY;
    if (c->P.n_tags == 0 || (c->total_known && c->total == 0)) return SX_OK;
    if (!d_out_records || (reinterpret_cast<uintptr_t>(d_out_records) & 15u)) return SX_E_INVALID_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    SX_CUDA(cudaSetDevice(c->device));
    uint32_t n = c->P.n_tags;
    float4* out = static_cast<float4*>(d_out_records);
    // the segment writer is bound by the latency of its dependent loads, the piece writer by instruction issue: they
    // run side by side (fork / join on events; everything stays ordered with respect to the caller's stream)
    SX_CUDA(cudaEventRecord(c->ev_fork, s));
    SX_CUDA(cudaStreamWaitEvent(c->side_stream, c->ev_fork, 0));
    sx::k_write_segments<<<(n + sx::kSegThreads - 1) / sx::kSegThreads, sx::kSegThreads, 0, c->side_stream>>>(
        c->P, c->seg_count, c->seg_off, out, cap_records, (uint32_t)c->piece_cap, ctx_piece_ctr(c), ctx_err(c));
    SX_CUDA(cudaEventRecord(c->ev_join, c->side_stream));
    sx::k_write_pieces<false><<<c->sm_count * sx::kWpBlocksPerSM, sx::kWpThreads, sx::kWpWarps * sizeof(sx::WarpTile), s>>>(
        c->P, c->pieces, (uint32_t)c->piece_cap, ctx_piece_ctr(c), ctx_side_stats(c), c->seg_off, out, cap_records, ctx_err(c));
    sx::k_write_pieces<true><<<c->sm_count * sx::kWpBlocksPerSM, sx::kWpThreads, sx::kWpWarps * sizeof(sx::WarpTile), s>>>(
        c->P, c->pieces, (uint32_t)c->piece_cap, ctx_piece_ctr(c), ctx_side_stats(c), c->seg_off, out, cap_records, ctx_err(c));
    SX_CUDA(cudaStreamWaitEvent(s, c->ev_join, 0));
    c->launches += 3;
    if (!c->cache_fits) {
        sx::k_write_fallback<<<(n + sx::kSegThreads - 1) / sx::kSegThreads, sx::kSegThreads, 0, s>>>(c->P, c->seg_count, c->seg_off, out, cap_records,
                                                                                                   (uint32_t)c->piece_cap, ctx_piece_ctr(c), ctx_err(c));
        c->launches += 1;
    }
    SX_CUDA(cudaGetLastError());
    return SX_OK;
}

sx_status stroke_expand(sx_ctx* c, const uint8_t* d_tags, uint64_t n_tags, const float* d_points_xy, uint64_t n_points,
                        const sx_style* d_styles, uint64_t n_paths, const float* h_affine, float tolerance, int32_t mode,
                        sx_alloc_fn alloc, void* user, void** d_out_records, uint64_t* h_n_records, uint64_t* d_path_offsets,
                        void* cuda_stream) {
    if (!alloc || !d_out_records || !h_n_records) return SX_E_INVALID_ARG;
    *d_out_records = nullptr;
    *h_n_records = 0;
    uint64_t total = 0;
    sx_status rc = sx_count(c, d_tags, n_tags, d_points_xy, n_points, d_styles, n_paths, h_affine, tolerance, mode, d_path_offsets, &total,
                            cuda_stream);
    if (rc != SX_OK) return rc;
    *h_n_records = total;
    if (total == 0) return SX_OK;
    uint64_t rec = mode == SX_MODE_ARC ? sizeof(sx_arc) : sizeof(sx_line);
    void* buf = alloc(total * rec, user);
    if (!buf) return SX_E_CAPACITY;
    *d_out_records = buf;
    return sx_write(c, buf, total, cuda_stream);
}

static sx_status grow(uint8_t** p, uint64_t* have, uint64_t need) {
    if (need <= *have) return SX_OK;
    if (*p) SX_CUDA(cudaFree(*p));
    *p = nullptr; *have = 0;
    uint64_t b = round_up(need + need / 8, 256);
    SX_CUDA(cudaMalloc(p, b));
    *have = b;
    return SX_OK;
}

sx_status stroke_expand_host(sx_ctx* c, const uint8_t* h_tags, uint64_t n_tags, const float* h_points_xy, uint64_t n_points,
                             const sx_style* h_styles, uint64_t n_paths, const float* h_affine, float tolerance, int32_t mode,
                             void* h_out_records, uint64_t cap_records, uint64_t* h_n_records, uint64_t* h_path_offsets,
                             void* cuda_stream) {
    if (!c || !h_n_records || !h_path_offsets) return SX_E_INVALID_ARG;
    if (n_tags > 0 && (!h_tags || !h_points_xy || !h_styles)) return SX_E_INVALID_ARG;
    *h_n_records = 0;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    SX_CUDA(cudaSetDevice(c->device));
    // staging layout: [tags | pad to 256][points][styles]
    uint64_t o_pts = round_up(n_tags, 256), o_sty = o_pts + round_up(n_points * 8, 256), in_bytes = o_sty + n_paths * 16 + 256;
    sx_status rc = grow(&c->st_in, &c->st_in_bytes, in_bytes);
    if (rc != SX_OK) return rc;
    uint64_t pbytes = (n_paths + 1) * 8;
    rc = grow(reinterpret_cast<uint8_t**>(&c->st_path), &c->st_path_n, pbytes);
    if (rc != SX_OK) return rc;
    if (n_tags > 0) {
        SX_CUDA(cudaMemcpyAsync(c->st_in, h_tags, n_tags, cudaMemcpyHostToDevice, s));
        SX_CUDA(cudaMemcpyAsync(c->st_in + o_pts, h_points_xy, n_points * 8, cudaMemcpyHostToDevice, s));
        SX_CUDA(cudaMemcpyAsync(c->st_in + o_sty, h_styles, n_paths * 16, cudaMemcpyHostToDevice, s));
    }
    uint64_t total = 0;
    rc = sx_count(c, c->st_in, n_tags, reinterpret_cast<const float*>(c->st_in + o_pts), n_points,
                  reinterpret_cast<const sx_style*>(c->st_in + o_sty), n_paths, h_affine, tolerance, mode, c->st_path, &total, s);
    if (rc != SX_OK) return rc;
    *h_n_records = total;
    SX_CUDA(cudaMemcpyAsync(h_path_offsets, c->st_path, pbytes, cudaMemcpyDeviceToHost, s));
    if (total > cap_records || (total > 0 && !h_out_records)) { cudaStreamSynchronize(s); return SX_E_CAPACITY; }
    uint64_t rec = mode == SX_MODE_ARC ? sizeof(sx_arc) : sizeof(sx_line);
    if (total > 0) {
        rc = grow(&c->st_out, &c->st_out_bytes, total * rec);
        if (rc != SX_OK) return rc;
        rc = sx_write(c, c->st_out, total, s);
        if (rc != SX_OK) return rc;
        SX_CUDA(cudaMemcpyAsync(h_out_records, c->st_out, total * rec, cudaMemcpyDeviceToHost, s));
    }
    SX_CUDA(cudaStreamSynchronize(s));
    return SX_OK;
}

sx_status sx_segment_info(sx_ctx* c, const uint32_t** d_pt_off, const uint32_t** d_path_idx, const uint32_t** d_sp_first,
                          const uint32_t** d_seg_count, const uint64_t** d_seg_offset) {
    if (!c) return SX_E_INVALID_ARG;
    if (!c->counted) return SX_E_STATE;
    if (d_pt_off) *d_pt_off = c->pt_off;
    if (d_path_idx) *d_path_idx = c->path_idx;
    if (d_sp_first) *d_sp_first = c->sp_first;
    if (d_seg_count) *d_seg_count = c->seg_count;
    if (d_seg_offset) *d_seg_offset = c->seg_off;
    return SX_OK;
}

sx_status sx_last_error(sx_ctx* c, void* cuda_stream) {
    if (!c) return SX_E_INVALID_ARG;
    if (!c->sync_area) return SX_OK;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    SX_CUDA(cudaSetDevice(c->device));
    SX_CUDA(cudaMemcpyAsync(&c->h_pinned[1], ctx_err(c), 4, cudaMemcpyDeviceToHost, s));
    SX_CUDA(cudaMemsetAsync(ctx_err(c), 0, 4, s));
    SX_CUDA(cudaStreamSynchronize(s));
    uint32_t flags = static_cast<uint32_t>(c->h_pinned[1] & 0xffffffffu);
    if (flags & sx::kErrBadStream) return SX_E_BAD_STREAM;
    if (flags & sx::kErrCapacity) return SX_E_CAPACITY;
    return SX_OK;
}

sx_status sx_set_piece_cache_limit(sx_ctx* c, uint64_t max_pieces) {
    if (!c) return SX_E_INVALID_ARG;
    cudaSetDevice(c->device);
    cudaDeviceSynchronize();
    c->piece_limit = max_pieces;
    if (max_pieces && c->piece_cap > max_pieces) {
        cudaFree(c->pieces);
        c->pieces = nullptr; c->piece_cap = 0;
    }
    c->counted = false;
    return SX_OK;
}

uint64_t sx_launch_count(const sx_ctx* c) { return c ? c->launches : 0; }

const char* sx_strerror(sx_status st) {
    switch (st) {
        case SX_OK: return "ok";
        case SX_E_INVALID_ARG: return "invalid argument";
        case SX_E_BAD_STREAM: return "malformed tag / point stream";
        case SX_E_CAPACITY: return "output capacity too small";
        case SX_E_CUDA: return cudaGetErrorString(g_last_cuda);
        case SX_E_STATE: return "sx_write without a successful sx_count";
        default: return "unknown status";
    }
}

}  // extern "C"
