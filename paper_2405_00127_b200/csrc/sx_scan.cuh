// sx_scan.cuh -- (a) k_tag_scan and (c) k_alloc_scan: single-pass prefix scans (decoupled look-back).
//
// PAPER.md L464-466 + Table 1 (L468-481): every tag carries stream-offset increments and the offsets are prefix
// sums over the "tag monoid".  Ours is (points, paths, first) with points += count + subpath_end (L470),
// paths += path_end, first = max(index+1 of subpath ends): the exclusive prefix gives segment i its first point,
// its path and the first segment of its subpath (which replaces the paper's stroke-cap-marker segment, L483-489).
//
// One pass over the data, thread-sequential -> warp-shuffle -> cross-warp in shared memory -> tile prefix by
// decoupled look-back (a tile publishes its aggregate, then looks back over its predecessors' aggregates /
// inclusive prefixes, one warp inspecting 32 predecessors at a time).  Tile ids come from an atomic ticket, so a
// tile only ever waits for tiles that already started.  (c) k_alloc_scan, the allocation scan over the record counts
// (replacing the atomic bump allocation of L448), uses the same protocol.
#pragma once
#include <stdint.h>
#include <cuda_runtime.h>

namespace sx {

constexpr int kScanThreads = 256;
constexpr int kTagItems = 16;                         // tags per thread: one 16-byte load
constexpr int kTagTile = kScanThreads * kTagItems;    // 4096

enum : uint32_t { kErrBadStream = 1u, kErrCapacity = 2u };

struct TagAgg { uint32_t pt, path, first; };
__device__ __forceinline__ TagAgg tag_identity() { TagAgg a; a.pt = 0; a.path = 0; a.first = 0; return a; }
__device__ __forceinline__ TagAgg tag_combine(TagAgg a, TagAgg b) {
    TagAgg r; r.pt = a.pt + b.pt; r.path = a.path + b.path; r.first = a.first > b.first ? a.first : b.first; return r;
}
__device__ __forceinline__ TagAgg tag_shfl_up(TagAgg a, int d) {
    TagAgg r; r.pt = __shfl_up_sync(0xffffffffu, a.pt, d); r.path = __shfl_up_sync(0xffffffffu, a.path, d);
    r.first = __shfl_up_sync(0xffffffffu, a.first, d); return r;
}
__device__ __forceinline__ TagAgg tag_shfl_xor(TagAgg a, int d) {
    TagAgg r; r.pt = __shfl_xor_sync(0xffffffffu, a.pt, d); r.path = __shfl_xor_sync(0xffffffffu, a.path, d);
    r.first = __shfl_xor_sync(0xffffffffu, a.first, d); return r;
}

// look-back descriptor of one tag tile: status 0 = nothing yet, 1 = aggregate valid, 2 = inclusive valid
struct __align__(16) TagTileState { uint32_t status, pad0, pad1, pad2; uint4 agg; uint4 inc; };

__device__ __forceinline__ uint32_t ld_volatile_u32(const uint32_t* p) { return *reinterpret_cast<const volatile uint32_t*>(p); }
__device__ __forceinline__ uint64_t ld_volatile_u64(const uint64_t* p) { return *reinterpret_cast<const volatile uint64_t*>(p); }

__global__ void __launch_bounds__(kScanThreads)
k_tag_scan(const uint8_t* __restrict__ tags, uint32_t n, uint32_t n_points, uint32_t n_paths, uint32_t* __restrict__ pt_off,
           uint32_t* __restrict__ path_idx, uint32_t* __restrict__ sp_first, TagTileState* states, uint32_t* ticket, uint32_t* err, uint32_t* hint) {
    __shared__ uint32_t s_tile;
    __shared__ TagAgg s_warp[kScanThreads / 32];
    __shared__ TagAgg s_prefix;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    // the first kernel of every call: the tile size the last expansion kernel proposed becomes the one of this call
    // (k_count reads hint[0] only)
    if (blockIdx.x == 0 && tid == 0) hint[0] = hint[1];
    __syncthreads();
    const uint32_t tile = s_tile;
    const uint32_t base = tile * (uint32_t)kTagTile + (uint32_t)tid * kTagItems;

    // ---- load 16 tags (identity beyond n)
    uint32_t w[4] = {0u, 0u, 0u, 0u};
    if (base + kTagItems <= n) {
        uint4 v = __ldg(reinterpret_cast<const uint4*>(tags + base));
        w[0] = v.x; w[1] = v.y; w[2] = v.z; w[3] = v.w;
    } else {
        for (int k = 0; k < kTagItems; k++)
            if (base + k < n) w[k >> 2] |= (uint32_t)tags[base + k] << (8 * (k & 3));
    }
    // ---- thread-sequential reduce + validation (Table 1: count 0 invalid, bit 3 unsupported)
    TagAgg mine = tag_identity();
    bool bad = false;
#pragma unroll
    for (int k = 0; k < kTagItems; k++) {
        uint32_t tag = (w[k >> 2] >> (8 * (k & 3))) & 0xffu;
        uint32_t cnt = tag & 3u, end = ((tag >> 2) | (tag >> 4)) & 1u;
        bool valid = base + k < n;
        bad |= valid && (cnt == 0u || (tag & 8u));
        mine.pt += cnt + end;
        mine.path += (tag >> 4) & 1u;
        if (end) mine.first = base + k + 1u;
    }
    if (bad) atomicOr(err, kErrBadStream);
    // ---- warp inclusive scan by shuffles, cross-warp through shared memory
    TagAgg incl = mine;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        TagAgg o = tag_shfl_up(incl, d);
        if (lane >= d) incl = tag_combine(o, incl);
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    TagAgg tile_agg = tag_identity(), warp_excl = tag_identity();
#pragma unroll
    for (int k = 0; k < kScanThreads / 32; k++) {
        if (k == warp) warp_excl = tile_agg;
        tile_agg = tag_combine(tile_agg, s_warp[k]);
    }
    // ---- decoupled look-back (warp 0)
    if (warp == 0) {
        TagTileState* me = states + tile;
        if (lane == 0 && tile > 0) {
            me->agg = make_uint4(tile_agg.pt, tile_agg.path, tile_agg.first, 0u);
            __threadfence();
            *reinterpret_cast<volatile uint32_t*>(&me->status) = 1u;
        }
        TagAgg excl = tag_identity();
        int idx = (int)tile - 1;
        while (idx >= 0) {
            int j = idx - lane;
            uint32_t st = 2u;
            if (j >= 0) { do { st = ld_volatile_u32(&states[j].status); } while (st == 0u); }
            __threadfence();
            TagAgg v = tag_identity();
            if (j >= 0) {
                const volatile uint4* src = st == 2u ? &states[j].inc : &states[j].agg;
                v.pt = src->x; v.path = src->y; v.first = src->z;
            }
            uint32_t m = __ballot_sync(0xffffffffu, st == 2u);
            int stop = __ffs((int)m) - 1;  // nearest predecessor with an inclusive prefix (lanes with j < 0 report 2)
            if (m && lane > stop) v = tag_identity();
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) v = tag_combine(v, tag_shfl_xor(v, d));
            excl = tag_combine(v, excl);
            if (m) break;
            idx -= 32;
        }
        if (lane == 0) {
            s_prefix = excl;
            TagAgg inc = tag_combine(excl, tile_agg);
            me->inc = make_uint4(inc.pt, inc.path, inc.first, 0u);
            __threadfence();
            *reinterpret_cast<volatile uint32_t*>(&me->status) = 2u;
        }
    }
    __syncthreads();
    // ---- exclusive prefix of this thread's first tag, then the 16 outputs
    TagAgg up = tag_shfl_up(incl, 1);
    if (lane == 0) up = tag_identity();
    TagAgg run = tag_combine(tag_combine(s_prefix, warp_excl), up);
    uint32_t o_pt[kTagItems], o_path[kTagItems], o_first[kTagItems];
#pragma unroll
    for (int k = 0; k < kTagItems; k++) {
        uint32_t tag = (w[k >> 2] >> (8 * (k & 3))) & 0xffu;
        uint32_t cnt = tag & 3u, end = ((tag >> 2) | (tag >> 4)) & 1u;
        o_pt[k] = run.pt; o_path[k] = run.path; o_first[k] = run.first;
        run.pt += cnt + end;
        run.path += (tag >> 4) & 1u;
        if (end) run.first = base + k + 1u;
    }
    if (base + kTagItems <= n) {
#pragma unroll
        for (int k = 0; k < kTagItems; k += 4) {
            *reinterpret_cast<uint4*>(pt_off + base + k) = make_uint4(o_pt[k], o_pt[k + 1], o_pt[k + 2], o_pt[k + 3]);
            *reinterpret_cast<uint4*>(path_idx + base + k) = make_uint4(o_path[k], o_path[k + 1], o_path[k + 2], o_path[k + 3]);
            *reinterpret_cast<uint4*>(sp_first + base + k) = make_uint4(o_first[k], o_first[k + 1], o_first[k + 2], o_first[k + 3]);
        }
    } else {
#pragma unroll
        for (int k = 0; k < kTagItems; k++)
            if (base + k < n) { pt_off[base + k] = o_pt[k]; path_idx[base + k] = o_path[k]; sp_first[base + k] = o_first[k]; }
    }
    // ---- whole-stream checks by the thread that owns the last tag (run = inclusive total there)
    if (base < n && n - base <= (uint32_t)kTagItems) {
        uint32_t k = n - 1u - base;
        uint32_t last = (w[k >> 2] >> (8 * (k & 3))) & 0xffu;
        if (!(last & 16u) || run.pt != n_points || run.path != n_paths) atomicOr(err, kErrBadStream);
    }
}

// ---------------------------------------------------------------- (c) allocation scan
// Exclusive 64-bit prefix sum of the per-segment record counts (replaces the atomic bump allocation of PAPER.md L448: the
// records come out grouped by segment, in segment order), the offset of every path's first record and the total.
// Same single-pass protocol as the tag scan; state word: status in bits 62-63 (0 nothing, 1 aggregate, 2 inclusive),
// value in bits 0-61.
constexpr uint64_t kValMask = (1ull << 62) - 1ull;
constexpr int kCntItems = 8;
constexpr int kCntTile = kScanThreads * kCntItems;    // 2048

__global__ void __launch_bounds__(kScanThreads)
k_alloc_scan(const uint32_t* __restrict__ count, uint32_t n, const uint8_t* __restrict__ tags, const uint32_t* __restrict__ path_idx,
             uint32_t n_paths, uint64_t* __restrict__ seg_off, uint64_t* __restrict__ path_off, uint64_t* d_total, uint64_t* states,
             uint32_t* ticket, const uint32_t* err) {
    __shared__ uint32_t s_tile;
    __shared__ uint64_t s_warp[kScanThreads / 32];
    __shared__ uint64_t s_prefix;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    const uint32_t base = tile * (uint32_t)kCntTile + (uint32_t)tid * kCntItems;
    uint32_t c[kCntItems];
    if (base + kCntItems <= n) {
        uint4 a = __ldg(reinterpret_cast<const uint4*>(count + base)), b = __ldg(reinterpret_cast<const uint4*>(count + base + 4));
        c[0] = a.x; c[1] = a.y; c[2] = a.z; c[3] = a.w; c[4] = b.x; c[5] = b.y; c[6] = b.z; c[7] = b.w;
    } else {
#pragma unroll
        for (int k = 0; k < kCntItems; k++) c[k] = base + k < n ? count[base + k] : 0u;
    }
    uint64_t mine = 0;
#pragma unroll
    for (int k = 0; k < kCntItems; k++) mine += c[k];
    uint64_t incl = mine;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        uint64_t o = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += o;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    uint64_t tile_agg = 0, warp_excl = 0;
#pragma unroll
    for (int k = 0; k < kScanThreads / 32; k++) {
        if (k == warp) warp_excl = tile_agg;
        tile_agg += s_warp[k];
    }
    if (warp == 0) {
        if (lane == 0 && tile > 0) *reinterpret_cast<volatile uint64_t*>(states + tile) = (1ull << 62) | tile_agg;
        uint64_t excl = 0;
        int idx = (int)tile - 1;
        while (idx >= 0) {
            int j = idx - lane;
            uint64_t word = 2ull << 62;
            if (j >= 0) { do { word = ld_volatile_u64(states + j); } while ((word >> 62) == 0ull); }
            uint32_t m = __ballot_sync(0xffffffffu, (word >> 62) == 2ull);
            int stop = __ffs((int)m) - 1;
            uint64_t v = (lane > stop && m) ? 0ull : (word & kValMask);
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
            excl += v;
            if (m) break;
            idx -= 32;
        }
        if (lane == 0) {
            s_prefix = excl;
            *reinterpret_cast<volatile uint64_t*>(states + tile) = (2ull << 62) | (excl + tile_agg);
        }
    }
    __syncthreads();
    uint64_t up = __shfl_up_sync(0xffffffffu, incl, 1);
    if (lane == 0) up = 0;
    uint64_t run = s_prefix + warp_excl + up;
    const bool ok = (*err & kErrBadStream) == 0u;
#pragma unroll
    for (int k = 0; k < kCntItems; k++) {
        uint32_t i = base + k;
        if (i < n) {
            seg_off[i] = run;
            // first segment of a path: the previous tag carries the path-end bit (Table 1)
            if (ok && (i == 0u || (tags[i - 1] & 16u))) { uint32_t p = path_idx[i]; if (p < n_paths) path_off[p] = run; }
            run += c[k];
            if (i == n - 1u) { path_off[n_paths] = run; *d_total = run; }
        }
    }
}

}  // namespace sx
