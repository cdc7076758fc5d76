// sx_bin.cuh -- tile binning of the line soup: count -> scan -> scatter over the records the stroke
// expansion wrote (line mode), the first stage of a tile-based renderer downstream (Fig. 14: "the line
// soup elements are spatially sorted by subsequent compute stages into a grid of 16x16 pixel tiles"; the paper leaves the
// details out, reading R-19 of DESIGN.md fixes them).
//
// Definition (R-19).  A coordinate v belongs to tile index floor(v / 16).  A record (x0, y0, x1, y1) is binned, row of
// tiles by row, into the tiles its part inside the row's closed slab 16 r <= y <= 16 r + 16 spans in x; the x-extent is
// evaluated in fp32 -- slope by one IEEE division, x = x0 + (y - y0) s with separate multiply and add (-fmad=false),
// clamped to the record's own x-range -- because it decides integers: the CPU oracle takes the same operations and the
// comparison is bit-exact.  Rows and columns outside the viewport, and records with a non-finite coordinate, are skipped.
//
// Kernels: k_bin_walk<false> (thread per record: one atomic add per (tile, record) pair on the tile's counter),
// k_scan_u32 (exclusive scan of the counters: CSR offsets, decoupled look-back as in sx_scan.cuh), k_bin_walk<true> (the
// same walk; a pair's slot is the tile's offset plus a ticket from the tile's cursor).  The order of a tile's records is
// the order the tickets came in: not defined (the soup is unordered, L450).  Bound: HBM / L2 atomics -- 16 B read per
// record twice, 4 B written per pair, 12 B per tile.
#pragma once
#include "sx_scan.cuh"

namespace sx {

constexpr int kBinThreads = 256;
constexpr float kTilePx = 16.0f, kInvTilePx = 0.0625f;

template <bool SCATTER>
__global__ void __launch_bounds__(kBinThreads)
k_bin_walk(const float4* __restrict__ lines, uint64_t n, uint32_t tiles_x, uint32_t tiles_y, uint32_t* __restrict__ counter,
           const uint32_t* __restrict__ offsets, uint32_t* __restrict__ out, uint64_t cap, uint32_t* err) {
    for (uint64_t i = (uint64_t)blockIdx.x * kBinThreads + threadIdx.x; i < n; i += (uint64_t)gridDim.x * kBinThreads) {
        const float4 l = __ldg(lines + i);
        const float x0 = l.x, y0 = l.y, x1 = l.z, y1 = l.w;
        if (!(fabsf(x0) < INFINITY) || !(fabsf(y0) < INFINITY) || !(fabsf(x1) < INFINITY) || !(fabsf(y1) < INFINITY)) continue;
        const float ya = fminf(y0, y1), yb = fmaxf(y0, y1), xmin = fminf(x0, x1), xmax = fmaxf(x0, x1);
        const float fr0 = floorf(ya * kInvTilePx), fr1 = floorf(yb * kInvTilePx);
        if (fr1 < 0.0f || fr0 >= (float)tiles_y || xmax < 0.0f || floorf(xmin * kInvTilePx) >= (float)tiles_x) continue;
        const uint32_t r0 = fr0 < 0.0f ? 0u : (uint32_t)fr0;
        const uint32_t r1 = fr1 >= (float)tiles_y ? tiles_y - 1u : (uint32_t)fr1;
        const bool horizontal = y0 == y1;
        const float s = horizontal ? 0.0f : (x1 - x0) / (y1 - y0);
        for (uint32_t r = r0; r <= r1; r++) {
            const float top = (float)r * kTilePx, bot = top + kTilePx;
            const float ylo = fmaxf(ya, top), yhi = fminf(yb, bot);
            float xlo = xmin, xhi = xmax;
            if (!horizontal) {
                const float xa = x0 + (ylo - y0) * s, xb = x0 + (yhi - y0) * s;
                xlo = fmaxf(fminf(xa, xb), xmin);
                xhi = fminf(fmaxf(xa, xb), xmax);
            }
            const float fc0 = floorf(xlo * kInvTilePx), fc1 = floorf(xhi * kInvTilePx);
            if (fc1 < 0.0f || fc0 >= (float)tiles_x) continue;
            const uint32_t c0 = fc0 < 0.0f ? 0u : (uint32_t)fc0;
            const uint32_t c1 = fc1 >= (float)tiles_x ? tiles_x - 1u : (uint32_t)fc1;
            for (uint32_t c = c0; c <= c1; c++) {
                const uint32_t t = r * tiles_x + c;
                const uint32_t k = atomicAdd(counter + t, 1u);
                if (SCATTER) {
                    const uint64_t pos = (uint64_t)offsets[t] + k;
                    if (pos < cap) out[pos] = (uint32_t)i;
                    else atomicOr(err, kErrCapacity);
                }
            }
        }
    }
}

// exclusive scan of n 32-bit counters: out[0 .. n - 1], the total in out[n] and (64-bit) in *d_total; the capacity flag is
// raised when the total does not fit 32 bits
constexpr int kScan32Items = 8;
constexpr int kScan32Tile = kScanThreads * kScan32Items;
__global__ void __launch_bounds__(kScanThreads)
k_scan_u32(const uint32_t* __restrict__ in, uint32_t n, uint32_t* __restrict__ out, uint64_t* d_total, uint64_t* states, uint32_t* ticket, uint32_t* err) {
    __shared__ uint32_t s_tile;
    __shared__ uint64_t s_warp[kScanThreads / 32];
    __shared__ uint64_t s_prefix;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    const uint32_t base = tile * (uint32_t)kScan32Tile + (uint32_t)tid * kScan32Items;
    uint32_t c[kScan32Items];
#pragma unroll
    for (int k = 0; k < kScan32Items; k++) c[k] = base + k < n ? in[base + k] : 0u;
    uint64_t mine = 0;
#pragma unroll
    for (int k = 0; k < kScan32Items; k++) mine += c[k];
    uint64_t incl = mine;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint64_t o = __shfl_up_sync(0xffffffffu, incl, d);
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
        if (lane == 0) {
            s_prefix = excl;
            *reinterpret_cast<volatile uint64_t*>(states + tile) = (2ull << 62) | (excl + tile_agg);
        }
    }
    __syncthreads();
    uint64_t up = __shfl_up_sync(0xffffffffu, incl, 1);
    if (lane == 0) up = 0;
    uint64_t run = s_prefix + warp_excl + up;
#pragma unroll
    for (int k = 0; k < kScan32Items; k++) {
        const uint32_t i = base + k;
        if (i < n) {
            out[i] = (uint32_t)run;
            run += c[k];
            if (i == n - 1u) {
                out[n] = (uint32_t)run;
                *d_total = run;
                if (run >> 32) atomicOr(err, kErrCapacity);
            }
        }
    }
}

}  // namespace sx
