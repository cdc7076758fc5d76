/*
 * bin_oracle.c -- CPU ORACLE for the tile binning of the line soup.
 *
 * TEST INFRASTRUCTURE ONLY (same rules as stroke_oracle.c: only tests/, __graft_entry__.smoke() and bench.py's CPU
 * legs may build, load or call it; it shares no code with paper_2405_00127_b200/csrc/).
 *
 * What it computes.  PAPER.md L450 (section 8.1): "the line soup elements are spatially sorted by subsequent compute
 * stages into a grid of 16x16 pixel tiles" (Fig. 14); the paper gives no more than that ("the details of which are
 * beyond the scope of this paper").  Reading R-19 of DESIGN.md fixes the definition:
 *
 *   The viewport is the grid of tiles_x x tiles_y tiles of 16 x 16 px; a coordinate v belongs to tile index floor(v / 16)
 *   (tile (r, c) is the half-open square [16 c, 16 c + 16) x [16 r, 16 r + 16)).  A line record (x0, y0, x1, y1) is binned,
 *   row of tiles by row, into the tiles its part inside that row's CLOSED slab 16 r <= y <= 16 r + 16 spans in x:
 *     ya = min(y0, y1), yb = max(y0, y1); rows floor(ya / 16) .. floor(yb / 16), restricted to the viewport;
 *     in row r: ylo = max(ya, 16 r), yhi = min(yb, 16 r + 16);
 *               y0 == y1:  [xlo, xhi] = [min(x0, x1), max(x0, x1)];
 *               otherwise: s = (x1 - x0) / (y1 - y0), xa = x0 + (ylo - y0) s, xb = x0 + (yhi - y0) s,
 *                          [xlo, xhi] = [min(xa, xb), max(xa, xb)] clamped to [min(x0, x1), max(x0, x1)];
 *               columns floor(xlo / 16) .. floor(xhi / 16), restricted to the viewport.
 *   All of it in fp32, one rounding per operation, no fused multiply-add (compile with -ffp-contract=off): this decides
 *   integers, so the kernel takes the same operations in the same order and the comparison is bit-exact.  A record with a
 *   non-finite coordinate is binned nowhere.
 *   Result: tile_offsets[tiles + 1] (CSR over tiles in row-major order) and, per tile, the indices of the records binned
 *   into it -- here in increasing order; the order within a tile is not part of the definition (the soup is unordered, L450).
 *
 * The set is conservative (every half-open tile the segment passes through is listed: each row's x-extent is that of the
 * exact sub-segment of the closed slab, up to ~1 ulp) and tight (a tile is listed only if the segment comes within rounding
 * distance of its closed square: the closed slab adds at most the tiles the segment touches at a grid line);
 * tests/test_oracle_binning.py pins both against the exact geometry.
 */
#define _GNU_SOURCE
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

#define TILE 16.0f
#define INV_TILE 0.0625f

typedef void (*tile_fn)(uint32_t tile, uint32_t line, void* user);

static void walk_line(const float* l, uint32_t line, uint32_t tiles_x, uint32_t tiles_y, tile_fn f, void* user) {
    float x0 = l[0], y0 = l[1], x1 = l[2], y1 = l[3];
    if (!isfinite(x0) || !isfinite(y0) || !isfinite(x1) || !isfinite(y1)) return;
    float ya = fminf(y0, y1), yb = fmaxf(y0, y1), xmin = fminf(x0, x1), xmax = fmaxf(x0, x1);
    float fr0 = floorf(ya * INV_TILE), fr1 = floorf(yb * INV_TILE);
    if (fr1 < 0.0f || fr0 >= (float)tiles_y || xmax < 0.0f || floorf(xmin * INV_TILE) >= (float)tiles_x) return;
    uint32_t r0 = fr0 < 0.0f ? 0u : (uint32_t)fr0;
    uint32_t r1 = fr1 >= (float)tiles_y ? tiles_y - 1u : (uint32_t)fr1;
    int horizontal = (y0 == y1);
    float s = horizontal ? 0.0f : (x1 - x0) / (y1 - y0);
    for (uint32_t r = r0; r <= r1; r++) {
        float top = (float)r * TILE, bot = top + TILE;
        float ylo = fmaxf(ya, top), yhi = fminf(yb, bot);
        float xlo = xmin, xhi = xmax;
        if (!horizontal) {
            float xa = x0 + (ylo - y0) * s, xb = x0 + (yhi - y0) * s;
            xlo = fmaxf(fminf(xa, xb), xmin);
            xhi = fminf(fmaxf(xa, xb), xmax);
        }
        float fc0 = floorf(xlo * INV_TILE), fc1 = floorf(xhi * INV_TILE);
        if (fc1 < 0.0f || fc0 >= (float)tiles_x) continue;
        uint32_t c0 = fc0 < 0.0f ? 0u : (uint32_t)fc0;
        uint32_t c1 = fc1 >= (float)tiles_x ? tiles_x - 1u : (uint32_t)fc1;
        for (uint32_t c = c0; c <= c1; c++) f(r * tiles_x + c, line, user);
    }
}

typedef struct { uint32_t* counts; uint32_t* offsets; uint32_t* cursor; uint32_t* out; } bin_state;
static void count_cb(uint32_t tile, uint32_t line, void* user) { (void)line; ((bin_state*)user)->counts[tile]++; }
static void fill_cb(uint32_t tile, uint32_t line, void* user) {
    bin_state* b = (bin_state*)user;
    b->out[b->offsets[tile] + b->cursor[tile]++] = line;
}

/* lines: n x 4 floats.  tile_offsets: tiles + 1 entries (written).  Returns the total number of (tile, line) pairs; when
 * tile_lines is non-NULL (room for that many entries) it is filled, every tile's lines in increasing order. */
uint64_t bo_bin_lines(const float* lines, uint64_t n, uint32_t tiles_x, uint32_t tiles_y, uint32_t* tile_offsets, uint32_t* tile_lines) {
    uint64_t tiles = (uint64_t)tiles_x * tiles_y;
    bin_state b;
    b.counts = (uint32_t*)calloc(tiles + 1, sizeof(uint32_t));
    b.cursor = (uint32_t*)calloc(tiles + 1, sizeof(uint32_t));
    b.offsets = tile_offsets;
    b.out = tile_lines;
    for (uint64_t i = 0; i < n; i++) walk_line(lines + 4 * i, (uint32_t)i, tiles_x, tiles_y, count_cb, &b);
    uint64_t run = 0;
    for (uint64_t t = 0; t < tiles; t++) { tile_offsets[t] = (uint32_t)run; run += b.counts[t]; }
    tile_offsets[tiles] = (uint32_t)run;
    if (tile_lines)
        for (uint64_t i = 0; i < n; i++) walk_line(lines + 4 * i, (uint32_t)i, tiles_x, tiles_y, fill_cb, &b);
    free(b.counts);
    free(b.cursor);
    return run;
}
