/*
 * stroke_expand.h -- C-ABI of the B200 (sm_100a) stroke-expansion library.
 *
 * What the library computes: "GPU-friendly Stroke Expansion" (arxiv 2405.00127, PAPER.md): every
 * input path segment (line / quadratic / cubic Bezier, fp32) of a stroked path is expanded, fully in
 * parallel, into the records of a strongly-correct outline: the two parallel curves
 * at +-half-width flattened to lines (section 4) or circular arcs (section 5)
 * through an Euler-spiral intermediate (section 7, Alg. 2), evolute patches where curvature
 * exceeds 1/half-width (section 6), joins and caps (Alg. 1).
 *
 * Pipeline behind these calls: (a) tag-stream scan, then ONE kernel that runs (b) the
 * per-segment count, (c) the allocation scan and (d) the write with every intermediate result in shared memory.
 * All of it runs in hand-written CUDA kernels; there is no CPU path.
 *
 * Conventions
 *  - Every function returns an sx_status (0 = OK, < 0 = error).  No exception crosses the boundary.
 *  - Pointers named d_* are DEVICE pointers, h_* are HOST pointers.  The caller owns every buffer it
 *    passes; the library never frees caller memory.  The context owns its scratch buffers.
 *  - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls are
 *    asynchronous on that stream unless stated otherwise.
 *  - One sx_ctx serves one stream at a time (it holds the scratch of the call in flight).
 */
#ifndef STROKE_EXPAND_H
#define STROKE_EXPAND_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ------------------------------------------------------------------ status codes */
typedef int32_t sx_status;
enum {
    SX_OK = 0,
    SX_E_INVALID_ARG = -1, /* null pointer, size out of range, mode/tolerance/affine invalid           */
    SX_E_BAD_STREAM = -2,  /* malformed tag stream, detected on the device (see sx_count)              */
    SX_E_CAPACITY = -3,    /* output buffer smaller than the record count                              */
    SX_E_CUDA = -4,        /* a CUDA runtime call failed; sx_strerror gives cudaGetErrorString text    */
    SX_E_STATE = -5        /* sx_write without a preceding successful sx_count; sx_segment_info with nothing kept */
};

/* ------------------------------------------------------------------ input encoding (PAPER.md 8.2, L460-489)
 * Tag stream: one byte per input segment (Table 1):
 *   bits 0-1  coordinate count: 1 line, 2 quadratic, 3 cubic (0 is invalid)
 *   bit 2     subpath end: set on the last segment of a subpath
 *   bit 3     must be 0 (16-bit coordinates are not supported; fp32 only)
 *   bit 4     path end: set on the last segment of a path (implies subpath end)
 *   bits 5,6  ignored (one transform per call; the style is indexed by path)
 *   bit 7     closed subpath; meaningful on a subpath-end tag (reading R-8: the paper
 *             leaves bit 7 unused and does not say how open/closed reaches the shader).  The caller
 *             supplies the closing segment, as the paper's encoder does (L483); there is no
 *             stroke-cap-marker segment: the scan gives every segment its subpath's first segment.
 * Point stream (L464, L470, L483): float2.  Segment i reads points pt_off[i] .. pt_off[i]+count_i
 *   (its first point is the previous segment's last) and pt_off[i+1] = pt_off[i] + count_i +
 *   subpath_end_i.  A subpath of k segments owns 1 + sum(count) points.
 * Style: one per path.  half-width = width/2 * sqrt|det(affine)| (R-14).  width <= 0 or non-finite:
 *   the path emits no records (not an error) -- unless it is a FILL (style bit, below). */
typedef struct {
    float width;
    float miter_limit; /* SVG definition: miter used while 1/sin(beta/2) <= miter_limit              */
    uint8_t join;      /* SX_JOIN_*                                                                   */
    uint8_t cap;       /* SX_CAP_*                                                                    */
    uint16_t fill;     /* bit 0: FILL the path instead of stroking it (Alg. 1: "if style is fill then
                          flatten_cubic(segment, 0)"): its segments are flattened at offset 0, one record chain per
                          segment in path direction, an open subpath is closed by one line from its last point to its
                          first (kind SX_KIND_CLOSE); width, join, cap and miter_limit are ignored.
                          bit 1: the stroke is DASHED with the context's dash pattern (sx_set_dash)                   */
    uint32_t _rsv;
} sx_style; /* 16 bytes */

enum { SX_JOIN_MITER = 0, SX_JOIN_ROUND = 1, SX_JOIN_BEVEL = 2 };
enum { SX_CAP_BUTT = 0, SX_CAP_SQUARE = 1, SX_CAP_ROUND = 2 };
/* Output modes.  SX_MODE_LINE_REFINED ("If higher flattening quality is desired at the expense
 * of slower computation, this approximation could be used to determine a good initial value for numeric techniques; two
 * iterations of Newton solving are enough to refine this guess to within 32-bit floating point accuracy"): lines as in
 * SX_MODE_LINE, with the exact subdivision density integral f of L135-139 for the counts and f_approx_inv + two Newton steps
 * for the subdivision points; the flatten tolerance rises from 0.8 to 0.9 of `tolerance` (the 6 % of f_approx no longer needs
 * its margin; reading R-22 of DESIGN.md): 3-6 % fewer records of the same sx_line layout. */
enum { SX_MODE_LINE = 0, SX_MODE_ARC = 1, SX_MODE_LINE_REFINED = 2 };

/* ------------------------------------------------------------------ output records
 * Records are grouped by input segment, in segment order (hence by path); path_offsets[p] is the
 * index of path p's first record and path_offsets[n_paths] the total (this replaces the paper's
 * per-record 32-bit path id, L452-458).  Within a segment the order is canonical:
 * for every Euler-spiral piece in increasing t: [-h side, forward][+h side, mirrored]; then the
 * join [-h side][+h side], or on the last segment of an open subpath [end cap][start cap].
 * All outlines are positively oriented (winding numbers >= 0, L197). */
typedef struct { float x0, y0, x1, y1; } sx_line; /* SX_MODE_LINE: 16 bytes, one 16-byte store */

typedef struct {
    float x0, y0, x1, y1;
    float angle;   /* signed turning from start tangent to end tangent, CCW positive; 0 = straight.
                      (The paper stores curvature, L452: kappa = 2 sin(angle/2) / |p1 - p0|.)        */
    uint32_t seg;  /* source segment index                                                         */
    uint32_t kind; /* SX_KIND_* | SX_KIND_PLUS                                                     */
    uint32_t _pad;
} sx_arc; /* SX_MODE_ARC: 32 bytes, two 16-byte stores */

enum {
    SX_KIND_OFFSET = 0,     /* parallel curve, regular range                                          */
    SX_KIND_OFFSET_REV = 1, /* parallel curve over a super-critical range, reversed (L191, L403)      */
    SX_KIND_EVOLUTE = 2,    /* evolute, output twice (L197); arc mode: arcs by the metric of L171 (R-20) */
    SX_KIND_CONNECTOR = 3,  /* offset <-> evolute connecting line, output twice (L197)                */
    SX_KIND_JOIN_OUTER = 4,
    SX_KIND_JOIN_INNER = 5, /* through the vertex (strong correctness, L35)                           */
    SX_KIND_CAP = 6,
    SX_KIND_CLOSE = 7,      /* the line that closes an open subpath of a FILLED path (Alg. 1)   */
    SX_KIND_PLUS = 8        /* flag: record belongs to the +h side                                    */
};

/* ------------------------------------------------------------------ context */
typedef struct sx_ctx sx_ctx;

/* Create a context on CUDA device `device` (host-synchronous).  Fails with SX_E_CUDA when no usable
 * device exists: there is no CPU fallback. */
sx_status sx_create(sx_ctx** out, int32_t device);
/* Free the context and its scratch (host-synchronous). */
sx_status sx_destroy(sx_ctx* ctx);

/* ------------------------------------------------------------------ phase 1: scan + count + scan
 * Runs kernels (a) tag-stream scan, (b) the count pass -- the cubic -> Euler-spiral fit of Alg. 2
 * (L351-438) and the per-side subdivision counts (sections 4-6), which also leaves one 32-byte record per
 * Euler-spiral piece in the context's scratch -- and (c) the allocation scan over the per-segment counts (replaces the
 * atomic bump allocation of L448).  Use this pair of calls when the output buffer can only be allocated once the record
 * count is known; stroke_expand_into below issues both phases in one asynchronous call.
 *   d_tags[n_tags], d_points_xy[2*n_points], d_styles[n_paths]   device, read-only.  ALIGNMENT: d_tags and d_styles
 *                 16 bytes, d_points_xy and d_path_offsets 8 bytes (the kernels use vector loads); a pointer that
 *                 is not aligned so is rejected with SX_E_INVALID_ARG (a contiguous but offset tensor view can be)
 *   h_affine[6]   HOST, row-major a b c d e f:  x' = a x + c y + e,  y' = b x + d y + f (L462);
 *                 must be finite and non-singular
 *   tolerance     > 0, device px (L37).  Internally split 0.1 / 0.8 between the cubic->Euler-spiral
 *                 fit and the flattening (R-13)
 *   d_path_offsets[n_paths+1]  device, written: first record index of every path, then the total
 *   h_total       HOST, optional.  When non-NULL the call synchronises the stream, checks the
 *                 device-side stream validation and writes the record count; SX_E_BAD_STREAM is
 *                 returned here (coordinate count 0, bit 3 set, last tag without path end,
 *                 sum(count+end) != n_points, path-end count != n_paths).  When NULL the call stays
 *                 asynchronous and a bad stream yields zero records; sx_write reports the error.
 * n_tags, n_points < 2^32.  n_tags == 0 is valid only with n_paths == 0 (total = 0).
 * The input pointers must stay valid until the matching sx_write has completed. */
sx_status sx_count(sx_ctx* ctx, const uint8_t* d_tags, uint64_t n_tags, const float* d_points_xy, uint64_t n_points,
                   const sx_style* d_styles, uint64_t n_paths, const float* h_affine, float tolerance, int32_t mode,
                   uint64_t* d_path_offsets, uint64_t* h_total, void* cuda_stream);

/* ------------------------------------------------------------------ phase 2: write
 * Writes the records of the preceding sx_count into d_out_records (sx_line[] or sx_arc[] by mode, 16-byte
 * aligned; a 32-byte aligned buffer lets the kernels write an arc record in one 256-bit store) of capacity cap_records: kernels (d), the writers, which read the per-segment offsets and the piece
 * records phase 1 left (the fit is not repeated).  SX_E_CAPACITY if the capacity is known to be too small (the total
 * is known on the host only when sx_count was given h_total; otherwise the kernels themselves refuse to write past
 * the capacity and the error is reported by sx_last_error after a stream sync). */
sx_status sx_write(sx_ctx* ctx, void* d_out_records, uint64_t cap_records, void* cuda_stream);

/* ------------------------------------------------------------------ one call into a caller-provided buffer
 * The whole path -- kernels (a), (b), (c), (d) -- in one asynchronous call without a host round trip: Alg. 1 / Alg. 2
 * run once per segment.  Inputs as for sx_count.  d_out_records (16-byte aligned) has room for cap_records
 * records.  The count is always computed in full: a segment whose records would pass the capacity is not
 * written, the device-side capacity flag is raised (sx_last_error) and the total is still exact, so the caller can
 * retry with a buffer of that size.  h_total (HOST, optional): when non-NULL the call synchronises the stream,
 * writes the record count and returns SX_E_BAD_STREAM / SX_E_CAPACITY (count > cap_records) accordingly; when NULL
 * the call stays asynchronous (the count is d_path_offsets[n_paths]). */
sx_status stroke_expand_into(sx_ctx* ctx, const uint8_t* d_tags, uint64_t n_tags, const float* d_points_xy, uint64_t n_points,
                             const sx_style* d_styles, uint64_t n_paths, const float* h_affine, float tolerance, int32_t mode,
                             void* d_out_records, uint64_t cap_records, uint64_t* d_path_offsets, uint64_t* h_total,
                             void* cuda_stream);

/* ------------------------------------------------------------------ one-shot, device buffers
 * sx_count + allocate + sx_write.  `alloc` is called once (host side, after the count is known) and
 * must return a device pointer of at least `bytes` bytes, 16-byte aligned, valid on `cuda_stream`
 * (e.g. the torch caching allocator); NULL means allocation failure (SX_E_CAPACITY).  The result
 * buffer belongs to the caller.  Synchronises the stream once (to read the 8-byte total). */
typedef void* (*sx_alloc_fn)(uint64_t bytes, void* user);
sx_status stroke_expand(sx_ctx* ctx, const uint8_t* d_tags, uint64_t n_tags, const float* d_points_xy, uint64_t n_points,
                        const sx_style* d_styles, uint64_t n_paths, const float* h_affine, float tolerance, int32_t mode,
                        sx_alloc_fn alloc, void* user, void** d_out_records, uint64_t* h_n_records,
                        uint64_t* d_path_offsets, void* cuda_stream);

/* ------------------------------------------------------------------ one-shot, HOST buffers (end to end)
 * Same computation with every buffer on the host (pinned memory gives asynchronous copies): copies
 * the streams to the device, runs stroke_expand_into on a staging buffer owned by the context (a second time only
 * when that buffer had to grow), copies records and path offsets back.
 * h_out_records has room for cap_records records; *h_n_records receives the count even when
 * SX_E_CAPACITY is returned (so the caller can retry).  Returns after the results are in host memory. */
sx_status stroke_expand_host(sx_ctx* ctx, const uint8_t* h_tags, uint64_t n_tags, const float* h_points_xy, uint64_t n_points,
                             const sx_style* h_styles, uint64_t n_paths, const float* h_affine, float tolerance, int32_t mode,
                             void* h_out_records, uint64_t cap_records, uint64_t* h_n_records, uint64_t* h_path_offsets,
                             void* cuda_stream);

/* ------------------------------------------------------------------ tile binning of the line soup
 * PAPER.md L450 (section 8.1, Fig. 14): "the line soup elements are spatially sorted by subsequent compute stages
 * into a grid of 16x16 pixel tiles" -- the first stage of the tile-based renderer downstream of the stroke expansion.
 * The paper leaves the details out; the definition is reading R-19 of DESIGN.md: a coordinate v belongs to tile index
 * floor(v / 16); a record is binned, row of tiles by row, into the tiles its part inside the row's closed slab
 * 16 r <= y <= 16 r + 16 spans in x (fp32, one rounding per operation); rows / columns outside the viewport of
 * tiles_x x tiles_y tiles and records with a non-finite coordinate are skipped.
 *   d_lines[n_lines]            device, read-only, 16-byte aligned: sx_line records (e.g. the line-mode output above)
 *   d_tile_offsets[tiles + 1]   device, written: CSR offsets over the tiles in row-major order (tile = r * tiles_x + c);
 *                               the last entry is the number of (tile, record) pairs
 *   d_tile_lines[cap_entries]   device, written: per tile the indices of its records, in NO defined order (the soup is
 *                               unordered, L450).  cap_entries == 0: count and scan only (d_tile_lines may be NULL)
 *   h_total                     HOST, optional: when non-NULL the call synchronises the stream and writes the pair count;
 *                               SX_E_CAPACITY when it exceeds cap_entries (nothing is written past the capacity; the
 *                               device-side flag is raised either way, see sx_last_error) or 2^32 - 1
 * n_lines < 2^32, tiles_x * tiles_y < 2^31.  Asynchronous on cuda_stream unless h_total is given. */
sx_status sx_bin_lines(sx_ctx* ctx, const sx_line* d_lines, uint64_t n_lines, uint32_t tiles_x, uint32_t tiles_y,
                       uint32_t* d_tile_offsets, uint32_t* d_tile_lines, uint64_t cap_entries, uint64_t* h_total,
                       void* cuda_stream);

/* The same binning for callers that CANNOT ALLOCATE (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): no context, and the scratch (per-tile counters and cursors, look-back words of the scan) lives in a static
 * device array of SX_STATIC_SCRATCH_BYTES that every GPU loading the library holds until the process exits.  The call issues
 * memsets, kernels and one 4-byte device-to-device copy on cuda_stream and nothing else: no cudaMalloc, no cudaFree, no
 * allocating library routine, no host synchronisation.
 *   device                      the GPU the pointers belong to (made current by the call)
 *   d_lines, n_lines, tiles_x, tiles_y, d_tile_offsets, d_tile_lines, cap_entries: as for sx_bin_lines; the pair total is
 *                               d_tile_offsets[tiles_x * tiles_y] (device memory: read it after the stream has run)
 *   d_flags                     device, optional, one word written at the end of the call: 0, or SX_STATIC_FLAG_CAPACITY when
 *                               the pairs did not fit cap_entries or 32 bits (nothing is written past the capacity)
 * LIMIT: tiles_x * tiles_y <= SX_STATIC_MAX_TILES (a viewport of 4096 x 4096 px); larger viewports are rejected with
 * SX_E_INVALID_ARG (use sx_bin_lines).  All calls on one GPU share the static array, which keeps the last call's contents:
 * each call clears what it uses first, and calls that OVERLAP on a GPU (different streams or host threads) RACE on it --
 * serialise them.  Results are those of sx_bin_lines bit for bit (the offsets; a tile's records in no defined order). */
#define SX_STATIC_MAX_TILES 65536u
#define SX_STATIC_SCRATCH_BYTES 524672u
#define SX_STATIC_FLAG_CAPACITY 2u
sx_status sx_bin_lines_static(int32_t device, const sx_line* d_lines, uint64_t n_lines, uint32_t tiles_x, uint32_t tiles_y,
                              uint32_t* d_tile_offsets, uint32_t* d_tile_lines, uint64_t cap_entries, uint32_t* d_flags,
                              void* cuda_stream);

/* ------------------------------------------------------------------ introspection
 * Device pointers into the context's scratch of the last sx_count (valid until the next call on the
 * context): the tag-scan results and the per-segment record counts / offsets.  Any out pointer may
 * be NULL.  Used by the parity tests and the bench report.  SX_E_STATE before the first count. */
sx_status sx_segment_info(sx_ctx* ctx, const uint32_t** d_pt_off, const uint32_t** d_path_idx, const uint32_t** d_sp_first,
                          const uint32_t** d_seg_count, const uint64_t** d_seg_offset);

/* Device-side error state of the last call(s) on the context; synchronises `cuda_stream`. Returns
 * SX_OK, SX_E_BAD_STREAM or SX_E_CAPACITY and clears the state. */
sx_status sx_last_error(sx_ctx* ctx, void* cuda_stream);

/* Options of a context. */
enum {
    SX_OPT_KEEP_SEGMENT_INFO = 1, /* accepted and ignored: the per-segment counts / offsets are always kept              */
    SX_OPT_TIME_KERNELS = 3,      /* value != 0: the library records CUDA events around its kernels (sx_kernel_times)          */
    SX_OPT_TILE_SEGMENTS = 2      /* test knob for the count pass, whose warps work on tiles of 32, 16, 12, 8 or 4 segments
                                     (adapted on the device to what fits a warp's shared-memory tables): 0 adaptive
                                     (default); any value from 4 to 32 fixed; 2 = every tile is redone in sub-tiles of 8 segments
                                     (the path of a tile that overflowed); 1 = every tile takes the thread-per-segment
                                     reference walk.  The records do not depend on it (tests/test_gpu_parity.py).      */
};
sx_status sx_set_option(sx_ctx* ctx, int32_t option, uint64_t value);

/* Dashing on the GPU.  PAPER.md L543: "It is conceptually straightforward to implement on GPU; the core
 * algorithm is prefix sum applied to segment length, and the Euler spiral representation is particularly well suited";
 * L589: "... an approach based on parallel prefix sums of segment arc lengths".  The paper dashes on the CPU; the definition
 * used here is reading R-23 of DESIGN.md (also at the top of csrc/sx_dash.cuh):
 *   h_lengths[n]: n in {2, 4, 6, 8} positive lengths (on, off, on, off, ...), phase >= 0, in OUTPUT px (after the affine);
 *   host pointer, copied.  n = 0 clears the pattern.  SX_E_INVALID_ARG otherwise.
 * While a pattern is set, every stroked path whose style has bit 1 of `fill` set is dashed in the following sx_count /
 * stroke_expand* calls on this context: the pattern restarts at every subpath; arc length is that of the Euler-spiral pieces
 * (integers in units of 2^-16 px, summed by a parallel prefix sum); every dash is an open sub-stroke with the path's caps at
 * both ends, whose parts inside the pieces go through the same flattening as undashed pieces; joins are emitted where a dash
 * covers the junction; a closed subpath is dashed like an open one.  Record order within a segment: per piece, per dash
 * [start cap][-h side][+h side][end cap], then the join.  A dashed segment of 65536 px or more is refused (SX_E_BAD_STREAM).
 * Calls with a pattern set run the thread-per-segment kernels of csrc/sx_dash.cuh for all their paths. */
sx_status sx_set_dash(sx_ctx* ctx, const float* h_lengths, int32_t n, float phase);

/* Statistics of the last count pass on the context (synchronises `cuda_stream`): h_out4[0] tiles done in one
 * go from shared memory, [1] tiles redone in sub-tiles, [2] segments that took the thread-per-segment walk, [3] the
 * tile size (segments) of the call. */
sx_status sx_call_stats(sx_ctx* ctx, uint64_t* h_out4, void* cuda_stream);

/* Device durations of the kernels of the last stroke_expand_into call made under SX_OPT_TIME_KERNELS, from CUDA events
 * recorded on the call's own stream: h_ms4[0] tag scan (a), [1] count pass (b), [2] allocation scan (c), [3] the
 * writers (d).  Waits for the call to finish.  SX_E_STATE when nothing was timed. */
sx_status sx_kernel_times(sx_ctx* ctx, float* h_ms4);

/* Issue-rate microbenchmarks on `device` (host-synchronous, ~20 ms): h_out3[0] FP32 FMA lane-operations per second
 * (independent FFMA chains on all SMs), [1] issued lane-operations per second of an FFMA + integer-ALU mix, [2]
 * special-function (MUFU) lane-operations per second.  bench.py uses them as the measured R_fp32 / R_mufu of the
 * roofline. */
sx_status sx_measure_issue_peaks(int32_t device, double* h_out3);

/* Probes of single device functions of the kernels, for the tests (host buffers, host-synchronous, one thread per item):
 *   SX_EVAL_ATAN2       h_in[2 i] = y, h_in[2 i + 1] = x  ->  the kernels' angle function (reading R-17 of DESIGN.md: the fp32
 *                       value nearest to atan2(y, x), by an own double-precision evaluation)
 *   SX_EVAL_NODE_ERROR  h_in[9 i ..] = u0.x u0.y u1.x u1.y |q0| |q1| chord.x chord.y dt  ->  the decision-grade error estimate
 *                       of section 7.1 that Alg. 2's accept / split test uses
 *   SX_EVAL_F_EXACT     h_in[i] = x  ->  the density integral f(x) of L135-139 as SX_MODE_LINE_REFINED evaluates it
 *   SX_EVAL_F_INV_REFINED  h_in[i] = u  ->  its inverse: f_approx_inv(u) refined by two Newton steps (L145) */
enum { SX_EVAL_ATAN2 = 0, SX_EVAL_NODE_ERROR = 1, SX_EVAL_F_EXACT = 2, SX_EVAL_F_INV_REFINED = 3 };
sx_status sx_eval(int32_t device, int32_t what, const float* h_in, float* h_out, uint64_t n);

/* Number of kernel launches the library has issued on this context so far. */
uint64_t sx_launch_count(const sx_ctx* ctx);

/* Static text for a status code (for SX_E_CUDA: the last CUDA error string seen by this thread). */
const char* sx_strerror(sx_status status);

#ifdef __cplusplus
}
#endif
#endif /* STROKE_EXPAND_H */
