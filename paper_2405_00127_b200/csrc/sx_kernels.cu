// sx_kernels.cu -- the C-ABI of include/stroke_expand.h and the host side of the pipeline.
//
// Kernels, all on the caller's stream: (a) k_tag_scan, (b) k_count (fit + counts + leaf records), (c) k_alloc_scan
// (sx_scan.cuh, sx_count.cuh); (d) the four writers of sx_write.cuh.  The curve mathematics is in sx_math.cuh /
// sx_piece.cuh, the thread-per-segment reference walk in sx_segment.cuh, the part tables of the record-parallel writer in
// sx_cache.cuh.  sx_peaks.cuh: issue-rate microbenchmarks.
//
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -fmad=false -lineinfo -shared (see ../build.py).
// -fmad=false is part of the design: see the arithmetic discipline note in sx_math.cuh.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>

#include "../../include/stroke_expand.h"
#include "sx_write.cuh"
#include "sx_bin.cuh"
#include "sx_peaks.cuh"
#include "sx_refined.h"
#include "sx_dash.h"

// ====================================================================== host side
static thread_local cudaError_t g_last_cuda = cudaSuccess;
// (for the library's other translation units: sx_strerror(SX_E_CUDA) reports the last CUDA error of the calling thread)
void sx_internal_note_cuda_error(int e) { g_last_cuda = static_cast<cudaError_t>(e); }

#define SX_CUDA(call)                                      \
    do {                                                   \
        cudaError_t e_ = (call);                           \
        if (e_ != cudaSuccess) { g_last_cuda = e_; return SX_E_CUDA; } \
    } while (0)

constexpr int kSideStreams = 3;
constexpr int kEvents = 5;   // SX_OPT_TIME_KERNELS: before the tag scan, after it, after the count, after the allocation scan, after the writers

struct sx_ctx {
    int device;
    // scratch of the call in flight
    uint32_t *pt_off, *path_idx, *sp_first, *seg_count, *seg_tail, *walk_list;
    uint64_t* seg_off;
    uint64_t cap_segs;
    sx::LeafRec* leaves;  // the Euler-spiral pieces between the count pass and the writers (32 B each)
    uint64_t leaf_cap;
    double leaves_per_seg;  // the most a call on this context has needed so far (learned whenever a call reads its total)
    uint8_t* sync_area;   // [flags, tickets, statistics, counters: 128 B][d_total 128 B][look-back words of the allocation scan][tag tile states]
    uint64_t sync_bytes;
    uint32_t* d_hint;     // [0] tile size of the call in flight, [1] the one the last count pass proposed, [2] [3] its feedback state (adapted on the device, kept across calls)
    uint64_t* h_pinned;   // pinned: [0] total, [1] flags, [2..3] stats, [4] leaf counter
    int sm_count;
    int count_blocks, simple_blocks, general_blocks;   // persistent grids: resident blocks on the device
    cudaEvent_t ev[kEvents];
    bool time_kernels, timed;
    cudaStream_t side[kSideStreams];   // the writers are independent of one another: three of them run beside the caller's stream
    cudaEvent_t fork, join[kSideStreams];
    // options
    uint32_t force_tiles; // SX_OPT_TILE_SEGMENTS
    // last sx_count / stroke_expand_into
    sx::CountArgs C;
    sx::WriteArgs W;
    bool counted, total_known;
    uint64_t total;
    uint64_t launches;
    // dashing (sx_set_dash): the pattern in units of 2^-16 px; scratch [ticket, total: 64 B][look-back words][path offsets of
    // the length scan] and the per-segment arrays [seg_pos u64][sp_total u64][seg_len u32]
    uint32_t n_dash;
    unsigned long long dash_q[8], dash_period, dash_phase_q;
    uint8_t* dash_area; uint64_t dash_area_bytes;
    uint8_t* dash_buf; uint64_t dash_buf_segs;
    sx_dash_launch D;
    // scratch of sx_bin_lines: [ticket, total: 64 B][look-back words][tile counters][tile cursors]
    uint8_t* bin_area; uint64_t bin_bytes;
    // staging for stroke_expand_host
    uint8_t* st_in;  uint64_t st_in_bytes;
    uint8_t* st_out; uint64_t st_out_bytes;
    uint64_t* st_path; uint64_t st_path_n;
};

constexpr uint64_t kHeadBytes = 256;
static uint32_t* ctx_word(sx_ctx* c, int k) { return reinterpret_cast<uint32_t*>(c->sync_area) + k; }
static uint32_t* ctx_err(sx_ctx* c) { return ctx_word(c, 0); }
static uint32_t* ctx_ticket(sx_ctx* c, int k) { return ctx_word(c, 4 + 4 * k); }   // 0 tag scan, 1 count, 2 allocation scan
static uint32_t* ctx_stats(sx_ctx* c) { return ctx_word(c, 16); }                   // sx::kStWords words
static unsigned long long* ctx_leaf_counter(sx_ctx* c) { return reinterpret_cast<unsigned long long*>(ctx_word(c, 24)); }
static uint32_t* ctx_leaf_end_inv(sx_ctx* c) { return ctx_word(c, 26); }
static uint32_t* ctx_walk_count(sx_ctx* c) { return ctx_word(c, 28); }
static uint64_t* ctx_total(sx_ctx* c) { return reinterpret_cast<uint64_t*>(c->sync_area + 128); }
static uint64_t* ctx_states(sx_ctx* c) { return reinterpret_cast<uint64_t*>(c->sync_area + kHeadBytes); }

static uint64_t round_up(uint64_t x, uint64_t m) { return (x + m - 1) / m * m; }
static uint64_t states_bytes(uint64_t n) { return round_up(((n + sx::kCntTile - 1) / sx::kCntTile + 1) * 8, 64); }

static sx_status ensure_scratch(sx_ctx* c, uint64_t n) {
    uint64_t n_tag_tiles = (n + sx::kTagTile - 1) / sx::kTagTile + 1;
    uint64_t need_sync = kHeadBytes + states_bytes(n) + n_tag_tiles * sizeof(sx::TagTileState);
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
        // one allocation: 6 u32 arrays then the u64 offsets (all 256-byte aligned since cap % 64 == 0)
        uint8_t* p;
        SX_CUDA(cudaMalloc(&p, cap * (6 * 4 + 8)));
        c->pt_off = reinterpret_cast<uint32_t*>(p);
        c->path_idx = c->pt_off + cap;
        c->sp_first = c->path_idx + cap;
        c->seg_count = c->sp_first + cap;
        c->seg_tail = c->seg_count + cap;
        c->walk_list = c->seg_tail + cap;
        c->seg_off = reinterpret_cast<uint64_t*>(c->walk_list + cap);
        c->cap_segs = cap;
    }
    // leaf buffer: 4 pieces per segment to begin with, or what the scenes seen on this context needed (+ 15 %); a buffer
    // that turns out too small costs speed, not correctness (the tiles that find no room take the walk)
    double per_seg = c->leaves_per_seg * 1.15 > 4.0 ? c->leaves_per_seg * 1.15 : 4.0;
    uint64_t need_leaves = static_cast<uint64_t>(per_seg * static_cast<double>(n)) + 4096;
    if (need_leaves > 0xfffffff0ull) need_leaves = 0xfffffff0ull;
    if (need_leaves > c->leaf_cap) {
        if (c->leaves) SX_CUDA(cudaFree(c->leaves));
        c->leaves = nullptr; c->leaf_cap = 0;
        SX_CUDA(cudaMalloc(&c->leaves, need_leaves * sizeof(sx::LeafRec)));
        c->leaf_cap = need_leaves;
    }
    return SX_OK;
}

static sx_status check_inputs(const uint8_t* d_tags, uint64_t n_tags, const float* d_points_xy, uint64_t n_points, const sx_style* d_styles,
                              uint64_t n_paths, const float* h_affine, float tolerance, int32_t mode, const uint64_t* d_path_offsets) {
    if (!h_affine || !d_path_offsets) return SX_E_INVALID_ARG;
    if (!(tolerance > 0.0f) || !(tolerance < INFINITY)) return SX_E_INVALID_ARG;
    if (mode != SX_MODE_LINE && mode != SX_MODE_ARC && mode != SX_MODE_LINE_REFINED) return SX_E_INVALID_ARG;
    if (n_tags >= (1ull << 32) - sx::kTagTile || n_points >= (1ull << 32) || n_paths > n_tags) return SX_E_INVALID_ARG;
    if (n_tags > 0 && (!d_tags || !d_points_xy || !d_styles)) return SX_E_INVALID_ARG;
    // the kernels read tags and styles with 16-byte loads, points and offsets with 8-byte accesses
    if ((reinterpret_cast<uintptr_t>(d_tags) & 15u) || (reinterpret_cast<uintptr_t>(d_styles) & 15u) ||
        (reinterpret_cast<uintptr_t>(d_points_xy) & 7u) || (reinterpret_cast<uintptr_t>(d_path_offsets) & 7u))
        return SX_E_INVALID_ARG;
    float det = h_affine[0] * h_affine[3] - h_affine[1] * h_affine[2];
    for (int k = 0; k < 6; k++)
        if (!(fabsf(h_affine[k]) < INFINITY)) return SX_E_INVALID_ARG;
    if (!(fabsf(det) < INFINITY) || det == 0.0f) return SX_E_INVALID_ARG;
    return SX_OK;
}

// dashing: the stages before the allocation scan (the pattern was set with sx_set_dash)
static sx_status run_dash_count(sx_ctx* c, const uint8_t* d_tags, uint32_t n, uint64_t n_paths, cudaStream_t s) {
    const uint64_t st_bytes = states_bytes(n), head = 64;
    const uint64_t need_area = head + st_bytes + (n_paths + 1) * 8;
    if (need_area > c->dash_area_bytes) {
        if (c->dash_area) SX_CUDA(cudaFree(c->dash_area));
        c->dash_area = nullptr; c->dash_area_bytes = 0;
        SX_CUDA(cudaMalloc(&c->dash_area, round_up(need_area + need_area / 4, 256)));
        c->dash_area_bytes = round_up(need_area + need_area / 4, 256);
    }
    if (n > c->dash_buf_segs) {
        if (c->dash_buf) SX_CUDA(cudaFree(c->dash_buf));
        c->dash_buf = nullptr; c->dash_buf_segs = 0;
        const uint64_t cap = round_up(n + n / 8 + 64, 64);
        SX_CUDA(cudaMalloc(&c->dash_buf, cap * (4 + 8 + 8)));
        c->dash_buf_segs = cap;
    }
    SX_CUDA(cudaMemsetAsync(c->dash_area, 0, head + st_bytes, s));
    sx_dash_launch& D = c->D;
    D.params = &c->C.P;
    D.nd = c->n_dash;
    for (int k = 0; k < 8; k++) D.dq[k] = c->dash_q[k];
    D.period = c->dash_period; D.phase_q = c->dash_phase_q;
    D.seg_pos = reinterpret_cast<unsigned long long*>(c->dash_buf);
    D.sp_total = D.seg_pos + c->dash_buf_segs;
    D.seg_len = reinterpret_cast<uint32_t*>(D.sp_total + c->dash_buf_segs);
    D.seg_count = c->seg_count; D.seg_off = c->seg_off;
    D.out = nullptr; D.cap_records = 0; D.wide = 0; D.err = ctx_err(c);
    sxd_launch(0, &D, n, s);
    uint32_t tiles = (n + sx::kCntTile - 1) / sx::kCntTile;
    sx::k_alloc_scan<<<tiles, sx::kScanThreads, 0, s>>>(D.seg_len, n, d_tags, c->path_idx, (uint32_t)n_paths, reinterpret_cast<uint64_t*>(D.seg_pos),
                                                       reinterpret_cast<uint64_t*>(c->dash_area + head + st_bytes), reinterpret_cast<uint64_t*>(c->dash_area + 8),
                                                       reinterpret_cast<uint64_t*>(c->dash_area + head), reinterpret_cast<uint32_t*>(c->dash_area), ctx_err(c));
    sxd_launch(1, &D, n, s);
    sxd_launch(2, &D, n, s);
    c->launches += 3;   // (+ the count launch the caller books)
    return SX_OK;
}

// phase 1: resets the per-call device state and runs (a) the tag scan, (b) the count pass, (c) the allocation scan
static sx_status run_count(sx_ctx* c, const uint8_t* d_tags, uint64_t n_tags, const float* d_points_xy, uint64_t n_points,
                           const sx_style* d_styles, uint64_t n_paths, const float* h_affine, float tolerance, int32_t mode,
                           uint64_t* d_path_offsets, cudaStream_t s) {
    SX_CUDA(cudaSetDevice(c->device));
    sx_status rc = ensure_scratch(c, n_tags);
    if (rc != SX_OK) return rc;
    sx::CountArgs& C = c->C;
    sx::Params& P = C.P;
    P.tags = d_tags; P.pts = d_points_xy; P.styles = reinterpret_cast<const uint8_t*>(d_styles);
    P.pt_off = c->pt_off; P.path_idx = c->path_idx; P.sp_first = c->sp_first;
    for (int k = 0; k < 6; k++) P.A[k] = h_affine[k];
    float det = h_affine[0] * h_affine[3] - h_affine[1] * h_affine[2];
    P.scale = sqrtf(fabsf(det));                 // R-14
    P.tol_es = 0.1f * tolerance;                 // R-13
    P.tol_fl = (mode == SX_MODE_LINE_REFINED ? 0.9f : 0.8f) * tolerance;   // R-22: the 6 % of f_approx no longer needs its margin
    P.mode = mode;
    P.n_tags = static_cast<uint32_t>(n_tags);
    C.n_paths = static_cast<uint32_t>(n_paths);
    C.ticket = ctx_ticket(c, 1);
    C.err = ctx_err(c);
    C.seg_count = c->seg_count; C.seg_tail = c->seg_tail;
    C.leaves = c->leaves; C.leaf_cap = static_cast<uint32_t>(c->leaf_cap);
    C.leaf_counter = ctx_leaf_counter(c); C.leaf_end_inv = ctx_leaf_end_inv(c);
    C.walk_list = c->walk_list; C.walk_count = ctx_walk_count(c);
    C.stats = ctx_stats(c);
    C.hint = c->d_hint;
    C.force = c->force_tiles;
    sx::WriteArgs& W = c->W;
    W.P = P;
    W.seg_count = c->seg_count; W.seg_tail = c->seg_tail; W.seg_off = c->seg_off;
    W.leaves = c->leaves; W.leaf_cap = C.leaf_cap; W.leaf_counter = C.leaf_counter; W.leaf_end_inv = C.leaf_end_inv;
    W.walk_list = c->walk_list; W.walk_count = C.walk_count;
    W.out = nullptr; W.cap_records = 0; W.err = C.err;
    c->total_known = false;
    c->total = 0;
    c->timed = false;
    // error flag, tickets, statistics, counters, total, look-back words of both scans
    SX_CUDA(cudaMemsetAsync(c->sync_area, 0, c->sync_bytes, s));
    if (n_tags == 0) {
        SX_CUDA(cudaMemsetAsync(d_path_offsets, 0, 8, s));
        return SX_OK;
    }
    uint32_t n = P.n_tags;
    if (c->time_kernels) SX_CUDA(cudaEventRecord(c->ev[0], s));
    uint32_t n_tag_tiles = (n + sx::kTagTile - 1) / sx::kTagTile;
    sx::TagTileState* tag_states = reinterpret_cast<sx::TagTileState*>(c->sync_area + kHeadBytes + states_bytes(n));
    sx::k_tag_scan<<<n_tag_tiles, sx::kScanThreads, 0, s>>>(d_tags, n, (uint32_t)n_points, (uint32_t)n_paths, c->pt_off, c->path_idx, c->sp_first,
                                                           tag_states, ctx_ticket(c, 0), ctx_err(c), c->d_hint);
    if (c->time_kernels) SX_CUDA(cudaEventRecord(c->ev[1], s));
    // persistent one-warp blocks: no more of them than there are tiles of the smallest size
    uint64_t tiles = (n + sx::kCtTileMin - 1) / sx::kCtTileMin;
    unsigned grid = (unsigned)(tiles < (uint64_t)c->count_blocks ? tiles : (uint64_t)c->count_blocks);
    if (c->n_dash) {
        // dashing (sx_dash.cuh): arc lengths, their prefix sum, subpath totals, then the count with the pattern
        sx_status rd = run_dash_count(c, d_tags, n, n_paths, s);
        if (rd != SX_OK) return rd;
    } else if (mode == SX_MODE_LINE_REFINED) sxr_launch_count(&C, grid, s);   // (sx_refined.cu: the same kernel with the refined density integral)
    else sx::k_count<<<grid, 32, sizeof(sx::CtWarp), s>>>(C);
    if (c->time_kernels) SX_CUDA(cudaEventRecord(c->ev[2], s));
    uint32_t n_cnt_tiles = (n + sx::kCntTile - 1) / sx::kCntTile;
    sx::k_alloc_scan<<<n_cnt_tiles, sx::kScanThreads, 0, s>>>(c->seg_count, n, d_tags, c->path_idx, (uint32_t)n_paths, c->seg_off, d_path_offsets,
                                                             ctx_total(c), ctx_states(c), ctx_ticket(c, 2), ctx_err(c));
    if (c->time_kernels) SX_CUDA(cudaEventRecord(c->ev[3], s));
    c->launches += 3;
    SX_CUDA(cudaGetLastError());
    return SX_OK;
}

// phase 2: (d) the writers
static sx_status run_write(sx_ctx* c, void* d_out_records, uint64_t cap_records, cudaStream_t s) {
    uint32_t n = c->W.P.n_tags;
    if (n == 0) return SX_OK;
    c->W.out = static_cast<float4*>(d_out_records);
    c->W.cap_records = cap_records;
    c->W.wide = (reinterpret_cast<uintptr_t>(d_out_records) & 31u) == 0u ? 1u : 0u;
    // the four writers side by side: the general writer (the long one on evolute-heavy scenes) on the caller's stream, the
    // others on the context's side streams, forked from and joined to the caller's stream with events
    SX_CUDA(cudaEventRecord(c->fork, s));
    for (int k = 0; k < kSideStreams; k++) SX_CUDA(cudaStreamWaitEvent(c->side[k], c->fork, 0));
    const unsigned segment_blocks = (n + sx::kWrThreads - 1) / sx::kWrThreads;
    if (c->n_dash) {   // dashing: one writer, thread per segment (sx_dash.cuh)
        c->D.out = d_out_records; c->D.cap_records = cap_records; c->D.wide = c->W.wide;
        sxd_launch(3, &c->D, n, s);
        c->launches += 1;
        if (c->time_kernels) { SX_CUDA(cudaEventRecord(c->ev[4], s)); c->timed = true; }
        SX_CUDA(cudaGetLastError());
        return SX_OK;
    }
    if (c->W.P.mode == SX_MODE_LINE_REFINED) {
        sxr_launch_writers(&c->W, c->general_blocks, c->simple_blocks, segment_blocks, c->sm_count, s, c->side[0], c->side[1], c->side[2]);
    } else {
        sx::k_write_general<<<c->general_blocks, sx::kWrThreads, 0, s>>>(c->W);
        sx::k_write_simple<<<c->simple_blocks, sx::kWrThreads, 0, c->side[0]>>>(c->W);
        sx::k_write_segments<<<segment_blocks, sx::kWrThreads, 0, c->side[1]>>>(c->W);
        sx::k_write_walk<<<c->sm_count, sx::kWrThreads, 0, c->side[2]>>>(c->W);
    }
    for (int k = 0; k < kSideStreams; k++) {
        SX_CUDA(cudaEventRecord(c->join[k], c->side[k]));
        SX_CUDA(cudaStreamWaitEvent(s, c->join[k], 0));
    }
    c->launches += 4;
    if (c->time_kernels) { SX_CUDA(cudaEventRecord(c->ev[4], s)); c->timed = true; }
    SX_CUDA(cudaGetLastError());
    return SX_OK;
}

// synchronises and reads total + device flags; SX_E_BAD_STREAM / SX_OK
static sx_status read_total(sx_ctx* c, cudaStream_t s, uint64_t* h_total) {
    SX_CUDA(cudaMemcpyAsync(&c->h_pinned[0], ctx_total(c), 8, cudaMemcpyDeviceToHost, s));
    SX_CUDA(cudaMemcpyAsync(&c->h_pinned[1], ctx_err(c), 4, cudaMemcpyDeviceToHost, s));
    SX_CUDA(cudaMemcpyAsync(&c->h_pinned[4], ctx_leaf_counter(c), 8, cudaMemcpyDeviceToHost, s));
    SX_CUDA(cudaStreamSynchronize(s));
    uint32_t flags = static_cast<uint32_t>(c->h_pinned[1] & 0xffffffffu);
    if (flags & sx::kErrBadStream) { *h_total = 0; return SX_E_BAD_STREAM; }
    *h_total = c->h_pinned[0];
    c->total = c->h_pinned[0];
    c->total_known = true;
    // how many pieces the scene has per segment: sizes the leaf buffer of the calls that follow
    uint64_t leaves = (c->h_pinned[4] & 0xffffffffull) + (c->h_pinned[4] >> 32);
    if (c->C.P.n_tags > 0) {
        double per_seg = static_cast<double>(leaves) / static_cast<double>(c->C.P.n_tags);
        if (per_seg > c->leaves_per_seg) c->leaves_per_seg = per_seg;
    }
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
    e = cudaMalloc(&c->d_hint, 64);
    uint32_t first[16] = {(uint32_t)sx::kCtTile, (uint32_t)sx::kCtTile};   // [2] the share of the tables (float bits, 0: unset), [3] pieces per segment last seen
    if (e == cudaSuccess) e = cudaMemcpy(c->d_hint, first, 64, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sx::k_count, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(sx::CtWarp));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sx::k_count, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    int per_sm = 0;
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, sx::k_count, 32, sizeof(sx::CtWarp));
    c->count_blocks = c->sm_count * (per_sm > 0 ? per_sm : 1);
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, sx::k_write_simple, sx::kWrThreads, 0);
    c->simple_blocks = c->sm_count * (per_sm > 0 ? per_sm : 1);
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, sx::k_write_general, sx::kWrThreads, 0);
    c->general_blocks = c->sm_count * (per_sm > 0 ? per_sm : 1);
    for (int k = 0; k < kEvents && e == cudaSuccess; k++) e = cudaEventCreate(&c->ev[k]);
    for (int k = 0; k < kSideStreams && e == cudaSuccess; k++) {
        e = cudaStreamCreateWithFlags(&c->side[k], cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->join[k], cudaEventDisableTiming);
    }
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->fork, cudaEventDisableTiming);
    if (e != cudaSuccess) { g_last_cuda = e; cudaFree(c->d_hint); cudaFreeHost(c->h_pinned); free(c); return SX_E_CUDA; }
    *out = c;
    return SX_OK;
}

sx_status sx_destroy(sx_ctx* c) {
    if (!c) return SX_E_INVALID_ARG;
    cudaSetDevice(c->device);
    cudaDeviceSynchronize();
    for (int k = 0; k < kEvents; k++) cudaEventDestroy(c->ev[k]);
    for (int k = 0; k < kSideStreams; k++) { cudaStreamDestroy(c->side[k]); cudaEventDestroy(c->join[k]); }
    cudaEventDestroy(c->fork);
    cudaFree(c->pt_off);
    cudaFree(c->leaves);
    cudaFree(c->sync_area);
    cudaFree(c->d_hint);
    cudaFree(c->bin_area);
    cudaFree(c->dash_area);
    cudaFree(c->dash_buf);
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
    sx_status rc = check_inputs(d_tags, n_tags, d_points_xy, n_points, d_styles, n_paths, h_affine, tolerance, mode, d_path_offsets);
    if (rc != SX_OK) return rc;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    rc = run_count(c, d_tags, n_tags, d_points_xy, n_points, d_styles, n_paths, h_affine, tolerance, mode, d_path_offsets, s);
    if (rc != SX_OK) return rc;
    c->counted = true;
    if (!h_total) return SX_OK;
    rc = read_total(c, s, h_total);
    if (rc != SX_OK) c->counted = false;
    return rc;
}

sx_status sx_write(sx_ctx* c, void* d_out_records, uint64_t cap_records, void* cuda_stream) {
    if (!c) return SX_E_INVALID_ARG;
    if (!c->counted) return SX_E_STATE;
    if (c->total_known && c->total > cap_records) return SX_E_CAPACITY;
    if (c->W.P.n_tags == 0 || (c->total_known && c->total == 0)) return SX_OK;
    if (!d_out_records || (reinterpret_cast<uintptr_t>(d_out_records) & 15u)) return SX_E_INVALID_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    SX_CUDA(cudaSetDevice(c->device));
    return run_write(c, d_out_records, cap_records, s);
}

sx_status stroke_expand_into(sx_ctx* c, const uint8_t* d_tags, uint64_t n_tags, const float* d_points_xy, uint64_t n_points,
                             const sx_style* d_styles, uint64_t n_paths, const float* h_affine, float tolerance, int32_t mode,
                             void* d_out_records, uint64_t cap_records, uint64_t* d_path_offsets, uint64_t* h_total, void* cuda_stream) {
    if (!c) return SX_E_INVALID_ARG;
    c->counted = false;
    sx_status rc = check_inputs(d_tags, n_tags, d_points_xy, n_points, d_styles, n_paths, h_affine, tolerance, mode, d_path_offsets);
    if (rc != SX_OK) return rc;
    if (cap_records > 0 && (!d_out_records || (reinterpret_cast<uintptr_t>(d_out_records) & 15u))) return SX_E_INVALID_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    rc = run_count(c, d_tags, n_tags, d_points_xy, n_points, d_styles, n_paths, h_affine, tolerance, mode, d_path_offsets, s);
    if (rc != SX_OK) return rc;
    c->counted = true;
    if (cap_records > 0) {
        rc = run_write(c, d_out_records, cap_records, s);
        if (rc != SX_OK) return rc;
    }
    if (!h_total) return SX_OK;
    rc = read_total(c, s, h_total);
    if (rc != SX_OK) return rc;
    return *h_total > cap_records ? SX_E_CAPACITY : SX_OK;
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
    // One pass into the device staging buffer as it stands (sized by earlier calls, or a first guess of 16 records per
    // segment, never more than the caller's capacity); when the records do not fit, the buffer grows to the count the
    // pass returned and the pass runs again.
    uint64_t rec = mode == SX_MODE_ARC ? sizeof(sx_arc) : sizeof(sx_line);
    uint64_t total = 0;
    for (int attempt = 0; attempt < 2; attempt++) {
        uint64_t want = attempt == 0 ? (c->st_out_bytes ? c->st_out_bytes / rec : 16 * n_tags + 1024) : total;
        if (want > cap_records) want = cap_records;
        rc = grow(&c->st_out, &c->st_out_bytes, want * rec);
        if (rc != SX_OK) return rc;
        uint64_t cap_dev = c->st_out_bytes / rec < cap_records ? c->st_out_bytes / rec : cap_records;
        rc = stroke_expand_into(c, c->st_in, n_tags, reinterpret_cast<const float*>(c->st_in + o_pts), n_points,
                                reinterpret_cast<const sx_style*>(c->st_in + o_sty), n_paths, h_affine, tolerance, mode, c->st_out, cap_dev,
                                c->st_path, &total, s);
        if (rc != SX_E_CAPACITY) break;
        *h_n_records = total;
        if (total > cap_records) return SX_E_CAPACITY;   // the caller's buffer is too small: the count is reported
        sx_last_error(c, s);                             // (clears the device-side capacity flag before the second pass)
    }
    if (rc != SX_OK) return rc;
    *h_n_records = total;
    SX_CUDA(cudaMemcpyAsync(h_path_offsets, c->st_path, pbytes, cudaMemcpyDeviceToHost, s));
    if (total > 0) {
        if (!h_out_records) { cudaStreamSynchronize(s); return SX_E_CAPACITY; }
        SX_CUDA(cudaMemcpyAsync(h_out_records, c->st_out, total * rec, cudaMemcpyDeviceToHost, s));
    }
    SX_CUDA(cudaStreamSynchronize(s));
    return SX_OK;
}

sx_status sx_bin_lines(sx_ctx* c, const sx_line* d_lines, uint64_t n_lines, uint32_t tiles_x, uint32_t tiles_y, uint32_t* d_tile_offsets,
                       uint32_t* d_tile_lines, uint64_t cap_entries, uint64_t* h_total, void* cuda_stream) {
    if (!c || !d_tile_offsets) return SX_E_INVALID_ARG;
    if (n_lines >= (1ull << 32) || tiles_x == 0 || tiles_y == 0 || (uint64_t)tiles_x * tiles_y >= (1ull << 31)) return SX_E_INVALID_ARG;
    if (n_lines > 0 && (!d_lines || (reinterpret_cast<uintptr_t>(d_lines) & 15u))) return SX_E_INVALID_ARG;
    if (cap_entries > 0 && !d_tile_lines) return SX_E_INVALID_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    SX_CUDA(cudaSetDevice(c->device));
    sx_status rc = ensure_scratch(c, 0);   // (the error flag lives in the context's sync area)
    if (rc != SX_OK) return rc;
    const uint32_t tiles = tiles_x * tiles_y;
    const uint32_t scan_tiles = (tiles + sx::kScan32Tile - 1) / sx::kScan32Tile;
    const uint64_t o_states = 64, o_counts = o_states + round_up((uint64_t)(scan_tiles + 1) * 8, 64), o_cursor = o_counts + round_up((uint64_t)tiles * 4, 64);
    const uint64_t need = o_cursor + round_up((uint64_t)tiles * 4, 64);
    rc = grow(&c->bin_area, &c->bin_bytes, need);
    if (rc != SX_OK) return rc;
    uint32_t* ticket = reinterpret_cast<uint32_t*>(c->bin_area);
    uint64_t* d_total = reinterpret_cast<uint64_t*>(c->bin_area + 8);
    uint64_t* states = reinterpret_cast<uint64_t*>(c->bin_area + o_states);
    uint32_t* counts = reinterpret_cast<uint32_t*>(c->bin_area + o_counts);
    uint32_t* cursor = reinterpret_cast<uint32_t*>(c->bin_area + o_cursor);
    SX_CUDA(cudaMemsetAsync(c->bin_area, 0, need, s));
    const float4* lines = reinterpret_cast<const float4*>(d_lines);
    const uint64_t want = (n_lines + sx::kBinThreads - 1) / sx::kBinThreads;
    const unsigned grid = (unsigned)(want < (uint64_t)c->sm_count * 16 ? (want ? want : 1) : (uint64_t)c->sm_count * 16);
    sx::k_bin_walk<false><<<grid, sx::kBinThreads, 0, s>>>(lines, n_lines, tiles_x, tiles_y, counts, nullptr, nullptr, 0, ctx_err(c));
    sx::k_scan_u32<<<scan_tiles, sx::kScanThreads, 0, s>>>(counts, tiles, d_tile_offsets, d_total, states, ticket, ctx_err(c));
    c->launches += 2;
    if (cap_entries > 0) {
        sx::k_bin_walk<true><<<grid, sx::kBinThreads, 0, s>>>(lines, n_lines, tiles_x, tiles_y, cursor, d_tile_offsets, d_tile_lines, cap_entries, ctx_err(c));
        c->launches += 1;
    }
    SX_CUDA(cudaGetLastError());
    if (!h_total) return SX_OK;
    SX_CUDA(cudaMemcpyAsync(&c->h_pinned[5], d_total, 8, cudaMemcpyDeviceToHost, s));
    SX_CUDA(cudaStreamSynchronize(s));
    *h_total = c->h_pinned[5];
    return (*h_total > cap_entries || (*h_total >> 32)) ? SX_E_CAPACITY : SX_OK;
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

sx_status sx_set_dash(sx_ctx* c, const float* h_lengths, int32_t n, float phase) {
    if (!c) return SX_E_INVALID_ARG;
    if (n == 0) { c->n_dash = 0; return SX_OK; }
    if (!h_lengths || n < 2 || n > 8 || (n & 1) || !(phase >= 0.0f) || !isfinite(phase)) return SX_E_INVALID_ARG;
    for (int k = 0; k < n; k++) if (!(h_lengths[k] > 0.0f) || !isfinite(h_lengths[k])) return SX_E_INVALID_ARG;
    c->dash_period = 0;
    for (int k = 0; k < 8; k++) c->dash_q[k] = 0;
    for (int k = 0; k < n; k++) {
        c->dash_q[k] = (unsigned long long)llrintf(h_lengths[k] * 65536.0f);   // units of 2^-16 px (R-23)
        if (c->dash_q[k] == 0) c->dash_q[k] = 1;
        c->dash_period += c->dash_q[k];
    }
    c->dash_phase_q = (unsigned long long)llrintf(phase * 65536.0f);
    c->n_dash = (uint32_t)n;
    return SX_OK;
}

sx_status sx_set_option(sx_ctx* c, int32_t option, uint64_t value) {
    if (!c) return SX_E_INVALID_ARG;
    switch (option) {
        case SX_OPT_KEEP_SEGMENT_INFO: return SX_OK;   // (kept for compatibility: the per-segment results are always there)
        case SX_OPT_TIME_KERNELS: c->time_kernels = value != 0; c->timed = false; return SX_OK;
        case SX_OPT_TILE_SEGMENTS:
            if (value != 0 && value != 1 && value != 2 && (value < 4 || value > 32)) return SX_E_INVALID_ARG;
            c->force_tiles = static_cast<uint32_t>(value);
            return SX_OK;
        default: return SX_E_INVALID_ARG;
    }
}

sx_status sx_call_stats(sx_ctx* c, uint64_t* h_out4, void* cuda_stream) {
    if (!c || !h_out4) return SX_E_INVALID_ARG;
    for (int k = 0; k < 4; k++) h_out4[k] = 0;
    if (!c->sync_area) return SX_OK;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    SX_CUDA(cudaSetDevice(c->device));
    uint32_t* hp = reinterpret_cast<uint32_t*>(&c->h_pinned[2]);
    SX_CUDA(cudaMemcpyAsync(hp, ctx_stats(c), 12, cudaMemcpyDeviceToHost, s));
    SX_CUDA(cudaMemcpyAsync(hp + 3, c->d_hint, 4, cudaMemcpyDeviceToHost, s));
    SX_CUDA(cudaStreamSynchronize(s));
    h_out4[0] = hp[0]; h_out4[1] = hp[1]; h_out4[2] = hp[2]; h_out4[3] = c->force_tiles >= 4 ? c->force_tiles : hp[3];
    return SX_OK;
}

sx_status sx_kernel_times(sx_ctx* c, float* h_ms4) {
    if (!c || !h_ms4) return SX_E_INVALID_ARG;
    for (int k = 0; k < 4; k++) h_ms4[k] = 0.0f;
    if (!c->timed) return SX_E_STATE;
    SX_CUDA(cudaSetDevice(c->device));
    SX_CUDA(cudaEventSynchronize(c->ev[kEvents - 1]));
    for (int k = 0; k < 4; k++) SX_CUDA(cudaEventElapsedTime(&h_ms4[k], c->ev[k], c->ev[k + 1]));
    return SX_OK;
}

// probes of single device functions (tests): one thread per item
__global__ void k_eval(int what, const float* in, float* out, uint64_t n) {
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    if (what == SX_EVAL_ATAN2) {
        out[i] = sx::atan2_r(in[2 * i], in[2 * i + 1]);
    } else if (what == SX_EVAL_NODE_ERROR) {
        const float* v = in + 9 * i;
        out[i] = sx::node_error(sx::v2(v[0], v[1]), sx::v2(v[2], v[3]), v[4], v[5], sx::v2(v[6], v[7]), v[8]);
    }
}

sx_status sx_eval(int32_t device, int32_t what, const float* h_in, float* h_out, uint64_t n) {
    if (!h_in || !h_out || what < SX_EVAL_ATAN2 || what > SX_EVAL_F_INV_REFINED) return SX_E_INVALID_ARG;
    if (n == 0) return SX_OK;
    const uint64_t per = what == SX_EVAL_ATAN2 ? 2 : (what == SX_EVAL_NODE_ERROR ? 9 : 1);
    SX_CUDA(cudaSetDevice(device));
    float *d_in = nullptr, *d_out = nullptr;
    SX_CUDA(cudaMalloc(&d_in, n * per * sizeof(float)));
    cudaError_t e = cudaMalloc(&d_out, n * sizeof(float));
    if (e == cudaSuccess) e = cudaMemcpy(d_in, h_in, n * per * sizeof(float), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        if (what >= SX_EVAL_F_EXACT) sxr_launch_eval(what, d_in, d_out, n);
        else k_eval<<<(unsigned)((n + 255) / 256), 256>>>(what, d_in, d_out, n);
        e = cudaMemcpy(h_out, d_out, n * sizeof(float), cudaMemcpyDeviceToHost);
    }
    cudaFree(d_in);
    cudaFree(d_out);
    if (e != cudaSuccess) { g_last_cuda = e; return SX_E_CUDA; }
    return SX_OK;
}

sx_status sx_measure_issue_peaks(int32_t device, double* h_out3) {
    if (!h_out3) return SX_E_INVALID_ARG;
    cudaError_t e = sx::measure_issue_peaks(device, h_out3);
    if (e != cudaSuccess) { g_last_cuda = e; return SX_E_CUDA; }
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
        case SX_E_STATE: return "call out of order (sx_write without sx_count, or no per-segment results kept)";
        default: return "unknown status";
    }
}

}  // extern "C"
