// sx_kernels.cu -- count kernel (b), write kernel (d) and the C-ABI of include/stroke_expand.h.
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
#include "sx_segment.cuh"

namespace sx {

constexpr int kSegThreads = 128;

// (b) count pass: one thread per input segment runs Alg. 2 without the writes
__global__ void __launch_bounds__(kSegThreads)
k_count(Params P, uint32_t* __restrict__ seg_count, const uint32_t* __restrict__ err) {
    uint32_t i = blockIdx.x * (uint32_t)kSegThreads + threadIdx.x;
    if (i >= P.n_tags) return;
    uint32_t n = 0;
    if (*err == 0u) n = process_segment<false>(P, i, nullptr);
    seg_count[i] = n;
}

// (d) write pass: one thread per input segment re-derives its pieces and stores its records
__global__ void __launch_bounds__(kSegThreads)
k_write(Params P, const uint32_t* __restrict__ seg_count, const uint64_t* __restrict__ seg_off, float4* __restrict__ out,
        uint64_t cap_records, uint32_t* err) {
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
    uint32_t *pt_off, *path_idx, *sp_first, *seg_count;
    uint64_t* seg_off;
    uint64_t cap_segs;
    uint8_t* sync_area;   // [flags 64 B][d_total 64 B][alloc tile states][tag tile states]
    uint64_t sync_bytes;
    uint64_t* h_pinned;   // pinned: [0] total, [1] flags
    // last sx_count
    sx::Params P;
    uint64_t n_paths;
    bool counted, total_known;
    uint64_t total;
    uint64_t launches;
    // staging for stroke_expand_host
    uint8_t* st_in;  uint64_t st_in_bytes;
    uint8_t* st_out; uint64_t st_out_bytes;
    uint64_t* st_path; uint64_t st_path_n;
};

static uint32_t* ctx_err(sx_ctx* c) { return reinterpret_cast<uint32_t*>(c->sync_area); }
static uint32_t* ctx_ticket(sx_ctx* c, int k) { return reinterpret_cast<uint32_t*>(c->sync_area) + 4 + 4 * k; }
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
        // one allocation: 4 u32 arrays then the u64 offsets (all 256-byte aligned since cap % 64 == 0)
        uint8_t* p;
        SX_CUDA(cudaMalloc(&p, cap * (4 * 4 + 8)));
        c->pt_off = reinterpret_cast<uint32_t*>(p);
        c->path_idx = c->pt_off + cap;
        c->sp_first = c->path_idx + cap;
        c->seg_count = c->sp_first + cap;
        c->seg_off = reinterpret_cast<uint64_t*>(c->seg_count + cap);
        c->cap_segs = cap;
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
    cudaError_t e = cudaMallocHost(reinterpret_cast<void**>(&c->h_pinned), 64);
    if (e != cudaSuccess) { g_last_cuda = e; free(c); return SX_E_CUDA; }
    *out = c;
    return SX_OK;
}

sx_status sx_destroy(sx_ctx* c) {
    if (!c) return SX_E_INVALID_ARG;
    cudaSetDevice(c->device);
    cudaDeviceSynchronize();
    cudaFree(c->pt_off);
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
    c->total = 0;

    // reset the error flag, the tickets, the total and the look-back states
    SX_CUDA(cudaMemsetAsync(c->sync_area, 0, c->sync_bytes, s));
    if (n_tags == 0) {
        SX_CUDA(cudaMemsetAsync(d_path_offsets, 0, 8, s));
    } else {
        uint32_t n = P.n_tags;
        uint32_t n_alloc_tiles = (n + sx::kCntTile - 1) / sx::kCntTile, n_tag_tiles = (n + sx::kTagTile - 1) / sx::kTagTile;
        uint64_t* alloc_states = reinterpret_cast<uint64_t*>(c->sync_area + 128);
        sx::TagTileState* tag_states = reinterpret_cast<sx::TagTileState*>(c->sync_area + 128 + round_up((uint64_t)(n_alloc_tiles + 1) * 8, 64));
        sx::k_tag_scan<<<n_tag_tiles, sx::kScanThreads, 0, s>>>(d_tags, n, (uint32_t)n_points, (uint32_t)n_paths, c->pt_off, c->path_idx,
                                                               c->sp_first, tag_states, ctx_ticket(c, 0), ctx_err(c));
        sx::k_count<<<(n + sx::kSegThreads - 1) / sx::kSegThreads, sx::kSegThreads, 0, s>>>(P, c->seg_count, ctx_err(c));
        sx::k_alloc_scan<<<n_alloc_tiles, sx::kScanThreads, 0, s>>>(c->seg_count, n, d_tags, c->path_idx, (uint32_t)n_paths, c->seg_off,
                                                                  d_path_offsets, ctx_total(c), alloc_states, ctx_ticket(c, 1), ctx_err(c));
        c->launches += 3;
        SX_CUDA(cudaGetLastError());
    }
    c->counted = true;
    if (h_total) {
        SX_CUDA(cudaMemcpyAsync(&c->h_pinned[0], ctx_total(c), 8, cudaMemcpyDeviceToHost, s));
        SX_CUDA(cudaMemcpyAsync(&c->h_pinned[1], ctx_err(c), 4, cudaMemcpyDeviceToHost, s));
        SX_CUDA(cudaStreamSynchronize(s));
        uint32_t flags = static_cast<uint32_t>(c->h_pinned[1] & 0xffffffffu);
        *h_total = c->h_pinned[0];
        c->total = c->h_pinned[0];
        c->total_known = true;
        if (flags & sx::kErrBadStream) { c->counted = false; *h_total = 0; return SX_E_BAD_STREAM; }
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
    sx::k_write<<<(n + sx::kSegThreads - 1) / sx::kSegThreads, sx::kSegThreads, 0, s>>>(c->P, c->seg_count, c->seg_off,
                                                                                      static_cast<float4*>(d_out_records), cap_records, ctx_err(c));
    c->launches += 1;
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
