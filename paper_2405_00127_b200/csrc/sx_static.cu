// sx_static.cu -- sx_bin_lines_static: the tile binning of the line soup (sx_bin.cuh) for callers that
// cannot allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// The scratch of the binning (ticket, device-side flags, pair total, look-back words of the scan, one counter and one
// cursor per tile) lives in a FILE-SCOPE device array of a fixed size: kStaticMaxTiles tiles (a viewport of 4096 x 4096 px),
// 524,672 bytes, held by every GPU that loads the library until the process exits.  The entry point calls no cudaMalloc,
// cudaFree or allocating library routine; it rejects larger viewports with SX_E_INVALID_ARG.
//
// In HOST code the array's name is a host-side stand-in, not a device address: its device address is taken once per device
// with cudaGetSymbolAddress (that device current) and that pointer is what the kernels get.
//
// Every call on a device shares the array, and the array keeps the last call's contents: each call clears the part it uses
// on its stream first.  Calls that overlap on one GPU (two streams, two host threads) RACE on it: serialise them.
//
// Same kernels as sx_bin_lines (the header compiled a second time into namespace sx_static: this translation unit defines
// its own copies, the existing code path is untouched).
#define sx sx_static
#include "sx_bin.cuh"
#undef sx
#include "../../include/stroke_expand.h"
#include <mutex>

void sx_internal_note_cuda_error(int e);   // sx_kernels.cu: what sx_strerror(SX_E_CUDA) reports

namespace {

constexpr uint32_t kStaticMaxTiles = SX_STATIC_MAX_TILES;
constexpr uint32_t kMaxScanTiles = (kStaticMaxTiles + sx_static::kScan32Tile - 1) / sx_static::kScan32Tile;
constexpr uint64_t align64(uint64_t x) { return (x + 63) / 64 * 64; }
// layout: [ticket u32 @0 | flags u32 @4 | total u64 @8 : 64 B][look-back words][tile counters][tile cursors]
constexpr uint64_t kOffStates = 64;
constexpr uint64_t kOffCounts = kOffStates + align64((uint64_t)(kMaxScanTiles + 1) * 8);
constexpr uint64_t kOffCursor = kOffCounts + align64((uint64_t)kStaticMaxTiles * 4);
constexpr uint64_t kStaticBytes = kOffCursor + align64((uint64_t)kStaticMaxTiles * 4);
static_assert(kStaticBytes == SX_STATIC_SCRATCH_BYTES, "the header states the size of the static scratch");

static __device__ __align__(256) unsigned char g_static_scratch[kStaticBytes];

constexpr int kMaxDevices = 64;
struct DeviceSetup { unsigned char* scratch; int sm_count; bool ready; };
DeviceSetup g_setup[kMaxDevices];
std::mutex g_setup_mutex;

// once per device, that device current: the DEVICE address of the array (its name is only a stand-in on the host)
sx_status setup_device(int device, DeviceSetup* out) {
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    DeviceSetup& d = g_setup[device];
    if (!d.ready) {
        unsigned char* ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_static_scratch);
        if (e != cudaSuccess || ptr == nullptr) { sx_internal_note_cuda_error((int)e); return SX_E_CUDA; }
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
        if (e != cudaSuccess) { sx_internal_note_cuda_error((int)e); return SX_E_CUDA; }
        d.scratch = ptr;
        d.sm_count = sms > 0 ? sms : 148;
        d.ready = true;
    }
    *out = d;
    return SX_OK;
}

}  // namespace

#define SXS_CUDA(call)                                                      \
    do {                                                                    \
        cudaError_t e_ = (call);                                            \
        if (e_ != cudaSuccess) { sx_internal_note_cuda_error((int)e_); return SX_E_CUDA; }    \
    } while (0)

sx_status sx_bin_lines_static(int32_t device, const sx_line* d_lines, uint64_t n_lines, uint32_t tiles_x, uint32_t tiles_y,
                              uint32_t* d_tile_offsets, uint32_t* d_tile_lines, uint64_t cap_entries, uint32_t* d_flags,
                              void* cuda_stream) {
    if (device < 0 || device >= kMaxDevices || !d_tile_offsets) return SX_E_INVALID_ARG;
    if (n_lines >= (1ull << 32) || tiles_x == 0 || tiles_y == 0) return SX_E_INVALID_ARG;
    if ((uint64_t)tiles_x * tiles_y > kStaticMaxTiles) return SX_E_INVALID_ARG;   // beyond the static scratch: use sx_bin_lines
    if (n_lines > 0 && (!d_lines || (reinterpret_cast<uintptr_t>(d_lines) & 15u))) return SX_E_INVALID_ARG;
    if (cap_entries > 0 && !d_tile_lines) return SX_E_INVALID_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    SXS_CUDA(cudaSetDevice(device));
    DeviceSetup d;
    sx_status rc = setup_device(device, &d);
    if (rc != SX_OK) return rc;
    const uint32_t tiles = tiles_x * tiles_y;
    const uint32_t scan_tiles = (tiles + sx_static::kScan32Tile - 1) / sx_static::kScan32Tile;
    uint32_t* ticket = reinterpret_cast<uint32_t*>(d.scratch);
    uint32_t* flags = reinterpret_cast<uint32_t*>(d.scratch + 4);
    uint64_t* total = reinterpret_cast<uint64_t*>(d.scratch + 8);
    uint64_t* states = reinterpret_cast<uint64_t*>(d.scratch + kOffStates);
    uint32_t* counts = reinterpret_cast<uint32_t*>(d.scratch + kOffCounts);
    uint32_t* cursor = reinterpret_cast<uint32_t*>(d.scratch + kOffCursor);
    // the array keeps the last call's contents: everything this call reads before writing starts at zero
    SXS_CUDA(cudaMemsetAsync(d.scratch, 0, kOffStates + (uint64_t)(scan_tiles + 1) * 8, s));
    SXS_CUDA(cudaMemsetAsync(counts, 0, (uint64_t)tiles * 4, s));
    SXS_CUDA(cudaMemsetAsync(cursor, 0, (uint64_t)tiles * 4, s));
    const float4* lines = reinterpret_cast<const float4*>(d_lines);
    const uint64_t want = (n_lines + sx_static::kBinThreads - 1) / sx_static::kBinThreads;
    const uint64_t most = (uint64_t)d.sm_count * 16;
    const unsigned grid = (unsigned)(want < most ? (want ? want : 1) : most);
    sx_static::k_bin_walk<false><<<grid, sx_static::kBinThreads, 0, s>>>(lines, n_lines, tiles_x, tiles_y, counts, nullptr, nullptr, 0, flags);
    sx_static::k_scan_u32<<<scan_tiles, sx_static::kScanThreads, 0, s>>>(counts, tiles, d_tile_offsets, total, states, ticket, flags);
    if (cap_entries > 0)
        sx_static::k_bin_walk<true><<<grid, sx_static::kBinThreads, 0, s>>>(lines, n_lines, tiles_x, tiles_y, cursor, d_tile_offsets, d_tile_lines, cap_entries, flags);
    SXS_CUDA(cudaGetLastError());
    if (d_flags) SXS_CUDA(cudaMemcpyAsync(d_flags, flags, 4, cudaMemcpyDeviceToDevice, s));
    return SX_OK;
}
