// sx_refined.cu -- the kernels of SX_MODE_LINE_REFINED.
//
// The count pass and the writers are bound by the instruction cache: the double-precision density
// integral and its Newton-refined inverse would cost the other modes 14 % of the count pass if they sat in the same kernels
// (measured).  So the same headers are compiled a second time here, with SX_REFINED = 1, into namespace sx_refined; the
// host side (sx_kernels.cu) launches these when the mode asks for them.
#define SX_REFINED 1
#define sx sx_refined
#include "sx_write.cuh"
#undef sx
#include "../../include/stroke_expand.h"
#include "sx_refined.h"
#include <string.h>

void sxr_launch_count(const void* count_args, unsigned grid, cudaStream_t s) {
    sx_refined::CountArgs C;
    memcpy(&C, count_args, sizeof(C));
    sx_refined::k_count<<<grid, 32, sizeof(sx_refined::CtWarp), s>>>(C);
}

void sxr_launch_writers(const void* write_args, unsigned general_blocks, unsigned simple_blocks, unsigned segment_blocks, unsigned walk_blocks,
                        cudaStream_t s_general, cudaStream_t s_simple, cudaStream_t s_segments, cudaStream_t s_walk) {
    sx_refined::WriteArgs W;
    memcpy(&W, write_args, sizeof(W));
    sx_refined::k_write_general<<<general_blocks, sx_refined::kWrThreads, 0, s_general>>>(W);
    sx_refined::k_write_simple<<<simple_blocks, sx_refined::kWrThreads, 0, s_simple>>>(W);
    sx_refined::k_write_segments<<<segment_blocks, sx_refined::kWrThreads, 0, s_segments>>>(W);
    sx_refined::k_write_walk<<<walk_blocks, sx_refined::kWrThreads, 0, s_walk>>>(W);
}

__global__ void k_eval_refined(int what, const float* in, float* out, uint64_t n) {
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    out[i] = what == SX_EVAL_F_EXACT ? sx_refined::f_exact(in[i]) : sx_refined::f_inv_refined(in[i]);
}
void sxr_launch_eval(int what, const float* d_in, float* d_out, uint64_t n) {
    k_eval_refined<<<(unsigned)((n + 255) / 256), 256>>>(what, d_in, d_out, n);
}
