// sx_refined.h -- launchers of the kernels of SX_MODE_LINE_REFINED (sx_refined.cu: the pipeline's headers compiled a second
// time, with the refined density integral switched on, in namespace sx_refined).  The argument structures have the layout of
// sx::CountArgs / sx::WriteArgs (the same headers); they are passed by address and copied.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

void sxr_launch_count(const void* count_args, unsigned grid, cudaStream_t s);
void sxr_launch_writers(const void* write_args, unsigned general_blocks, unsigned simple_blocks, unsigned segment_blocks, unsigned walk_blocks,
                        cudaStream_t s_general, cudaStream_t s_simple, cudaStream_t s_segments, cudaStream_t s_walk);
// probes (sx_eval): what = SX_EVAL_F_EXACT / SX_EVAL_F_INV_REFINED, one thread per item, device buffers
void sxr_launch_eval(int what, const float* d_in, float* d_out, uint64_t n);
