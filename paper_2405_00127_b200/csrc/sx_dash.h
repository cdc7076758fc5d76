// sx_dash.h -- launchers of the dashing kernels (sx_dash.cu / sx_dash.cuh).  `params` points to an sx::Params
// (same layout in every translation unit: the same header).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

struct sx_dash_launch {
    const void* params;                     // sx::Params of the call
    uint32_t nd;                            // pattern entries
    unsigned long long dq[8], period, phase_q;   // units of 2^-16 px
    uint32_t* seg_len;                      // [n] scratch
    unsigned long long* seg_pos;            // [n] scratch: prefix sum of seg_len
    unsigned long long* sp_total;           // [n] scratch
    uint32_t* seg_count;
    const uint64_t* seg_off;
    void* out; uint64_t cap_records; uint32_t wide;
    uint32_t* err;
};
// stage 0: k_dash_len; 1: k_dash_totals; 2: k_dash_count; 3: k_dash_write
void sxd_launch(int stage, const sx_dash_launch* a, uint32_t n_tags, cudaStream_t s);
