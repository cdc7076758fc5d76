// sx_dash.cu -- the dashing kernels (sx_dash.cuh), a translation unit of their own in namespace sx_dash: the
// kernels of the undashed pipeline do not carry this code (they are bound by the instruction cache).
#define SX_REFINED 1   // (all three output modes: these kernels are not the ones the instruction cache decides)
#define sx sx_dash
#include "sx_dash.cuh"
#undef sx
#include "sx_dash.h"
#include <string.h>

void sxd_launch(int stage, const sx_dash_launch* a, uint32_t n_tags, cudaStream_t s) {
    sx_dash::DashArgs A;
    memcpy(&A.P, a->params, sizeof(A.P));
    A.nd = a->nd;
    for (int k = 0; k < 8; k++) A.dq[k] = a->dq[k];
    A.period = a->period; A.phase_q = a->phase_q;
    A.seg_len = a->seg_len; A.seg_pos = a->seg_pos; A.sp_total = a->sp_total;
    A.seg_count = a->seg_count; A.seg_off = a->seg_off;
    A.out = static_cast<float4*>(a->out); A.cap_records = a->cap_records; A.wide = a->wide; A.err = a->err;
    const unsigned grid = (n_tags + sx_dash::kDashThreads - 1) / sx_dash::kDashThreads;
    if (stage == 0) sx_dash::k_dash_len<<<grid, sx_dash::kDashThreads, 0, s>>>(A);
    else if (stage == 1) sx_dash::k_dash_totals<<<grid, sx_dash::kDashThreads, 0, s>>>(A);
    else if (stage == 2) sx_dash::k_dash_count<<<grid, sx_dash::kDashThreads, 0, s>>>(A);
    else sx_dash::k_dash_write<<<grid, sx_dash::kDashThreads, 0, s>>>(A);
}
