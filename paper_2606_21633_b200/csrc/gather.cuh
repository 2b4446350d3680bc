// Gather of the selected K/V rows from the paged full cache into the idle sparse pool
// (step a4 of DESIGN.md; "gathers the selected entries into a contiguous ... buffer",
// PAPER.md:175 idle pool).  Pure bit copies: 256 B per row and tensor, 16 B per lane, four independent
// 128-bit loads in flight per lane; rows past sel_cnt are left untouched.
#pragma once
#include "common.cuh"

namespace herald {

constexpr int kGatherThreads = 256;
constexpr int kGatherRowsPerWarp = 4;

struct GatherParams {
    const __nv_bfloat16* k_pages;
    const __nv_bfloat16* v_pages;
    int64_t page_stride, token_stride, head_stride;
    const int32_t* page_table;
    const int32_t* sel_idx;   // [units][cap]
    const int32_t* sel_cnt;   // [units]
    __nv_bfloat16* pool_k;    // [units][cap][128]
    __nv_bfloat16* pool_v;
    int32_t n_kv_heads, max_pages, cap;
};

__global__ void __launch_bounds__(kGatherThreads) gather_kernel(const GatherParams p) {
    const int unit = blockIdx.y;
    const int b = unit / p.n_kv_heads, h = unit % p.n_kv_heads;
    const int n = min(p.sel_cnt[unit], p.cap);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int half = lane >> 4, chunk = lane & 15;
    const int32_t* idx = p.sel_idx + (int64_t)unit * p.cap;
    const int32_t* pt = p.page_table + (int64_t)b * p.max_pages;
    const int warps_total = gridDim.x * (kGatherThreads / 32);

    for (int j0 = (blockIdx.x * (kGatherThreads / 32) + warp) * kGatherRowsPerWarp; j0 < n;
         j0 += warps_total * kGatherRowsPerWarp) {
        int rows[2] = {j0 + half, j0 + 2 + half};
        int64_t src[2];
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            src[r] = -1;
            if (rows[r] < n) {
                const int pos = __ldg(idx + rows[r]);
                const int phys = __ldg(pt + (pos >> 4));
                src[r] = (int64_t)phys * p.page_stride + (int64_t)(pos & (kPageSize - 1)) * p.token_stride +
                         (int64_t)h * p.head_stride + chunk * 8;
            }
        }
        uint4 kv[2], vv[2];
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            if (src[r] >= 0) {
                kv[r] = ldg_stream_u4(p.k_pages + src[r]);
                vv[r] = ldg_stream_u4(p.v_pages + src[r]);
            }
        }
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            if (src[r] >= 0) {
                const int64_t dst = ((int64_t)unit * p.cap + rows[r]) * kHeadDim + chunk * 8;
                *reinterpret_cast<uint4*>(p.pool_k + dst) = kv[r];
                *reinterpret_cast<uint4*>(p.pool_v + dst) = vv[r];
            }
        }
    }
}

}  // namespace herald
