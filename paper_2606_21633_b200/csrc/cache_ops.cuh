// Block-boundary cache operations (NEXT-3 of DESIGN.md).  PAPER.md:189: the draft KV of block n is "appended temporarily"
// to the full KV pool for the selection of block n+1; at the end of the block the true KV is written "to
// both block n+1's GPU pool and the full KV pool, replacing the draft".  Pure bit copies of B x H_kv rows of 256 B per
// sequence: one half warp per row (16 B per lane), K and V together.
#pragma once
#include "common.cuh"

namespace herald {

struct CacheWriteParams {
    __nv_bfloat16* k_pages;
    __nv_bfloat16* v_pages;
    int64_t page_stride, token_stride, head_stride;
    const int32_t* page_table;
    const int32_t* write_pos;          // [batch]: logical position of block row 0
    const __nv_bfloat16* k_new;        // [batch][B][H_kv][128]
    const __nv_bfloat16* v_new;
    int32_t batch, block_size, n_kv_heads, max_pages;
};

// K[b, write_pos[b] + i, h, :] = k_new[b, i, h, :] (same for V): grid-stride over the batch * B * H_kv rows
__global__ void __launch_bounds__(256) cache_write_block_kernel(const CacheWriteParams p) {
    const int half = threadIdx.x >> 4, chunk = threadIdx.x & 15;
    const int rows = p.batch * p.block_size * p.n_kv_heads;
    for (int r = blockIdx.x * 16 + half; r < rows; r += gridDim.x * 16) {
        const int h = r % p.n_kv_heads, i = (r / p.n_kv_heads) % p.block_size, b = r / (p.n_kv_heads * p.block_size);
        const int t = p.write_pos[b] + i;
        const int phys = __ldg(p.page_table + (int64_t)b * p.max_pages + (t >> 4));
        const int64_t dst = (int64_t)phys * p.page_stride + (int64_t)(t & (kPageSize - 1)) * p.token_stride + (int64_t)h * p.head_stride + chunk * 8;
        const int64_t src = (int64_t)r * kHeadDim + chunk * 8;
        *reinterpret_cast<uint4*>(p.k_pages + dst) = ldg_u4(p.k_new + src);
        *reinterpret_cast<uint4*>(p.v_pages + dst) = ldg_u4(p.v_new + src);
    }
}

struct PoolAppendParams {
    __nv_bfloat16* pool_k;             // [batch][H_kv][cap][128]
    __nv_bfloat16* pool_v;
    int32_t* pool_len;                 // [batch][H_kv]: advanced by B
    const __nv_bfloat16* k_new;        // [batch][B][H_kv][128]
    const __nv_bfloat16* v_new;
    int32_t batch, block_size, n_kv_heads, cap;
};

// pool[b, h, pool_len[b,h] + i, :] = k_new[b, i, h, :]; pool_len[b,h] += B.  One block per unit (it alone updates the length);
// rows that would pass the capacity are dropped and the length clamps to cap.
__global__ void __launch_bounds__(256) pool_append_block_kernel(const PoolAppendParams p) {
    const int unit = blockIdx.x, b = unit / p.n_kv_heads, h = unit % p.n_kv_heads;
    const int half = threadIdx.x >> 4, chunk = threadIdx.x & 15;
    const int n = max(0, min(p.pool_len[unit], p.cap));
    for (int i = half; i < p.block_size; i += 16) {
        if (n + i >= p.cap) break;
        const int64_t src = (((int64_t)b * p.block_size + i) * p.n_kv_heads + h) * kHeadDim + chunk * 8;
        const int64_t dst = ((int64_t)unit * p.cap + n + i) * kHeadDim + chunk * 8;
        *reinterpret_cast<uint4*>(p.pool_k + dst) = ldg_u4(p.k_new + src);
        *reinterpret_cast<uint4*>(p.pool_v + dst) = ldg_u4(p.v_new + src);
    }
    __syncthreads();                    // every thread has read the old length
    if (threadIdx.x == 0) p.pool_len[unit] = min(n + p.block_size, p.cap);
}

}  // namespace herald
