// Score scan with x queries per sequence (NEXT-4 of DESIGN.md; PAPER.md:137 Fig. 8, :143, :161: "the selection
// kernel as the number of queries is reduced from B = 32 to one").
//
//   scores[b, h, t] = sm_scale * max over j < x, g < G of  q_x[b, j, h*G+g] . K[b, t, h]        (reading 25)
//
// x = 1 is the representative-query scan (scan.cuh).  K is streamed once whatever x is: per page (16 tokens of one KV
// head, 4 KB) a warp holds the K fragments in registers and runs ceil(x*G / 8) score tiles of 8 query rows against
// them -- mma.sync m16n8k16, tokens on M, query rows on N, the B fragments read from shared memory where the x*G rows
// of the current KV head are kept pre-arranged (one conflict-free LDS.128 per two MMAs).  The running maximum per token
// stays in registers.  Bytes per token do not grow with x, FLOPs do: 2 * 128 * x*G per token and KV head, so the kernel
// leaves the HBM roofline for the mma.sync one somewhere in x (bench.py reports the sweep).
//   Head-major flat persistent grid like scan_kernel<0> (one CTA per SM, 32 warps): the (unit, page) space is cut into
//   gridDim.x equal ranges; where a range meets a unit the CTA stages that unit's query rows (<= 64 KB) and its warps
//   stride over the pages.  Level-1 histogram of the top-k is fused as in the other scans.
#pragma once
#include "scan.cuh"

namespace herald {

constexpr int kXqMaxTiles = 32;                       // 8-row score tiles per KV head: x * G <= 256 rows
constexpr int kXqTileBytes = 4 * 32 * 16;             // one tile's B fragments: [4 channel blocks][32 lanes] uint4
constexpr int kXqMaxSmemBytes = kXqMaxTiles * kXqTileBytes;

struct ScanXqParams {
    const __nv_bfloat16* k_pages;
    int64_t page_stride, token_stride, head_stride;
    const int32_t* page_table;
    const int32_t* seq_lens;
    const __nv_bfloat16* q_x;     // [batch][x][H_q][128]
    float* scores;                // [units][max_seq_len]
    uint32_t* hist1;              // [units][kBins1]
    int32_t batch, n_q_heads, n_kv_heads, max_seq_len, max_pages, x;
    float sm_scale;
};

__global__ void __launch_bounds__(kScanThreads, 1) scan_xq_kernel(const ScanXqParams p) {
    extern __shared__ __align__(16) uint4 s_q[];      // [n_tiles][4][32]: lane (g, tig) of tile r, block i: row 8r+g, channels 32i+8tig..+8
    __shared__ uint32_t s_hist[kBins1];
    __shared__ int64_t s_total;

    const int G = p.n_q_heads / p.n_kv_heads;
    const int rows = p.x * G, n_tiles = (rows + 7) / 8;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 2, tig = lane & 3;

    if (threadIdx.x == 0) {
        int64_t total = 0;
        for (int b = 0; b < p.batch; ++b) total += (int64_t)((min(p.seq_lens[b], p.max_seq_len) + kPageSize - 1) / kPageSize) * p.n_kv_heads;
        s_total = total;
    }
    for (int i = threadIdx.x; i < kBins1; i += kScanThreads) s_hist[i] = 0;
    __syncthreads();
    const int64_t total = s_total;
    const int64_t g0 = cta_range_begin(total, blockIdx.x, gridDim.x), g1 = cta_range_begin(total, blockIdx.x + 1, gridDim.x);

    int64_t unit_begin = 0;
    for (int b = 0; b < p.batch && unit_begin < g1; ++b) {
        const int L = min(p.seq_lens[b], p.max_seq_len);
        const int n_pages = (L + kPageSize - 1) / kPageSize;
        const int32_t* pt = p.page_table + (int64_t)b * p.max_pages;
        for (int h = 0; h < p.n_kv_heads; ++h, unit_begin += n_pages) {
            const int64_t lo = max(g0, unit_begin), hi = min(g1, unit_begin + n_pages);
            if (lo >= hi) continue;                       // block-uniform
            const int unit = b * p.n_kv_heads + h;
            const int page_lo = (int)(lo - unit_begin), page_hi = (int)(hi - unit_begin);

            // stage the x*G query rows of this KV head as B fragments; row rho = j*G + g' is query j, head h*G + g'.
            // The last tile is padded by repeating row 0: a maximum does not change under duplicates.
            for (int e = threadIdx.x; e < n_tiles * 128; e += kScanThreads) {
                const int r = e >> 7, i = (e >> 5) & 3, ln = e & 31;
                int rho = 8 * r + (ln >> 2);
                if (rho >= rows) rho = 0;
                const int j = rho / G, gq = rho % G;
                s_q[e] = ldg_u4(p.q_x + (((int64_t)b * p.x + j) * p.n_q_heads + h * G + gq) * kHeadDim + 32 * i + 8 * (ln & 3));
            }
            __syncthreads();
            float* score_row = p.scores + (int64_t)unit * p.max_seq_len;

            int page = page_lo + warp;
            int phys = page < page_hi ? __ldg(pt + page) : 0;
            while (page < page_hi) {
                const int next = page + kScanWarps;
                const int phys_next = next < page_hi ? __ldg(pt + next) : 0;
                const __nv_bfloat16* base = p.k_pages + (int64_t)phys * p.page_stride + (int64_t)h * p.head_stride + 8 * tig;
                const __nv_bfloat16* r0 = base + (int64_t)g * p.token_stride;
                const __nv_bfloat16* r1 = base + (int64_t)(g + 8) * p.token_stride;
                uint4 a[4], c[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    a[i] = ldg_stream_u4(r0 + 32 * i);
                    c[i] = ldg_stream_u4(r1 + 32 * i);
                }
                float m0 = -INFINITY, m1 = -INFINITY;   // token rows g, g+8: maximum over this lane's columns of every tile
                const uint4* sq = s_q + lane;
#pragma unroll 2
                for (int r = 0; r < n_tiles; ++r, sq += 128) {
                    float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const uint4 qf = sq[32 * i];
                        mma_bf16_16816(acc, a[i].x, c[i].x, a[i].y, c[i].y, qf.x, qf.y);
                        mma_bf16_16816(acc, a[i].z, c[i].z, a[i].w, c[i].w, qf.z, qf.w);
                    }
                    m0 = fmaxf(m0, fmaxf(acc[0], acc[1]));
                    m1 = fmaxf(m1, fmaxf(acc[2], acc[3]));
                }
                m0 = fmaxf(m0, __shfl_xor_sync(0xffffffffu, m0, 1));
                m1 = fmaxf(m1, __shfl_xor_sync(0xffffffffu, m1, 1));
                m0 = fmaxf(m0, __shfl_xor_sync(0xffffffffu, m0, 2));
                m1 = fmaxf(m1, __shfl_xor_sync(0xffffffffu, m1, 2));
                // lanes with tig 0 publish row g, lanes with tig 1 publish row g+8: 16 lanes -> 64 contiguous bytes
                const int t = page * kPageSize + (tig == 0 ? g : g + 8);
                if (tig < 2 && t < L) {
                    const float v = (tig == 0 ? m0 : m1) * p.sm_scale;
                    score_row[t] = v;
                    atomicAdd(&s_hist[score_key(v) >> (32 - kBits1)], 1u);
                }
                page = next;
                phys = phys_next;
            }
            // ---- end of this CTA's share of the unit: flush the histogram; s_q is restaged for the next unit ----
            __syncthreads();
            uint32_t* gh = p.hist1 + (int64_t)unit * kBins1;
            for (int i = threadIdx.x; i < kBins1; i += kScanThreads) {
                const uint32_t v = s_hist[i];
                if (v) {
                    atomicAdd(gh + i, v);
                    s_hist[i] = 0;
                }
            }
            __syncthreads();
        }
    }
}

}  // namespace herald
