// Score scan: one fp32 importance score per cached token and KV head (steps a1 + a2 of DESIGN.md).
//
//   s[g,t] = sm_scale * q_rep[b, h*G+g, :] . K[b, t, h, :]          (Eq.(1))
//   mode 0 : a[t] = max_g s[g,t]  -> score plane + fused level-1 radix histogram for the top-k
//   mode 1 : raw s[g,t] planes + per-CTA online-softmax statistics (m_g, l_g)
//
// The scan is an HBM stream over K: 256 B read per (token, KV head), G*128 MACs.  One warp owns one
// (page, KV head) tile = 16 token rows x 256 B and feeds them straight from 128-bit global loads into
// mma.sync.m16n8k16 (A = 16 tokens x 16 channels, B = 16 channels x 8 query heads, G <= 8), so the
// arithmetic is 8 MMAs per 4 KB and the kernel stays bandwidth-bound.  The channel index is permuted
// identically in A and B (a dot product does not care), which lets every lane use plain 16-byte loads:
// lane (g = lane/4, t = lane%4) loads channels [32i + 8t, 32i + 8t + 8) of token rows g and g+8.
#pragma once
#include "common.cuh"

namespace herald {

constexpr int kScanThreads = 1024;             // one CTA per SM: 32 warps x 8 x 16-byte loads in flight per lane
constexpr int kScanWarps = kScanThreads / 32;
constexpr int kScanMaxCtas = 2048;             // bound on the grid (sizes the mode-1 partial statistics)

struct ScanParams {
    const __nv_bfloat16* k_pages;
    int64_t page_stride, token_stride, head_stride;
    const int32_t* page_table;
    const int32_t* seq_lens;
    const __nv_bfloat16* q_rep;
    float* scores;        // [batch][H_kv][max_seq_len]              (mode 0)
    float* raw;           // [batch][H_kv][G][max_seq_len]           (mode 1)
    float2* stats_part;   // [batch*H_kv][G][gridDim.x] (m, l)       (mode 1)
    uint32_t* hist1;      // [batch*H_kv][kBins1]                    (mode 0)
    int32_t batch, n_q_heads, n_kv_heads, max_seq_len, max_pages;
    int32_t l2_prefetch;        // page-major scan with 32-byte loads: bytes of a page to prefetch into L2 one iteration ahead (0 = off); set for grids of
                                // a few CTAs, where latency and not HBM bounds the stream (it costs 6 % when every SM scans)
    int32_t part_lo, part_hi;   // this launch covers [part_lo, part_hi) thousandths of the tile space (0, 1000 = all of it): the
                                // pipeline runs a head part on every SM before the denoising steps and the rest beside them
    float sm_scale;
};

// The grid is flat and persistent: the (unit, page) tiles of the whole batch, in unit-major order, are cut into
// gridDim.x equal contiguous ranges, one per CTA (units are ragged: sequence b has ceil(L_b / 16) pages per KV head).
// A CTA therefore touches one or two units and keeps one shared-memory histogram at a time.  The grid size is the
// number of SMs the scan may occupy: all of them when it runs alone, the SMs the attention kernel leaves free when
// it runs beside the denoising steps.
struct ScanRange {
    int64_t g0, g1;   // this CTA's range of global tile indices
};
__device__ __forceinline__ int seq_pages(const ScanParams& p, int b) {
    return (min(p.seq_lens[b], p.max_seq_len) + kPageSize - 1) / kPageSize;
}
__device__ __forceinline__ int64_t cta_range_begin(int64_t total, int cta, int n_ctas) { return total * cta / n_ctas; }
// the same cut inside the part [lo, hi) thousandths of the tile space
__device__ __forceinline__ int64_t cta_part_begin(int64_t total, int lo, int hi, int cta, int n_ctas) {
    const int64_t r0 = total * lo / 1000, r1 = total * hi / 1000;
    return r0 + (r1 - r0) * cta / n_ctas;
}

template <int kMode>
__global__ void __launch_bounds__(kScanThreads, 1) scan_kernel(const ScanParams p) {
    __shared__ uint32_t s_hist[kMode == 0 ? kBins1 : 1];
    __shared__ float2 s_stats[kMode == 1 ? kScanWarps * 8 : 1];
    __shared__ int64_t s_total;

    const int G = p.n_q_heads / p.n_kv_heads;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 2, tig = lane & 3;

    if (threadIdx.x == 0) {
        int64_t total = 0;
        for (int b = 0; b < p.batch; ++b) total += (int64_t)seq_pages(p, b) * p.n_kv_heads;
        s_total = total;
    }
    if (kMode == 0)
        for (int i = threadIdx.x; i < kBins1; i += kScanThreads) s_hist[i] = 0;
    __syncthreads();
    const int64_t total = s_total;
    // (mode 1 always covers the whole space: its partial statistics are indexed by the same cut in aggregate_softmax_kernel)
    const int64_t g0 = kMode == 0 ? cta_part_begin(total, p.part_lo, p.part_hi, blockIdx.x, gridDim.x) : cta_range_begin(total, blockIdx.x, gridDim.x);
    const int64_t g1 = kMode == 0 ? cta_part_begin(total, p.part_lo, p.part_hi, blockIdx.x + 1, gridDim.x) : cta_range_begin(total, blockIdx.x + 1, gridDim.x);

    // walk the units that intersect [g0, g1)
    int64_t unit_begin = 0;   // global tile index of the current unit's page 0
    for (int b = 0; b < p.batch && unit_begin < g1; ++b) {
        const int L = min(p.seq_lens[b], p.max_seq_len);
        const int n_pages = (L + kPageSize - 1) / kPageSize;
        const int32_t* pt = p.page_table + (int64_t)b * p.max_pages;
        for (int h = 0; h < p.n_kv_heads; ++h, unit_begin += n_pages) {
            const int64_t lo = max(g0, unit_begin), hi = min(g1, unit_begin + n_pages);
            if (lo >= hi) continue;                       // block-uniform
            const int unit = b * p.n_kv_heads + h;
            const int page_lo = (int)(lo - unit_begin), page_hi = (int)(hi - unit_begin);

            // B operand: query head g of this KV head's group (zeros for g >= G), channel-permuted like A.
            uint4 qf[4];
            {
                const __nv_bfloat16* qrow = p.q_rep + ((int64_t)b * p.n_q_heads + h * G + g) * kHeadDim + 8 * tig;
#pragma unroll
                for (int i = 0; i < 4; ++i) qf[i] = (g < G) ? ldg_u4(qrow + 32 * i) : make_uint4(0, 0, 0, 0);
            }
            // running softmax statistics of columns 2*tig, 2*tig+1 over this thread's rows (mode 1)
            float run_m[2] = {-INFINITY, -INFINITY}, run_l[2] = {0.f, 0.f};
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
                float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    mma_bf16_16816(acc, a[i].x, c[i].x, a[i].y, c[i].y, qf[i].x, qf[i].y);
                    mma_bf16_16816(acc, a[i].z, c[i].z, a[i].w, c[i].w, qf[i].z, qf[i].w);
                }
                // acc[0],acc[1]: token row g, heads 2*tig, 2*tig+1 ; acc[2],acc[3]: token row g+8
                const int t0 = page * kPageSize;
                if (kMode == 0) {
                    const bool v0 = 2 * tig < G, v1 = 2 * tig + 1 < G;
                    float m0 = fmaxf(v0 ? acc[0] : -INFINITY, v1 ? acc[1] : -INFINITY);
                    float m1 = fmaxf(v0 ? acc[2] : -INFINITY, v1 ? acc[3] : -INFINITY);
                    m0 = fmaxf(m0, __shfl_xor_sync(0xffffffffu, m0, 1));
                    m1 = fmaxf(m1, __shfl_xor_sync(0xffffffffu, m1, 1));
                    m0 = fmaxf(m0, __shfl_xor_sync(0xffffffffu, m0, 2));
                    m1 = fmaxf(m1, __shfl_xor_sync(0xffffffffu, m1, 2));
                    // lanes with tig 0 publish row g, lanes with tig 1 publish row g+8: 16 lanes -> 64 contiguous bytes
                    const int t = t0 + (tig == 0 ? g : g + 8);
                    if (tig < 2 && t < L) {
                        const float v = (tig == 0 ? m0 : m1) * p.sm_scale;
                        score_row[t] = v;
                        atomicAdd(&s_hist[score_key(v) >> (32 - kBits1)], 1u);
                    }
                } else {
                    float* raw_unit = p.raw + (int64_t)unit * G * p.max_seq_len;
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const int col = 2 * tig + (e & 1);
                        const int t = t0 + g + ((e >> 1) ? 8 : 0);
                        if (col < G && t < L) {
                            const float v = acc[e] * p.sm_scale;
                            raw_unit[(int64_t)col * p.max_seq_len + t] = v;
                            const int c2 = e & 1;
                            const float mn = fmaxf(run_m[c2], v);
                            run_l[c2] = run_l[c2] * __expf(run_m[c2] - mn) + __expf(v - mn);
                            run_m[c2] = mn;
                        }
                    }
                }
                page = next;
                phys = phys_next;
            }

            // ---- end of this CTA's share of the unit: flush ----
            if (kMode == 0) {
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
            } else {
                // merge (m, l) over the 8 token-row groups of the warp (lanes with equal tig), then over warps
#pragma unroll
                for (int c2 = 0; c2 < 2; ++c2) {
                    float m = run_m[c2], l = run_l[c2];
#pragma unroll
                    for (int o = 4; o < 32; o <<= 1) {
                        const float mo = __shfl_xor_sync(0xffffffffu, m, o), lo2 = __shfl_xor_sync(0xffffffffu, l, o);
                        const float mn = fmaxf(m, mo);
                        l = (m == -INFINITY ? 0.f : l * __expf(m - mn)) + (mo == -INFINITY ? 0.f : lo2 * __expf(mo - mn));
                        m = mn;
                    }
                    if (g == 0) s_stats[warp * 8 + 2 * tig + c2] = make_float2(m, l);
                }
                __syncthreads();
                if (threadIdx.x < G) {
                    float m = -INFINITY, l = 0.f;
                    for (int w = 0; w < kScanWarps; ++w) {
                        const float2 st = s_stats[w * 8 + threadIdx.x];
                        const float mn = fmaxf(m, st.x);
                        l = (m == -INFINITY ? 0.f : l * __expf(m - mn)) + (st.x == -INFINITY ? 0.f : st.y * __expf(st.x - mn));
                        m = mn;
                    }
                    p.stats_part[((int64_t)unit * G + threadIdx.x) * gridDim.x + blockIdx.x] = make_float2(m, l);
                }
                __syncthreads();
            }
        }
    }
}

// Mode 0, page-major order (H_kv divides 32, H_kv <= 8: every BASELINE.json shape).  A page of the cache holds the 16
// rows of ALL KV heads contiguously (16 x H_kv x 256 B); here the H_kv warps next to each other read the H_kv head
// tiles of the same page at the same time, so DRAM sees whole 4-16 KB pages instead of 256-byte pieces 1 KB apart
// (+6 % bandwidth on B200).  Work = the pages of the batch in sequence-major order, cut into gridDim.x equal
// contiguous ranges; a CTA keeps one histogram per KV head in shared memory (H_kv x 16 KB, dynamic).
//
// kWide (rows 32-byte aligned): a lane loads 32 bytes at a time (ld.global.v8.b32, sm_100), so the four lanes that share a
// token row cover one whole 128-byte line per load instruction.  The SM's load pipe handles one line per clock whether a warp
// uses 64 or 128 bytes of it: with 16-byte loads (8 rows x 64 B per instruction) ncu shows the L1 data pipe 76 % busy on the
// SMs of a 20-CTA scan and the SM streams at 78 GB/s (a load-only kernel with this pattern: 118); with 32-byte loads the
// same pattern reaches 170 GB/s per SM.  That is what the retrieval stream has beside the attention.
// 768 threads there: the tile of a lane is 32 registers + 16 of q; at 1024 threads (64 registers) that kernel spills and gains
// nothing, at 512 too few bytes are in flight.  When every SM scans, HBM is the bound and bytes in flight are what counts: the
// launcher then takes the 16-byte loads with 1024 threads (76.6 against 73.8 % of 8 TB/s on C2).
constexpr int kScanPmWideThreads = 768;

template <bool kWide, int kThreads>
__global__ void __launch_bounds__(kThreads, 1) scan_pm_kernel(const ScanParams p) {
    constexpr int kScanPmThreads = kThreads, kScanPmWarps = kThreads / 32;
    extern __shared__ uint32_t s_hist_pm[];   // [H_kv][kBins1]
    __shared__ int64_t s_total;

    const int G = p.n_q_heads / p.n_kv_heads, H = p.n_kv_heads;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 2, tig = lane & 3;
    const int h = warp % H;                    // fixed per warp: H divides the warp count
    const int pages_per_iter = kScanPmWarps / H;

    if (threadIdx.x == 0) {
        int64_t total = 0;
        for (int b = 0; b < p.batch; ++b) total += seq_pages(p, b);
        s_total = total;
    }
    for (int i = threadIdx.x; i < H * kBins1; i += kScanPmThreads) s_hist_pm[i] = 0;
    __syncthreads();
    const int64_t total = s_total;
    const int64_t g0 = cta_part_begin(total, p.part_lo, p.part_hi, blockIdx.x, gridDim.x);
    const int64_t g1 = cta_part_begin(total, p.part_lo, p.part_hi, blockIdx.x + 1, gridDim.x);
    uint32_t* my_hist = s_hist_pm + h * kBins1;
    const bool v0 = 2 * tig < G, v1 = 2 * tig + 1 < G;

    int64_t seq_begin = 0;
    for (int b = 0; b < p.batch && seq_begin < g1; ++b) {
        const int L = min(p.seq_lens[b], p.max_seq_len);
        const int n_pages = (L + kPageSize - 1) / kPageSize;
        const int64_t lo = max(g0, seq_begin), hi = min(g1, seq_begin + n_pages);
        seq_begin += n_pages;
        if (lo >= hi) continue;                            // block-uniform
        const int page_lo = (int)(lo - (seq_begin - n_pages)), page_hi = (int)(hi - (seq_begin - n_pages));
        const int32_t* pt = p.page_table + (int64_t)b * p.max_pages;
        // B operand: query head g of this KV head's group (zeros for g >= G), channel-permuted like A: register 4i + r of the
        // lane holds channels [32 i + 8 tig + 2r, +2) (16-byte loads) or register 8j + r channels [64 j + 16 tig + 2r, +2) (32-byte)
        uint32_t qf[16];
        {
            const __nv_bfloat16* qrow = p.q_rep + ((int64_t)b * p.n_q_heads + h * G + g) * kHeadDim + (kWide ? 16 : 8) * tig;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const uint4 v = (g < G) ? ldg_u4(kWide ? qrow + 64 * (i >> 1) + 8 * (i & 1) : qrow + 32 * i) : make_uint4(0, 0, 0, 0);
                qf[4 * i] = v.x, qf[4 * i + 1] = v.y, qf[4 * i + 2] = v.z, qf[4 * i + 3] = v.w;
            }
        }
        float* score_row = p.scores + (int64_t)(b * H + h) * p.max_seq_len;

        // wide kernel: page ids run two iterations ahead of the loads, so that the id of the next page is in a register when its
        // prefetch is issued (the 64-register kernel has no register for that and looks one iteration ahead)
        int page = page_lo + warp / H;
        int phys = page < page_hi ? __ldg(pt + page) : 0;
        int phys_next = kWide && page + pages_per_iter < page_hi ? __ldg(pt + page + pages_per_iter) : 0;
        while (page < page_hi) {
            const int next = page + pages_per_iter;
            int phys_next2 = 0;
            if (kWide) {
                phys_next2 = next + pages_per_iter < page_hi ? __ldg(pt + next + pages_per_iter) : 0;
                // the page of the next iteration is pulled into L2 while this one is multiplied (one request per page: its H head
                // tiles are contiguous): the loads then find it there, and the few SMs of an overlapped scan need fewer bytes in flight
                if (p.l2_prefetch && h == 0 && lane == 0 && next < page_hi)
                    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p.k_pages + (int64_t)phys_next * p.page_stride), "r"((uint32_t)p.l2_prefetch) : "memory");
            } else {
                phys_next = next < page_hi ? __ldg(pt + next) : 0;
            }
            const __nv_bfloat16* base = p.k_pages + (int64_t)phys * p.page_stride + (int64_t)h * p.head_stride + (kWide ? 16 : 8) * tig;
            const __nv_bfloat16* r0 = base + (int64_t)g * p.token_stride;
            const __nv_bfloat16* r1 = base + (int64_t)(g + 8) * p.token_stride;
            uint32_t a[16], c[16];   // token rows g and g + 8
            if (kWide) {
                ldg_stream_u8(r0, a);
                ldg_stream_u8(r1, c);
                ldg_stream_u8(r0 + 64, a + 8);
                ldg_stream_u8(r1 + 64, c + 8);
            } else {
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const uint4 va = ldg_stream_u4(r0 + 32 * i), vc = ldg_stream_u4(r1 + 32 * i);
                    a[4 * i] = va.x, a[4 * i + 1] = va.y, a[4 * i + 2] = va.z, a[4 * i + 3] = va.w;
                    c[4 * i] = vc.x, c[4 * i + 1] = vc.y, c[4 * i + 2] = vc.z, c[4 * i + 3] = vc.w;
                }
            }
            float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int i = 0; i < 8; ++i) mma_bf16_16816(acc, a[2 * i], c[2 * i], a[2 * i + 1], c[2 * i + 1], qf[2 * i], qf[2 * i + 1]);
            float m0 = fmaxf(v0 ? acc[0] : -INFINITY, v1 ? acc[1] : -INFINITY);
            float m1 = fmaxf(v0 ? acc[2] : -INFINITY, v1 ? acc[3] : -INFINITY);
            m0 = fmaxf(m0, __shfl_xor_sync(0xffffffffu, m0, 1));
            m1 = fmaxf(m1, __shfl_xor_sync(0xffffffffu, m1, 1));
            m0 = fmaxf(m0, __shfl_xor_sync(0xffffffffu, m0, 2));
            m1 = fmaxf(m1, __shfl_xor_sync(0xffffffffu, m1, 2));
            const int t = page * kPageSize + (tig == 0 ? g : g + 8);
            if (tig < 2 && t < L) {
                const float v = (tig == 0 ? m0 : m1) * p.sm_scale;
                score_row[t] = v;
                atomicAdd(&my_hist[score_key(v) >> (32 - kBits1)], 1u);
            }
            page = next;
            phys = phys_next;
            if (kWide) phys_next = phys_next2;
        }
        // ---- end of this CTA's share of sequence b: flush the H histograms ----
        __syncthreads();
        uint32_t* gh = p.hist1 + (int64_t)b * H * kBins1;   // units b*H .. b*H + H-1 are contiguous
        for (int i = threadIdx.x; i < H * kBins1; i += kScanPmThreads) {
            const uint32_t v = s_hist_pm[i];
            if (v) {
                atomicAdd(gh + i, v);
                s_hist_pm[i] = 0;
            }
        }
        __syncthreads();
    }
}

// Mode 1, second pass: a[t] = sum_g exp(s[g,t] - m_g) / l_g, score plane + level-1 histogram.
struct AggParams {
    const float* raw;
    const float2* stats_part;
    int32_t n_parts;      // grid size of the scan that wrote stats_part
    const float* lse;     // optional [batch][H_q]: finished log-sum-exp per head (herald_select_rep); replaces stats_part
    const int32_t* seq_lens;
    float* scores;
    uint32_t* hist1;
    int32_t batch, n_q_heads, n_kv_heads, max_seq_len;
};

__global__ void __launch_bounds__(256) aggregate_softmax_kernel(const AggParams p) {
    __shared__ uint32_t s_hist[kBins1];
    __shared__ float s_m[8], s_inv_l[8];
    const int b = blockIdx.z, h = blockIdx.y;
    const int unit = b * p.n_kv_heads + h;
    const int G = p.n_q_heads / p.n_kv_heads;
    const int L = min(p.seq_lens[b], p.max_seq_len);
    for (int i = threadIdx.x; i < kBins1; i += blockDim.x) s_hist[i] = 0;
    if (p.lse) {
        if (threadIdx.x < G) {   // exp(s - m) / l with m = lse, l = 1
            s_m[threadIdx.x] = p.lse[(int64_t)b * p.n_q_heads + h * G + threadIdx.x];
            s_inv_l[threadIdx.x] = 1.f;
        }
    } else if (threadIdx.x < G) {
        // the scan CTAs whose tile range intersects this unit wrote a partial (same range arithmetic as scan_kernel)
        int64_t total = 0, unit_begin = 0;
        for (int bb = 0; bb < p.batch; ++bb) {
            const int np = (min(p.seq_lens[bb], p.max_seq_len) + kPageSize - 1) / kPageSize;
            if (bb < b) unit_begin += (int64_t)np * p.n_kv_heads;
            total += (int64_t)np * p.n_kv_heads;
        }
        const int n_pages = (L + kPageSize - 1) / kPageSize;
        unit_begin += (int64_t)h * n_pages;
        float m = -INFINITY, l = 0.f;
        const float2* sp = p.stats_part + ((int64_t)unit * G + threadIdx.x) * p.n_parts;
        for (int i = 0; i < p.n_parts; ++i) {
            const int64_t lo = max(cta_range_begin(total, i, p.n_parts), unit_begin);
            const int64_t hi = min(cta_range_begin(total, i + 1, p.n_parts), unit_begin + n_pages);
            if (lo >= hi) continue;
            const float2 s = sp[i];
            const float mn = fmaxf(m, s.x);
            l = (m == -INFINITY ? 0.f : l * __expf(m - mn)) + (s.x == -INFINITY ? 0.f : s.y * __expf(s.x - mn));
            m = mn;
        }
        s_m[threadIdx.x] = m;
        s_inv_l[threadIdx.x] = 1.f / l;
    }
    __syncthreads();
    const float* raw_unit = p.raw + (int64_t)unit * G * p.max_seq_len;
    float* score_row = p.scores + (int64_t)unit * p.max_seq_len;
    for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < L; t += gridDim.x * blockDim.x) {
        float a = 0.f;
        for (int gq = 0; gq < G; ++gq) a += __expf(raw_unit[(int64_t)gq * p.max_seq_len + t] - s_m[gq]) * s_inv_l[gq];
        score_row[t] = a;
        atomicAdd(&s_hist[score_key(a) >> (32 - kBits1)], 1u);
    }
    __syncthreads();
    uint32_t* gh = p.hist1 + (int64_t)unit * kBins1;
    for (int i = threadIdx.x; i < kBins1; i += blockDim.x) {
        const uint32_t v = s_hist[i];
        if (v) atomicAdd(gh + i, v);
    }
}

}  // namespace herald
