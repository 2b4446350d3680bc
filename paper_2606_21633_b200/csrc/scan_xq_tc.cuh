// The x-query score scan as a tcgen05 contraction (NEXT-4 of DESIGN.md; "B queries perform attention in
// GEMM form").  With x*G >= 32 score rows per KV head the scan is a dense GEMM per 128-token tile,
//
//   D[token, rho] = sum_c K[token, c] * Q[rho, c]        M = 128 tokens (TMEM lanes), N = x*G rows (<= 256), K = 128,
//
// and the per-token maximum over rho (reading 25) is a reduction along one TMEM lane: one thread, no shuffles.
//   A = the K tile: 8 pages of the paged cache fetched by TMA (16 tokens x 64 channels per box and half), 128B swizzle
//   B = the x*G query rows of the current KV head, one TMA box per half, resident for the whole unit
//   D = fp32 in TMEM, two buffers of 256 columns: the MMAs of tile j+1 overlap the read-out of tile j
// Per tile the MMA costs 8 x (128 x N x 16) = 512 cycles at N = 256, the read-out about as much on 8 warps, the 32 KB of
// K 1400 cycles at the chip's HBM rate: the kernel stays on the HBM roofline at every x, which the mma.sync form
// (scan_xq.cuh) leaves at x*G ~ 32.
//   warps 0-7: read-out (TMEM lane quarter = warp % 4, column chunks of 32 alternate between warp / 4 = 0, 1), score
//   plane + level-1 histogram; warp 8: TMA producer; warp 9: MMA issuer.  One persistent CTA per SM.  The query rows of
//   one KV head fill the shared memory left beside the K ring, so a CTA works on one head at a time; to keep DRAM on
//   whole pages all the same (a page holds the rows of all H_kv heads side by side) the CTAs form sets of H_kv: a set
//   shares a range of the (sequence, tile) space and CTA i of the set takes head i of it, so the H_kv head slices of a
//   page are requested at about the same time (p.set_size = H_kv).  Grids smaller than H_kv fall back to ranges of the
//   (unit, tile) space (p.set_size = 1).
#pragma once
#include "attn_tc.cuh"
#include "scan.cuh"

namespace herald {

constexpr int kXtThreads = 10 * 32;
constexpr int kXtEpiWarps = 8, kXtTmaWarp = 8, kXtMmaWarp = 9;
constexpr int kXtStages = 4;                                  // K ring
constexpr int kXtQHalfBytes = 256 * 128;                      // [256 rows x 64 el] swizzled half of the query tile (32 KB)
constexpr int kXtSmemQ = 0;
constexpr int kXtSmemK = kXtSmemQ + 2 * kXtQHalfBytes;        // 64 KB
constexpr int kXtSmemHist = kXtSmemK + kXtStages * kTcTileBytes;   // + 128 KB
constexpr int kXtSmemEx = kXtSmemHist + kBins1 * 4;           // float [2 buffers][2 column halves][128 tokens]
constexpr int kXtSmemBar = kXtSmemEx + 2 * 2 * 128 * 4;
constexpr int kXtSmemBytes = kXtSmemBar + 256;
enum { kXtBarKFull = 0, kXtBarKEmpty = kXtStages, kXtBarQFull = 2 * kXtStages, kXtBarQFree, kXtBarDFull, kXtBarDEmpty = kXtBarDFull + 2, kXtBarCount = kXtBarDEmpty + 2 };
constexpr int kXtTmemPtrOff = 8 * kXtBarCount;
static_assert(kXtTmemPtrOff + 4 <= 256 && kXtSmemBytes <= 232448 - 1024, "shared memory of the x-query tcgen05 scan");

struct ScanXqTcParams {
    const int32_t* page_table;
    const int32_t* seq_lens;
    float* scores;                // [units][max_seq_len]
    uint32_t* hist1;              // [units][kBins1]
    int32_t batch, n_q_heads, n_kv_heads, max_seq_len, max_pages, x;
    int32_t set_size;             // H_kv: CTA sets share (sequence, tile) ranges, one head each; 1: ranges of the (unit, tile) space
    float sm_scale;
};

// Walk the segments of this CTA: f(b, h, L, tile_lo, tile_hi, seg).  With sets, [g0, g1) is a range of the (sequence,
// tile) space and the CTA's head is fixed; without, a range of the (unit, tile) space.
template <typename F>
__device__ __forceinline__ void xt_for_each_segment(const ScanXqTcParams& p, int64_t g0, int64_t g1, int my_h, F&& f) {
    int64_t begin = 0;
    int seg = 0;
    for (int b = 0; b < p.batch && begin < g1; ++b) {
        const int L = min(p.seq_lens[b], p.max_seq_len);
        const int n_t = (L + kTcBN - 1) / kTcBN;
        const int h_lo = my_h >= 0 ? my_h : 0, h_hi = my_h >= 0 ? my_h + 1 : p.n_kv_heads;
        for (int h = h_lo; h < h_hi; ++h, begin += n_t) {
            const int64_t lo = max(g0, begin), hi = min(g1, begin + n_t);
            if (lo >= hi) continue;
            f(b, h, L, (int)(lo - begin), (int)(hi - begin), seg);
            ++seg;
        }
    }
}

__global__ void __launch_bounds__(kXtThreads, 1)
scan_xq_tc_kernel(const __grid_constant__ CUtensorMap tm_k, const __grid_constant__ CUtensorMap tm_q, const ScanXqTcParams p) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t sbase = smem_u32(smem_raw);
    if (sbase & 1023u) __trap();   // the 128B-swizzled tiles need a 1024 B aligned base
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int G = p.n_q_heads / p.n_kv_heads;
    const int rows = p.x * G, n_pad = (rows + 15) & ~15;     // UMMA N: a multiple of 16; the pad rows are never read out
    auto bar = [&](int i) { return sbase + kXtSmemBar + 8u * i; };
    uint32_t* s_hist = reinterpret_cast<uint32_t*>(smem_raw + kXtSmemHist);
    float* s_ex = reinterpret_cast<float*>(smem_raw + kXtSmemEx);
    volatile uint32_t* tmem_ptr_gen = reinterpret_cast<volatile uint32_t*>(smem_raw + kXtSmemBar + kXtTmemPtrOff);

    if (warp == kXtMmaWarp) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(sbase + kXtSmemBar + kXtTmemPtrOff), "n"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    } else if (warp == kXtTmaWarp) {
        if (lane == 0) {
            for (int s = 0; s < kXtStages; ++s) {
                mbar_init(bar(kXtBarKFull + s), 1);
                mbar_init(bar(kXtBarKEmpty + s), 1);
            }
            mbar_init(bar(kXtBarQFull), 1);
            mbar_init(bar(kXtBarQFree), 1);
            for (int s = 0; s < 2; ++s) {
                mbar_init(bar(kXtBarDFull + s), 1);
                mbar_init(bar(kXtBarDEmpty + s), kXtEpiWarps);
            }
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_q) : "memory");
            asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_k) : "memory");
        }
    } else {
        for (int i = tid; i < kBins1; i += kXtEpiWarps * 32) s_hist[i] = 0;
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_ptr_gen;

    // the range of this CTA (every role computes it from the inputs alone)
    const bool sets = p.set_size > 1;
    const int my_h = sets ? (int)(blockIdx.x % p.set_size) : -1;
    const int n_ranges = sets ? (int)(gridDim.x / p.set_size) : (int)gridDim.x, range = sets ? (int)(blockIdx.x / p.set_size) : (int)blockIdx.x;
    int64_t total = 0;
    for (int b = 0; b < p.batch; ++b) total += (int64_t)((min(p.seq_lens[b], p.max_seq_len) + kTcBN - 1) / kTcBN) * (sets ? 1 : p.n_kv_heads);
    // (CTAs past the last whole set have no range)
    const int64_t g0 = range < n_ranges ? cta_range_begin(total, range, n_ranges) : 0, g1 = range < n_ranges ? cta_range_begin(total, range + 1, n_ranges) : 0;

    if (warp == kXtTmaWarp) {
        // =========================== producer: the unit's query rows, then its K tiles ===========================
        int kt = 0;
        xt_for_each_segment(p, g0, g1, my_h, [&](int b, int h, int L, int tile_lo, int tile_hi, int seg) {
            auto load_q = [&]() {
                if (seg > 0) mbar_wait(bar(kXtBarQFree), (seg - 1) & 1);    // the MMAs of the previous unit are done with Q
                if (elect_one()) {
                    // q_x [batch][x][H_q][128]: box = (64 channels, G heads, x queries) per half -> rows rho = j*G + g
                    mbar_arrive_expect_tx(bar(kXtBarQFull), (uint32_t)rows * 256u);
                    tma_load_4d(sbase + kXtSmemQ, &tm_q, 0, h * G, 0, b, bar(kXtBarQFull));
                    tma_load_4d(sbase + kXtSmemQ + kXtQHalfBytes, &tm_q, 64, h * G, 0, b, bar(kXtBarQFull));
                }
                __syncwarp();
            };
            // At a unit boundary the K ring keeps filling with the new unit's tiles while the MMAs finish the old one;
            // only the query rows wait for them (after up to kXtStages - 1 tiles are on their way).
            const int q_after = seg == 0 ? -1 : min(kXtStages - 1, tile_hi - tile_lo) - 1;
            if (q_after < 0) load_q();
            // the 128 tokens of a tile are 8 pages of the cache; page i lands on tile rows [16i, 16i+16) (2 KB per half: whole
            // 1 KB swizzle atoms).  Pages past the sequence are not requested: their rows are never read out.  The page
            // ids of the next tile are fetched before waiting for its ring slot.
            const int32_t* pt = p.page_table + (int64_t)b * p.max_pages;
            auto tile_pages = [&](int t) { return (min(kTcBN, L - t * kTcBN) + kPageSize - 1) / kPageSize; };
            int n_pg = tile_pages(tile_lo);
            int my_phys = lane < n_pg ? __ldg(pt + tile_lo * (kTcBN / kPageSize) + lane) : 0;
            for (int t = tile_lo; t < tile_hi; ++t, ++kt) {
                const int stage = kt % kXtStages;
                const int n_pg_next = t + 1 < tile_hi ? tile_pages(t + 1) : 0;
                const int phys_next = lane < n_pg_next ? __ldg(pt + (t + 1) * (kTcBN / kPageSize) + lane) : 0;
                if (kt >= kXtStages) mbar_wait(bar(kXtBarKEmpty + stage), ((kt / kXtStages) - 1) & 1);
                const uint32_t dst = sbase + kXtSmemK + stage * kTcTileBytes, full = bar(kXtBarKFull + stage);
                if (lane == 0) mbar_arrive_expect_tx(full, (uint32_t)n_pg * kPageSize * 256u);
                __syncwarp();
                if (lane < n_pg) {
                    tma_load_4d(dst + lane * (kPageSize * 128), &tm_k, 0, h, 0, my_phys, full);
                    tma_load_4d(dst + kTcHalfBytes + lane * (kPageSize * 128), &tm_k, 64, h, 0, my_phys, full);
                }
                __syncwarp();
                if (t - tile_lo == q_after) load_q();
                n_pg = n_pg_next;
                my_phys = phys_next;
            }
        });
    } else if (warp == kXtMmaWarp) {
        // =========================== MMA issuer ===========================
        constexpr uint32_t hi_sw = umma_desc_hi(1024);
        const uint32_t q_lo = umma_desc_lo(sbase + kXtSmemQ, 16);
        const uint32_t idesc = umma_idesc(/*A bf16*/ 1, /*B bf16*/ 1, /*K-major*/ 0, 0, kTcBM, n_pad);
        int kt = 0;
        xt_for_each_segment(p, g0, g1, my_h, [&](int, int, int, int tile_lo, int tile_hi, int seg) {
            mbar_wait(bar(kXtBarQFull), seg & 1);
            for (int t = tile_lo; t < tile_hi; ++t, ++kt) {
                const int stage = kt % kXtStages, buf = kt & 1;
                mbar_wait(bar(kXtBarKFull + stage), (kt / kXtStages) & 1);
                if (kt >= 2) mbar_wait(bar(kXtBarDEmpty + buf), ((kt >> 1) - 1) & 1);
                tc_fence_after();
                if (elect_one()) {
                    const uint32_t k_lo = umma_desc_lo(sbase + kXtSmemK + stage * kTcTileBytes, 16);
                    const uint32_t d = tmem + buf * 256;
#pragma unroll
                    for (int ks = 0; ks < 8; ++ks) {
                        const uint32_t off_a = ((ks >> 2) * kTcHalfBytes + (ks & 3) * 32) >> 4;
                        const uint32_t off_b = ((ks >> 2) * kXtQHalfBytes + (ks & 3) * 32) >> 4;
                        if (ks == 0) umma_ss<false>(d, k_lo + off_a, hi_sw, q_lo + off_b, hi_sw, idesc);
                        else umma_ss<true>(d, k_lo + off_a, hi_sw, q_lo + off_b, hi_sw, idesc);
                    }
                    umma_commit(bar(kXtBarDFull + buf));
                    umma_commit(bar(kXtBarKEmpty + stage));
                }
                __syncwarp();
            }
            if (elect_one()) umma_commit(bar(kXtBarQFree));
            __syncwarp();
        });
    } else {
        // =========================== read-out: per-token maximum over the x*G columns ===========================
        const int quarter = warp & 3, half = warp >> 2;
        const int row = quarter * 32 + lane;                  // token of the tile == TMEM lane
        const uint32_t lane_base = tmem + ((uint32_t)(quarter * 32) << 16);
        const int n_chunks = (rows + 31) >> 5;
        int dt = 0;
        xt_for_each_segment(p, g0, g1, my_h, [&](int b, int h, int L, int tile_lo, int tile_hi, int) {
            const int unit = b * p.n_kv_heads + h;
            float* score_row = p.scores + (int64_t)unit * p.max_seq_len;
            for (int t = tile_lo; t < tile_hi; ++t, ++dt) {
                const int buf = dt & 1;
                mbar_wait(bar(kXtBarDFull + buf), (dt >> 1) & 1);
                tc_fence_after();
                float m = -INFINITY;
                for (int c = half; c < n_chunks; c += 2) {
                    float v[32];
                    tmem_ld32_async(lane_base + buf * 256 + 32 * c, v);
                    tmem_wait_ld();
                    const int lim = rows - 32 * c;
                    if (lim >= 32) {
#pragma unroll
                        for (int i = 0; i < 32; i += 2) m = fmax3(m, v[i], v[i + 1]);
                    } else {
#pragma unroll
                        for (int i = 0; i < 32; ++i) m = fmaxf(m, i < lim ? v[i] : -INFINITY);
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(kXtBarDEmpty + buf));       // the MMAs of tile dt + 2 may overwrite the buffer
                s_ex[(buf * 2 + half) * 128 + row] = m;
                named_bar_sync(1, kXtEpiWarps * 32);
                const int tok = t * kTcBN + row;
                if (half == 0 && tok < L) {
                    const float v = fmaxf(m, s_ex[(buf * 2 + 1) * 128 + row]) * p.sm_scale;
                    score_row[tok] = v;
                    atomicAdd(&s_hist[score_key(v) >> (32 - kBits1)], 1u);
                }
            }
            // ---- end of this CTA's share of the unit: flush the histogram ----
            named_bar_sync(1, kXtEpiWarps * 32);
            uint32_t* gh = p.hist1 + (int64_t)unit * kBins1;
            for (int i = tid; i < kBins1; i += kXtEpiWarps * 32) {
                const uint32_t v = s_hist[i];
                if (v) {
                    atomicAdd(gh + i, v);
                    s_hist[i] = 0;
                }
            }
            named_bar_sync(1, kXtEpiWarps * 32);
        });
    }
    tc_fence_before();
    __syncthreads();
    if (warp == kXtMmaWarp) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(512));
    }
}

}  // namespace herald
