// Exact per-(sequence, KV head) top-k of the score plane (step a3 of DESIGN.md).
//
// The paper keeps a min-heap on the CPU; on the GPU the same result (the k largest scores, ties to
// the lower position, emitted in ascending position) is an MSB-first radix select on an order-preserving
// 32-bit key (12 + 10 + 10 bits).  One 1024-thread CTA per unit.
//   level 1 histogram : already accumulated by the scan kernel's epilogue (hist1) -> threshold bin b1
//   fast path (the threshold bin holds <= cand_cap scores, positions < 32 * bitmap_words; both sized by the launcher
//   from max_seq_len so that two CTAs share an SM on the common shapes):
//     ONE pass over the score plane: scores above bin b1 set their bit in a shared-memory position bitmap,
//     scores inside bin b1 are appended (key, position) to a shared-memory candidate list (warp-aggregated);
//     levels 2 and 3 run on the candidate list; exact ties keep the lowest positions through a second bitmap
//     and a block prefix sum; the result is emitted in ascending position from the bitmap (popcount prefix).
//   slow path (anything else, e.g. all scores equal): levels 2 and 3 re-read the plane from L2 and an ordered
//     compaction by block prefix sums emits the positions.
#pragma once
#include "common.cuh"

namespace herald {

constexpr int kTopkThreads = 1024;
constexpr int kTopkMaxCandCap = 12288;              // (key, position) pairs of the threshold bin held in shared memory, at most
constexpr int kTopkMaxBitmapWords = 8192;           // one bit per position: fast path for L <= 262144
constexpr int kTopkMaxSmemBytes = kTopkMaxCandCap * 8 + 2 * kTopkMaxBitmapWords * 4;   // candidates, selected bitmap, tie bitmap

// Find bin j with  count(bins > j) < kk <= count(bins >= j).  Returns j, *above = count(bins > j).
// hist has nbins (multiple of blockDim) entries in shared memory; every thread must call.
__device__ __forceinline__ uint32_t find_threshold_bin(const uint32_t* hist, int nbins, uint32_t kk,
                                                        uint32_t* warp_sums, uint32_t* res, uint32_t* above) {
    const int per = nbins / kTopkThreads;          // 4 or 1
    const int r0 = threadIdx.x * per;              // reversed index: r = nbins-1-bin
    uint32_t local = 0;
    for (int e = 0; e < per; ++e) local += hist[nbins - 1 - (r0 + e)];
    uint32_t total;
    const uint32_t before = block_exclusive_scan(local, warp_sums, &total);
    if (before < kk && kk <= before + local) {
        uint32_t acc = before;
        for (int e = 0; e < per; ++e) {
            const uint32_t c = hist[nbins - 1 - (r0 + e)];
            if (kk <= acc + c) {
                res[0] = nbins - 1 - (r0 + e);
                res[1] = acc;
                break;
            }
            acc += c;
        }
    }
    __syncthreads();
    *above = res[1];
    return res[0];
}

#ifndef HERALD_TOPK_UNROLL
#define HERALD_TOPK_UNROLL 4
#endif
constexpr int kTopkUnroll = HERALD_TOPK_UNROLL;

struct TopkParams {
    const float* scores;       // [units][max_seq_len]
    const uint32_t* hist1;     // [units][kBins1]
    const int32_t* seq_lens;   // [batch]
    const int32_t* k_per_seq;  // [batch]
    int32_t* sel_idx;          // [units][cap]
    int32_t* sel_cnt;          // [units]
    int32_t n_kv_heads, max_seq_len, cap;
    int32_t cand_cap, bitmap_words;   // dynamic shared memory = cand_cap * 8 + 2 * bitmap_words * 4 bytes
};

__global__ void __launch_bounds__(kTopkThreads, 2) topk_kernel(const TopkParams p) {
    __shared__ uint32_t s_hist[kBins1];
    __shared__ uint32_t s_warp[33];
    __shared__ uint32_t s_res[2];
    __shared__ uint32_t s_ncand;

    // herald_select_rep launches this grid programmatically behind the K+V pass and the partial merge behind this one:
    // wait for the pass (scores, histogram), then let the merge start beside us.  No-ops in an ordinary launch.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;");
    const int unit = blockIdx.x;
    const int b = unit / p.n_kv_heads;
    const int L = min(p.seq_lens[b], p.max_seq_len);
    const int kk = min(min(p.k_per_seq[b], L), p.cap);
    if (kk <= 0) {
        if (threadIdx.x == 0) p.sel_cnt[unit] = 0;
        return;
    }
    const float* sc = p.scores + (int64_t)unit * p.max_seq_len;
    int32_t* out = p.sel_idx + (int64_t)unit * p.cap;
    const int tid = threadIdx.x;

    if (tid == 0) { s_res[0] = 0; s_res[1] = 0; s_ncand = 0; }
    {   // the level-1 histogram: all loads of a thread in flight at once
        static_assert(kBins1 % kTopkThreads == 0, "histogram load");
        uint32_t hv[kBins1 / kTopkThreads];
#pragma unroll
        for (int j = 0; j < kBins1 / kTopkThreads; ++j) hv[j] = __ldg(p.hist1 + (int64_t)unit * kBins1 + j * kTopkThreads + tid);
#pragma unroll
        for (int j = 0; j < kBins1 / kTopkThreads; ++j) s_hist[j * kTopkThreads + tid] = hv[j];
    }
    __syncthreads();
    uint32_t above1, above2, above3;
    const uint32_t b1 = find_threshold_bin(s_hist, kBins1, (uint32_t)kk, s_warp, s_res, &above1);
    const uint32_t k2 = kk - above1;

    const uint32_t n_c = s_hist[b1];                   // scores inside the threshold bin
    if (n_c <= (uint32_t)p.cand_cap && L <= 32 * p.bitmap_words) {
        // ---------------- fast path: one pass over the plane ----------------
        extern __shared__ __align__(16) uint8_t topk_smem[];
        uint2* cand = reinterpret_cast<uint2*>(topk_smem);                                   // (key, position)
        uint32_t* bitmap = reinterpret_cast<uint32_t*>(topk_smem + (size_t)p.cand_cap * 8);  // selected positions
        uint32_t* tiemap = bitmap + p.bitmap_words;                                          // positions with key == T
        const int n_words = (L + 31) >> 5;
        const int lane = tid & 31;
        for (int i = tid; i < n_words; i += kTopkThreads) tiemap[i] = 0;
        const uint32_t k_lo = b1 << (32 - kBits1), k_top = k_lo | ((1u << (32 - kBits1)) - 1u);   // the keys of the threshold bin
        __syncthreads();
        // kTopkUnroll independent 16-byte loads per thread are issued before the first of them is used: at L = 131072
        // the pass is 32 trips of one load each otherwise, and each trip waits for a whole L2 round trip.
        // The candidates among the 4 * kTopkUnroll scores of a trip are appended with ONE shared-memory atomic per warp: a
        // ballot + atomic + shuffle per score made the pass a chain of ~30 atomic round trips per warp on one address.
        // The order of the candidate list does not matter.
        for (int tile = 0; tile < L; tile += kTopkThreads * 4 * kTopkUnroll) {
            float4 vv[kTopkUnroll];
#pragma unroll
            for (int u = 0; u < kTopkUnroll; ++u) {
                const int i = tile + (u * kTopkThreads + tid) * 4;
                vv[u] = i < L ? *reinterpret_cast<const float4*>(sc + i) : make_float4(0.f, 0.f, 0.f, 0.f);
            }
            uint32_t cmask = 0;                    // bit 4u + e: score e of load u lies in the threshold bin [k_lo, k_top]
#pragma unroll
            for (int u = 0; u < kTopkUnroll; ++u) {
                const int i = tile + (u * kTopkThreads + tid) * 4;
                if (tile + u * kTopkThreads * 4 >= L) break;   // uniform over the block
                const float ve[4] = {vv[u].x, vv[u].y, vv[u].z, vv[u].w};
                uint32_t above = 0, cm = 0;
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const uint32_t key = score_key(ve[e]);
                    above |= (key > k_top ? 1u : 0u) << e;
                    cm |= (key >= k_lo ? 1u : 0u) << e;
                }
                cm &= ~above;
                if (i + 3 >= L) {                  // the last load of the plane: positions past L do not count
                    const uint32_t valid = i < L ? (1u << (L - i)) - 1u : 0u;
                    above &= valid;
                    cm &= valid;
                }
                cmask |= cm << (4 * u);
                // 8 neighbouring lanes hold the 32 positions of one bitmap word (bit 4 * (lane & 7) + e): the word is put
                // together with three shuffles and written once by the first of them -- no atomics, and every word below
                // n_words is written, so none needs clearing
                uint32_t word = above << (4 * (lane & 7));
                word |= __shfl_xor_sync(0xffffffffu, word, 1);
                word |= __shfl_xor_sync(0xffffffffu, word, 2);
                word |= __shfl_xor_sync(0xffffffffu, word, 4);
                if ((lane & 7) == 0 && i < L) bitmap[i >> 5] = word;
            }
            if (__any_sync(0xffffffffu, cmask != 0)) {
                // warp-inclusive scan of the candidate counts, one atomic for the warp's total of the trip
                const uint32_t mine = __popc(cmask);
                uint32_t incl = mine;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const uint32_t n = __shfl_up_sync(0xffffffffu, incl, o);
                    if (lane >= o) incl += n;
                }
                uint32_t base = 0;
                if (lane == 31) base = atomicAdd(&s_ncand, incl);
                base = __shfl_sync(0xffffffffu, base, 31) + incl - mine;
#pragma unroll
                for (int u = 0; u < kTopkUnroll; ++u) {
                    if ((cmask >> (4 * u)) & 15u) {
                        const int i = tile + (u * kTopkThreads + tid) * 4;
                        const float ve[4] = {vv[u].x, vv[u].y, vv[u].z, vv[u].w};
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            if (cmask & (1u << (4 * u + e))) cand[base++] = make_uint2(score_key(ve[e]), (uint32_t)(i + e));
                    }
                }
            }
        }
        __syncthreads();
        // levels 2 and 3 on the candidates: the k2 largest of the low 20 key bits
        for (int i = tid; i < kBins2; i += kTopkThreads) s_hist[i] = 0;
        __syncthreads();
        for (uint32_t c = tid; c < n_c; c += kTopkThreads) atomicAdd(&s_hist[(cand[c].x >> kBits3) & (kBins2 - 1)], 1u);
        __syncthreads();
        uint32_t above2f, above3f;
        const uint32_t b2f = find_threshold_bin(s_hist, kBins2, k2, s_warp, s_res, &above2f);
        const uint32_t k3f = k2 - above2f;
        __syncthreads();
        for (int i = tid; i < kBins3; i += kTopkThreads) s_hist[i] = 0;
        __syncthreads();
        for (uint32_t c = tid; c < n_c; c += kTopkThreads) {
            const uint32_t key = cand[c].x;
            if (((key >> kBits3) & (kBins2 - 1)) == b2f) atomicAdd(&s_hist[key & (kBins3 - 1)], 1u);
        }
        __syncthreads();
        const uint32_t b3f = find_threshold_bin(s_hist, kBins3, k3f, s_warp, s_res, &above3f);
        const uint32_t need_f = k3f - above3f;          // exact ties (key == T) to keep, lowest positions first
        const uint32_t T = (b1 << (32 - kBits1)) | (b2f << kBits3) | b3f;
        // the level-3 count of the threshold bin is the number of scores equal to T: when all of them are kept (the usual case:
        // one score sits on the threshold) they go straight into the bitmap and the tie phase with its block scan is skipped
        const bool all_ties = s_hist[b3f] == need_f;
        for (uint32_t c = tid; c < n_c; c += kTopkThreads) {
            const uint2 kc = cand[c];
            if (kc.x > T || (all_ties && kc.x == T)) atomicOr(&bitmap[kc.y >> 5], 1u << (kc.y & 31));
            else if (kc.x == T) atomicOr(&tiemap[kc.y >> 5], 1u << (kc.y & 31));
        }
        __syncthreads();
        const int wpt = (n_words + kTopkThreads - 1) / kTopkThreads;   // words per thread (<= 8), contiguous
        const int w0 = tid * wpt, w1 = min(n_words, w0 + wpt);
        if (!all_ties) {   // ties: keep the first need_f in position order (block-uniform branch)
            uint32_t cnt = 0;
            for (int wd = w0; wd < w1; ++wd) cnt += __popc(tiemap[wd]);
            uint32_t total;
            uint32_t before = block_exclusive_scan(cnt, s_warp, &total);
            for (int wd = w0; wd < w1 && before < need_f; ++wd) {
                uint32_t t = tiemap[wd], keep = 0;
                while (t && before < need_f) {
                    const uint32_t bit = t & (0u - t);
                    keep |= bit;
                    t ^= bit;
                    ++before;
                }
                bitmap[wd] |= keep;                     // this thread owns word wd in this phase
            }
            __syncthreads();
        }
        {   // emit the set positions in ascending order: staged in the candidate list's memory (dead by now) when they fit, so
            // that the global stores are coalesced instead of ~6 consecutive ints per thread
            uint32_t cnt = 0;
            for (int wd = w0; wd < w1; ++wd) cnt += __popc(bitmap[wd]);
            uint32_t total;
            uint32_t at = block_exclusive_scan(cnt, s_warp, &total);
            const bool staged = kk <= 2 * p.cand_cap;       // block-uniform
            int32_t* dst = staged ? reinterpret_cast<int32_t*>(cand) : out;
            for (int wd = w0; wd < w1; ++wd) {
                uint32_t t = bitmap[wd];
                while (t) {
                    dst[at++] = wd * 32 + __ffs(t) - 1;
                    t &= t - 1;
                }
            }
            if (staged) {
                __syncthreads();
                for (int i = tid; i < kk; i += kTopkThreads) out[i] = dst[i];
            }
        }
        if (tid == 0) p.sel_cnt[unit] = kk;
        return;
    }

    // ---------------- slow path: levels 2 and 3 and the compaction re-read the plane ----------------
    // level 2: next 10 bits, restricted to level-1 bin b1
    __syncthreads();
    for (int i = tid; i < kBins2; i += kTopkThreads) s_hist[i] = 0;
    __syncthreads();
    for (int i = tid * 4; i < L; i += kTopkThreads * 4) {
        const float4 v = *reinterpret_cast<const float4*>(sc + i);
        const float ve[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            if (i + e < L) {
                const uint32_t key = score_key(ve[e]);
                if ((key >> (32 - kBits1)) == b1) atomicAdd(&s_hist[(key >> kBits3) & (kBins2 - 1)], 1u);
            }
        }
    }
    __syncthreads();
    const uint32_t b2 = find_threshold_bin(s_hist, kBins2, k2, s_warp, s_res, &above2);
    const uint32_t k3 = k2 - above2;
    const uint32_t prefix22 = (b1 << kBits2) | b2;

    // level 3: last 10 bits, restricted to the 22-bit prefix
    __syncthreads();
    for (int i = tid; i < kBins3; i += kTopkThreads) s_hist[i] = 0;
    __syncthreads();
    for (int i = tid * 4; i < L; i += kTopkThreads * 4) {
        const float4 v = *reinterpret_cast<const float4*>(sc + i);
        const float ve[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            if (i + e < L) {
                const uint32_t key = score_key(ve[e]);
                if ((key >> kBits3) == prefix22) atomicAdd(&s_hist[key & (kBins3 - 1)], 1u);
            }
        }
    }
    __syncthreads();
    const uint32_t b3 = find_threshold_bin(s_hist, kBins3, k3, s_warp, s_res, &above3);
    const uint32_t need = k3 - above3;                 // ties (key == T) to keep, lowest positions first
    const uint32_t T = (prefix22 << kBits3) | b3;

    // ordered compaction
    uint32_t base_gt = 0, base_eq = 0;
    for (int tile = 0; tile < L; tile += kTopkThreads * 4) {
        const int i = tile + tid * 4;
        uint32_t flag_gt = 0, flag_eq = 0;
        if (i < L) {
            const float4 v = *reinterpret_cast<const float4*>(sc + i);
            const float ve[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                if (i + e < L) {
                    const uint32_t key = score_key(ve[e]);
                    flag_gt |= (key > T ? 1u : 0u) << e;
                    flag_eq |= (key == T ? 1u : 0u) << e;
                }
            }
        }
        const uint32_t packed = __popc(flag_gt) | (__popc(flag_eq) << 16);
        uint32_t total;
        const uint32_t excl = block_exclusive_scan(packed, s_warp, &total);
        uint32_t gt_before = base_gt + (excl & 0xffffu);
        uint32_t eq_before = base_eq + (excl >> 16);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            if (flag_gt & (1u << e)) {
                out[gt_before + min(eq_before, need)] = i + e;
                ++gt_before;
            } else if (flag_eq & (1u << e)) {
                if (eq_before < need) out[gt_before + eq_before] = i + e;
                ++eq_before;
            }
        }
        base_gt += total & 0xffffu;
        base_eq += total >> 16;
    }
    if (tid == 0) p.sel_cnt[unit] = kk;
}

}  // namespace herald
