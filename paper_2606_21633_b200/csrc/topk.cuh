// Exact per-(sequence, KV head) top-k of the score plane (step a3 of DESIGN.md).
//
// The paper keeps a min-heap on the CPU; on the GPU the same result (the k largest scores, ties to
// the lower position, emitted in ascending position) is a three-level MSB-first radix select on an
// order-preserving 32-bit key (12 + 10 + 10 bits) followed by an ordered compaction:
//   level 1 histogram : already accumulated by the scan kernel's epilogue (hist1),
//   level 2, 3        : histograms of the elements inside the threshold bin (few smem atomics),
//   compaction        : keys > T, plus the first `need` keys == T in position order, via block scans.
// One 1024-thread CTA per unit; the score plane (<= 512 KB per unit) is read from L2.
#pragma once
#include "common.cuh"

namespace herald {

constexpr int kTopkThreads = 1024;

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

struct TopkParams {
    const float* scores;       // [units][max_seq_len]
    const uint32_t* hist1;     // [units][kBins1]
    const int32_t* seq_lens;   // [batch]
    const int32_t* k_per_seq;  // [batch]
    int32_t* sel_idx;          // [units][cap]
    int32_t* sel_cnt;          // [units]
    int32_t n_kv_heads, max_seq_len, cap;
};

__global__ void __launch_bounds__(kTopkThreads, 1) topk_kernel(const TopkParams p) {
    __shared__ uint32_t s_hist[kBins1];
    __shared__ uint32_t s_warp[33];
    __shared__ uint32_t s_res[2];

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

    if (tid == 0) { s_res[0] = 0; s_res[1] = 0; }
    for (int i = tid; i < kBins1; i += kTopkThreads) s_hist[i] = p.hist1[(int64_t)unit * kBins1 + i];
    __syncthreads();
    uint32_t above1, above2, above3;
    const uint32_t b1 = find_threshold_bin(s_hist, kBins1, (uint32_t)kk, s_warp, s_res, &above1);
    const uint32_t k2 = kk - above1;

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
