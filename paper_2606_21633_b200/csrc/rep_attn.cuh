// Attention output of the representative query itself (NEXT-2 of DESIGN.md; section IV-B4: the fused
// selection kernel "maintains the FlashAttention statistics (m_g, l_g, o_g)" next to the raw scores, and PAPER.md:193:
// that output goes back to the layer's FFN).
//
//   o[b, hq, :] = softmax_t( sm_scale * q_rep[b, hq] . K[b, t, h] ) . V[b, t, h, :]   over every cached t < seq_lens[b]
//
// One query row per head: there is no dense contraction to give to tcgen05 (M = G <= 8), and the kernel is a second
// HBM stream, now over K AND V (512 B per token and KV head).  Scores come from the same mma.sync trick as the score
// scan (fed from 128-bit global loads); the P.V product runs on mma.sync too (G x 128 FMAs per token on the CUDA cores
// made the kernel FMA-pipe bound at G = 7), in the transposed form described at the kernel.
//   Page-major like the score scan: a page holds the rows of all KV heads side by side (256 B per head and token), so
//   the CTA's 8 warps take `hg` heads of the same pages at once (hg = the largest of 8, 4, 2, 1 dividing H_kv) and
//   DRAM sees whole pages instead of 256-byte pieces.  A "group" is (sequence, hg consecutive heads).
//   The grid is flat and persistent (two CTAs per SM): the (group, page) space is cut into gridDim.x equal ranges, so
//   ragged lengths cost no wave tail.  Where a range meets a group, warp w takes head w % hg and strides over those
//   pages from slot w / hg with its own online softmax; warps merge in shared memory and write one partial (m, l, o)
//   per head to slot cta + group (unique: both indices only grow along the ranges).  rep_attn_merge_kernel (one block
//   per output row, every partial load independent) combines the partials of a row into out / lse.
//   Each warp keeps its NEXT page in flight while it works on the current one: the K fragments of page i+1 are loaded
//   into the fragment registers as soon as the score MMAs of page i have consumed them, and the V rows of page i+1 go
//   by cp.async into the other half of a per-warp double buffer (2 x 4 KB).  Without that each page costs a warp one
//   exposed DRAM round trip and the kernel is latency-bound.
#pragma once
#include "common.cuh"

namespace herald {

constexpr int kRepThreads = 256;
constexpr int kRepWarps = kRepThreads / 32;
constexpr int kRepMaxCtas = 512;                      // partial slots are cta + group: the workspace holds (kRepMaxCtas + groups) x hg head partials
constexpr int kRepPartFloats = 8 * (kHeadDim + 2);    // per (range, unit): 8 head slots x (128 channels, m, l)
constexpr int kRepVStageBytes = kPageSize * kHeadDim * 2;                 // one page of V rows of one head: 4 KB
constexpr int kRepSmemV = kRepWarps * 2 * kRepVStageBytes;                 // V double buffers; reused as s_o after the loop
constexpr int kRepSmemBytes = kRepSmemV;
static_assert(kRepWarps * 8 * (kHeadDim + 4) * 4 <= kRepSmemV, "s_o must fit in the V stages it reuses");

__device__ __forceinline__ void cp_async_16(uint32_t dst, const void* src, uint32_t src_bytes) {   // src_bytes 0: zero fill
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

struct RepAttnParams {
    const __nv_bfloat16* k_pages;
    const __nv_bfloat16* v_pages;
    int64_t page_stride, token_stride, head_stride;
    const int32_t* page_table;
    const int32_t* seq_lens;
    const __nv_bfloat16* q_rep;
    float* part;          // [gridDim.x + groups][hg][8][130], slot = cta + group
    float* out;           // [batch][H_q][128]
    float* lse;           // optional [batch][H_q]
    float* scores;        // optional [units][max_seq_len]: the selection scores of the same pass (herald_select_rep), mode 0
    uint32_t* hist1;      // with scores: [units][kBins1] level-1 histogram of the top-k (zeroed before the launch)
    float* raw;           // optional [units][G][max_seq_len]: the per-head scaled logits, for the softmax-sum aggregation (mode 1)
    float sm_scale;
    int32_t merge_waits;  // the merge grid waits for its predecessor (0: it is launched behind a grid that already did)
    int32_t batch, n_q_heads, n_kv_heads, max_seq_len, max_pages, hg;
    float scale_log2;     // sm_scale * log2(e): the softmax runs in base 2
};

__device__ __forceinline__ void ldmatrix_x4_trans(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
                 : "r"(addr));
}

// Both products run TRANSPOSED on mma.sync so that the weights never leave the registers:
//   S^T[head, token]   = Q[head, :] . K[token, :]      A = Q (rows 8..15 zero), B = K fragments straight from global
//   O^T[channel, head] += V^T[channel, token] P^T[token, head]
// The accumulator of the first product (head g; tokens 2tig, 2tig+1, 8+2tig, 9+2tig) IS the B fragment of the second
// once exponentiated and packed; V^T comes from ldmatrix.trans on the V rows staged in shared memory (16-byte columns
// XOR-swizzled by the row).  P goes in as a bf16 pair hi + lo (two MMAs): the weights keep ~16 mantissa bits.
// CTA whose range holds global page x:  begin(i) = total * i / n  <=  x   <=>   i <= ceil((x + 1) n / total) - 1
__device__ __forceinline__ int rep_cta_of(int64_t x, int64_t total, int n) { return (int)(((x + 1) * n + total - 1) / total) - 1; }

__global__ void __launch_bounds__(kRepThreads, 2) rep_attn_kernel(const RepAttnParams p) {
    extern __shared__ __align__(128) unsigned char rep_smem[];
    __shared__ int64_t s_total;
    float (*s_o)[8][kHeadDim + 4] = reinterpret_cast<float (*)[8][kHeadDim + 4]>(rep_smem);   // per-warp results for the merge (rows of 528 B), over the V stages
    const int G = p.n_q_heads / p.n_kv_heads;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 2, tig = lane & 3;
    const int n_ctas = gridDim.x, cta = blockIdx.x;
    asm volatile("griddepcontrol.launch_dependents;");       // the merge grid may be scheduled as this grid's CTAs retire
    const int hg = p.hg, n_groups = p.n_kv_heads / hg, n_slots = kRepWarps / hg;
    const int w_head = warp % hg, w_slot = warp / hg;         // this warp: head inside the group, first page slot
    if (threadIdx.x == 0) {
        int64_t total = 0;
        for (int b = 0; b < p.batch; ++b) total += (int64_t)((min(p.seq_lens[b], p.max_seq_len) + kPageSize - 1) / kPageSize) * (p.n_kv_heads / p.hg);
        s_total = total;
    }
    __syncthreads();
    const int64_t total = s_total;
    const int64_t g0 = total * cta / n_ctas, g1 = total * (cta + 1) / n_ctas;
    const uint32_t v_stage = smem_u32(rep_smem + warp * 2 * kRepVStageBytes);
    // ldmatrix row address of this lane inside a stage, for channel tile 0: matrix j = lane/8 is (tokens 8(j/2).., 16-byte
    // column j%2), row lane%8; the column index is XORed with (token & 7) = lane%8
    const int lm_tok = (lane & 7) + 8 * (lane >> 4), lm_col = (lane >> 3) & 1;

    int64_t unit_begin = 0;   // global page index of the current group's page 0
    for (int b = 0; b < p.batch && unit_begin < g1; ++b) {
      const int L = min(p.seq_lens[b], p.max_seq_len);
      const int n_pages = (L + kPageSize - 1) / kPageSize;
      const int32_t* pt = p.page_table + (int64_t)b * p.max_pages;
      for (int hgrp = 0; hgrp < n_groups; ++hgrp, unit_begin += n_pages) {
        const int64_t lo = max(g0, unit_begin), hi = min(g1, unit_begin + n_pages);
        if (lo >= hi) continue;                               // block-uniform
        const int unit = b * n_groups + hgrp, h = hgrp * hg + w_head;
        const int page_lo = (int)(lo - unit_begin), page_end = (int)(hi - unit_begin), t_end = L;
        float* part = p.part + (int64_t)(cta + unit) * hg * kRepPartFloats;
        uint4 qf[4];              // A operand of the score MMA: query head g (zeros for g >= G), channel-permuted like K
        {
            const __nv_bfloat16* qrow = p.q_rep + ((int64_t)b * p.n_q_heads + h * G + g) * kHeadDim + 8 * tig;
#pragma unroll
            for (int i = 0; i < 4; ++i) qf[i] = (g < G) ? ldg_u4(qrow + 32 * i) : make_uint4(0, 0, 0, 0);
        }
        // online softmax of this warp: the lane keeps head g's running maximum (equal in the 4 lanes of a head) and its
        // share of the row sum; o[c] = O^T[channels 16c+g, 16c+g+8][heads 2tig, 2tig+1]
        float m_run = -INFINITY, l_run = 0.f, o[8][4];
#pragma unroll
        for (int c = 0; c < 8; ++c) {
#pragma unroll
            for (int j = 0; j < 4; ++j) o[c][j] = 0.f;
        }

        uint4 a[4], c[4];         // K fragments (as in the score scan) of the page in flight: token rows g and g+8
        // issue the loads of one page: K fragments into (a, c), V rows into stage `st` (rows past t_end zero-filled: their
        // weight is 0, but 0 x NaN of an unwritten cache slot is NaN)
        auto issue_page = [&](int pg, int phys, int st) {
            const int64_t tile = (int64_t)phys * p.page_stride + (int64_t)h * p.head_stride;
            const __nv_bfloat16* r0 = p.k_pages + tile + (int64_t)g * p.token_stride + 8 * tig;
            const __nv_bfloat16* r1 = p.k_pages + tile + (int64_t)(g + 8) * p.token_stride + 8 * tig;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                a[i] = ldg_stream_u4(r0 + 32 * i);
                c[i] = ldg_stream_u4(r1 + 32 * i);
            }
#pragma unroll
            for (int j = 0; j < 8; ++j) {            // 256 x 16 B: row = 2j + lane/16, 16-byte column = lane % 16
                const int row = 2 * j + (lane >> 4), col = lane & 15;
                cp_async_16(v_stage + st * kRepVStageBytes + row * (kHeadDim * 2) + ((col ^ (row & 7)) << 4),
                            p.v_pages + tile + (int64_t)row * p.token_stride + 8 * col, pg * kPageSize + row < t_end ? 16u : 0u);
            }
        };
        int page = page_lo + w_slot;
        int phys_next = 0;
        if (page < page_end) {
            issue_page(page, __ldg(pt + page), 0);
            if (page + n_slots < page_end) phys_next = __ldg(pt + page + n_slots);
        }
        cp_async_commit();
        for (int st = 0; page < page_end; page += n_slots, st ^= 1) {
            float sa[4] = {0.f, 0.f, 0.f, 0.f}, sb[4] = {0.f, 0.f, 0.f, 0.f};   // tokens 0..7 / 8..15 of the page
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                mma_bf16_16816(sa, qf[i].x, 0u, qf[i].y, 0u, a[i].x, a[i].y);
                mma_bf16_16816(sa, qf[i].z, 0u, qf[i].w, 0u, a[i].z, a[i].w);
                mma_bf16_16816(sb, qf[i].x, 0u, qf[i].y, 0u, c[i].x, c[i].y);
                mma_bf16_16816(sb, qf[i].z, 0u, qf[i].w, 0u, c[i].z, c[i].w);
            }
            // the K fragments are consumed: put the next page of this warp in flight
            if (page + n_slots < page_end) {
                issue_page(page + n_slots, phys_next, st ^ 1);
                if (page + 2 * n_slots < page_end) phys_next = __ldg(pt + page + 2 * n_slots);
            }
            cp_async_commit();
            // sa[0], sa[1]: head g, tokens 2tig, 2tig+1 ; sb[0], sb[1]: tokens 8+2tig, 9+2tig.  Mask the tail of the last page.
            const int t0 = page * kPageSize + 2 * tig;
            const bool ok0 = t0 < t_end, ok1 = t0 + 1 < t_end, ok2 = t0 + 8 < t_end, ok3 = t0 + 9 < t_end;
            if (p.raw && g < G) {
                // mode 1: a[t] = sum_g exp(s[g,t] - lse_g) needs the finished statistics; keep the logits
                float* rr = p.raw + ((int64_t)(b * p.n_kv_heads + h) * G + g) * p.max_seq_len + t0;
                if (ok0) rr[0] = sa[0] * p.sm_scale;
                if (ok1) rr[1] = sa[1] * p.sm_scale;
                if (ok2) rr[8] = sb[0] * p.sm_scale;
                if (ok3) rr[9] = sb[1] * p.sm_scale;
            }
            if (p.scores) {
                // the fused retrieval kernel: the raw scores of this pass are the selection scores too;
                // max-logit aggregation = maximum over the G heads = over the lanes with equal tig
                float r0 = g < G ? sa[0] : -INFINITY, r1 = g < G ? sa[1] : -INFINITY;
                float r2 = g < G ? sb[0] : -INFINITY, r3 = g < G ? sb[1] : -INFINITY;
#pragma unroll
                for (int off = 4; off < 32; off <<= 1) {
                    r0 = fmaxf(r0, __shfl_xor_sync(0xffffffffu, r0, off));
                    r1 = fmaxf(r1, __shfl_xor_sync(0xffffffffu, r1, off));
                    r2 = fmaxf(r2, __shfl_xor_sync(0xffffffffu, r2, off));
                    r3 = fmaxf(r3, __shfl_xor_sync(0xffffffffu, r3, off));
                }
                if (g == 0) {
                    // score plane + level-1 histogram (fire-and-forget reductions in L2: 64 KB of shared histograms per
                    // CTA would cost the second CTA of the SM)
                    float* sr = p.scores + (int64_t)(b * p.n_kv_heads + h) * p.max_seq_len + t0;
                    uint32_t* hh = p.hist1 + (int64_t)(b * p.n_kv_heads + h) * kBins1;
                    const float v0 = r0 * p.sm_scale, v1 = r1 * p.sm_scale, v2 = r2 * p.sm_scale, v3 = r3 * p.sm_scale;
                    if (ok0) { sr[0] = v0; atomicAdd(hh + (score_key(v0) >> (32 - kBits1)), 1u); }
                    if (ok1) { sr[1] = v1; atomicAdd(hh + (score_key(v1) >> (32 - kBits1)), 1u); }
                    if (ok2) { sr[8] = v2; atomicAdd(hh + (score_key(v2) >> (32 - kBits1)), 1u); }
                    if (ok3) { sr[9] = v3; atomicAdd(hh + (score_key(v3) >> (32 - kBits1)), 1u); }
                }
            }
            const float s0 = ok0 ? sa[0] * p.scale_log2 : -INFINITY, s1 = ok1 ? sa[1] * p.scale_log2 : -INFINITY;
            const float s2 = ok2 ? sb[0] * p.scale_log2 : -INFINITY, s3 = ok3 ? sb[1] * p.scale_log2 : -INFINITY;
            float mx = fmaxf(fmaxf(s0, s1), fmaxf(s2, s3));     // page maximum of head g: 4 values here, 4 lanes per head
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 2));
            const float m_new = fmaxf(m_run, mx);               // finite: token 0 of the page is valid
            const float alpha = (m_run == -INFINITY) ? 0.f : fast_exp2(m_run - m_new);
            m_run = m_new;
            const float p0 = ok0 ? fast_exp2(s0 - m_new) : 0.f, p1 = ok1 ? fast_exp2(s1 - m_new) : 0.f;
            const float p2 = ok2 ? fast_exp2(s2 - m_new) : 0.f, p3 = ok3 ? fast_exp2(s3 - m_new) : 0.f;
            l_run = l_run * alpha + ((p0 + p1) + (p2 + p3));
            const uint32_t h01 = pack_bf16(p0, p1), h23 = pack_bf16(p2, p3);
            const uint32_t l01 = pack_bf16(p0 - __uint_as_float(h01 << 16), p1 - __uint_as_float(h01 & 0xffff0000u));
            const uint32_t l23 = pack_bf16(p2 - __uint_as_float(h23 << 16), p3 - __uint_as_float(h23 & 0xffff0000u));
            if (__any_sync(0xffffffffu, alpha != 1.f)) {        // a maximum moved: rescale (heads 2tig, 2tig+1 live in lanes 8tig, 8tig+4)
                const float a0 = __shfl_sync(0xffffffffu, alpha, 8 * tig), a1 = __shfl_sync(0xffffffffu, alpha, 8 * tig + 4);
#pragma unroll
                for (int cc = 0; cc < 8; ++cc) {
                    o[cc][0] *= a0;
                    o[cc][1] *= a1;
                    o[cc][2] *= a0;
                    o[cc][3] *= a1;
                }
            }
            cp_async_wait<1>();       // this page's V rows (every group but the one just committed)
            __syncwarp();
            const uint32_t lm_base = v_stage + st * kRepVStageBytes + lm_tok * (kHeadDim * 2);
#pragma unroll
            for (int cc = 0; cc < 8; ++cc) {                    // channels [16cc, 16cc+16)
                uint32_t v0, v1, v2, v3;
                ldmatrix_x4_trans(lm_base + (((2 * cc + lm_col) ^ (lane & 7)) << 4), v0, v1, v2, v3);
                mma_bf16_16816(o[cc], v0, v1, v2, v3, h01, h23);
                mma_bf16_16816(o[cc], v0, v1, v2, v3, l01, l23);
            }
            __syncwarp();             // the stage is refilled two pages from now
        }
        cp_async_wait<0>();
        __syncthreads();              // s_o lies over the V stages of every warp

        // ---- merge the warps of the CTA, write the partial of (this range, this unit) ----
        l_run += __shfl_xor_sync(0xffffffffu, l_run, 1);
        l_run += __shfl_xor_sync(0xffffffffu, l_run, 2);
        if (tig == 0) {
            s_o[warp][g][kHeadDim] = m_run;
            s_o[warp][g][kHeadDim + 1] = l_run;
        }
#pragma unroll
        for (int cc = 0; cc < 8; ++cc) {
            s_o[warp][2 * tig][16 * cc + g] = o[cc][0];
            s_o[warp][2 * tig + 1][16 * cc + g] = o[cc][1];
            s_o[warp][2 * tig][16 * cc + g + 8] = o[cc][2];
            s_o[warp][2 * tig + 1][16 * cc + g + 8] = o[cc][3];
        }
        __syncthreads();
        for (int idx = threadIdx.x; idx < hg * 8 * kHeadDim; idx += kRepThreads) {   // (head of the group, head slot, channel)
            const int hh = idx >> 10, q = (idx >> 7) & 7, ch = idx & (kHeadDim - 1);
            float ms = -INFINITY;
            for (int wv = hh; wv < kRepWarps; wv += hg) ms = fmaxf(ms, s_o[wv][q][kHeadDim]);
            float num = 0.f, den = 0.f;
            for (int wv = hh; wv < kRepWarps; wv += hg) {
                const float mw = s_o[wv][q][kHeadDim];
                const float wgt = (mw == -INFINITY) ? 0.f : fast_exp2(mw - ms);
                num += wgt * s_o[wv][q][ch];
                den += wgt * s_o[wv][q][kHeadDim + 1];
            }
            float* ph = part + hh * kRepPartFloats + q * (kHeadDim + 2);
            ph[ch] = num;
            if (ch == 0) {
                ph[kHeadDim] = ms;
                ph[kHeadDim + 1] = den;
            }
        }

        __syncthreads();                                      // s_o is reused (as V stages) by the next group of the range
      }
    }
}

constexpr int kRepMergeSlices = 4;

// out[b, hq, :] = sum_c 2^(m_c - m*) o_c / sum_c 2^(m_c - m*) l_c over the partials c of the row's group; one block per
// output row, blockDim = (128 channels, 4 slices of the partial list).  No load depends on another load except through
// the row maximum, so the kernel is three short latency steps rather than a chain over the partials.
__global__ void __launch_bounds__(kHeadDim * kRepMergeSlices) rep_attn_merge_kernel(const RepAttnParams p, int n_ctas) {
    __shared__ float s_w[kRepMaxCtas];
    __shared__ float s_red[kRepMergeSlices][kHeadDim + 1];
    __shared__ float s_max[32];
    __shared__ int s_first, s_nparts;
    __shared__ int64_t s_total;
    const int row = blockIdx.x, ch = threadIdx.x, slice = threadIdx.y, tid = slice * kHeadDim + ch;
    const int G = p.n_q_heads / p.n_kv_heads, hg = p.hg, n_groups = p.n_kv_heads / hg;
    const int b = row / p.n_q_heads, hq = row % p.n_q_heads, h = hq / G, q = hq % G, hgrp = h / hg, hh = h % hg;
    const int L = min(p.seq_lens[b], p.max_seq_len), n_pages = (L + kPageSize - 1) / kPageSize;
    if (n_pages == 0) {       // no cached token: zeros, lse = -inf
        if (slice == 0) p.out[(int64_t)row * kHeadDim + ch] = 0.f;
        if (p.lse && tid == 0) p.lse[row] = -INFINITY;
        // (see the end of the kernel) completion of this grid must imply completion of the top-k it runs beside
        if (!p.merge_waits) asm volatile("griddepcontrol.wait;" ::: "memory");
        return;
    }
    if (tid == 0) {           // the row's partial list: one thread does the 64-bit divisions
        int64_t total = 0, unit_begin = 0;
        for (int bb = 0; bb < p.batch; ++bb) {
            const int64_t np = (int64_t)((min(p.seq_lens[bb], p.max_seq_len) + kPageSize - 1) / kPageSize) * n_groups;
            if (bb < b) unit_begin += np;
            total += np;
        }
        unit_begin += (int64_t)hgrp * n_pages;
        const int c_first = rep_cta_of(unit_begin, total, n_ctas);
        s_first = c_first;
        s_nparts = rep_cta_of(unit_begin + n_pages - 1, total, n_ctas) - c_first + 1;
        s_total = total;
    }
    __syncthreads();
    const int c_first = s_first, n_parts = s_nparts;
    const int64_t total = s_total;
    if (p.merge_waits) asm volatile("griddepcontrol.wait;" ::: "memory");   // launched programmatically: the partials are complete from here on
    const int group = b * n_groups + hgrp;
    const float* pq = p.part + ((int64_t)(c_first + group) * hg + hh) * kRepPartFloats + q * (kHeadDim + 2);
    const int64_t cstride = (int64_t)hg * kRepPartFloats;
    // 1. the partials' maxima (a range without pages wrote nothing: -inf), the row maximum
    float mx = -INFINITY;
    for (int c = tid; c < n_parts; c += kHeadDim * kRepMergeSlices) {
        const int cc = c_first + c;
        const bool live = total >= n_ctas || total * cc / n_ctas < total * (cc + 1) / n_ctas;   // with fewer pages than CTAs some ranges are empty
        const float m = live ? __ldcg(pq + c * cstride + kHeadDim) : -INFINITY;
        s_w[c] = m;
        mx = fmaxf(mx, m);
    }
#pragma unroll
    for (int off = 16; off; off >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, off));
    if ((tid & 31) == 0) s_max[tid >> 5] = mx;
    __syncthreads();
    float ms = (tid & 31) < kHeadDim * kRepMergeSlices / 32 ? s_max[tid & 31] : -INFINITY;
#pragma unroll
    for (int off = 16; off; off >>= 1) ms = fmaxf(ms, __shfl_xor_sync(0xffffffffu, ms, off));
    // 2. this thread's slice of the weighted sums
    float num = 0.f, den = 0.f;
#pragma unroll 8
    for (int c = slice; c < n_parts; c += kRepMergeSlices) {   // branch-free: the loads of all iterations go out together
        const float m = s_w[c];
        const bool live = m != -INFINITY;                    // an empty range's slot is unwritten memory
        const float wgt = live ? fast_exp2(m - ms) : 0.f;
        const float oc = live ? __ldcg(pq + c * cstride + ch) : 0.f, lc = live ? __ldcg(pq + c * cstride + kHeadDim + 1) : 0.f;
        num += wgt * oc;
        den += wgt * lc;
    }
    s_red[slice][ch] = num;
    if (ch == 0) s_red[slice][kHeadDim] = den;
    __syncthreads();
    // 3. across the slices
    if (slice == 0) {
        num = 0.f, den = 0.f;
#pragma unroll
        for (int i = 0; i < kRepMergeSlices; ++i) {
            num += s_red[i][ch];
            den += s_red[i][kHeadDim];
        }
        p.out[(int64_t)row * kHeadDim + ch] = num / den;
        if (p.lse && ch == 0) p.lse[row] = (ms + log2f(den)) * 0.6931471805599453f;
    }
    // herald_select_rep (merge_waits == 0): this grid runs BESIDE the top-k it was launched behind (the top-k releases its
    // dependents at once; the partials were complete before that).  It is the last kernel the entry enqueues, so whatever is
    // ordered behind it -- a programmatic launch, the next node of a captured graph -- must also be behind the top-k, which is
    // still reading the score plane / histogram and writing sel_idx / sel_cnt: wait for it here, after the outputs are written.
    if (!p.merge_waits) asm volatile("griddepcontrol.wait;" ::: "memory");
}

}  // namespace herald
