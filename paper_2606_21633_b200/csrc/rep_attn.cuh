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
//   grid = (chunks of kRepChunkTokens tokens, units); 8 warps stride over the pages of their chunk with an online
//   softmax per warp; warps merge in shared memory; one partial (m, l, o) per (unit, chunk) goes to the workspace and
//   rep_attn_merge_kernel combines the chunks of a unit.
//   Each warp keeps its NEXT page in flight while it works on the current one: the K fragments of page i+1 are loaded
//   into the fragment registers as soon as the score MMAs of page i have consumed them, and the V rows of page i+1 go
//   by cp.async into the other half of a per-warp double buffer (2 x 4 KB).  Without that each page costs a warp one
//   exposed DRAM round trip and the kernel is latency-bound.
#pragma once
#include "common.cuh"

namespace herald {

constexpr int kRepThreads = 256;
constexpr int kRepWarps = kRepThreads / 32;
constexpr int kRepChunkTokens = 2048;                 // tokens per CTA (128 pages)
constexpr int kRepPartFloats = 8 * (kHeadDim + 2);    // per (unit, chunk): 8 head slots x (128 channels, m, l)
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
    float* part;          // [units][n_chunks][8][130]
    float* out;           // [batch][H_q][128]
    float* lse;           // optional [batch][H_q]
    int32_t n_q_heads, n_kv_heads, max_seq_len, max_pages, n_chunks;
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
__global__ void __launch_bounds__(kRepThreads, 2) rep_attn_kernel(const RepAttnParams p) {
    extern __shared__ __align__(128) unsigned char rep_smem[];
    float (*s_o)[8][kHeadDim + 4] = reinterpret_cast<float (*)[8][kHeadDim + 4]>(rep_smem);   // per-warp results for the merge (rows of 528 B), over the V stages
    const int chunk = blockIdx.x, unit = blockIdx.y;
    const int b = unit / p.n_kv_heads, h = unit % p.n_kv_heads;
    const int G = p.n_q_heads / p.n_kv_heads;
    const int L = min(p.seq_lens[b], p.max_seq_len);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 2, tig = lane & 3;
    const int t_begin = chunk * kRepChunkTokens, t_end = min(L, t_begin + kRepChunkTokens);
    float* part = p.part + ((int64_t)unit * p.n_chunks + chunk) * kRepPartFloats;
    if (t_begin >= t_end) {   // chunk past the sequence: an empty partial (m = -inf) for the merge
        for (int i = threadIdx.x; i < 8; i += kRepThreads) part[i * (kHeadDim + 2) + kHeadDim] = -INFINITY;
        return;
    }

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

    const int32_t* pt = p.page_table + (int64_t)b * p.max_pages;
    const int page_end = (t_end + kPageSize - 1) / kPageSize;
    const uint32_t v_stage = smem_u32(rep_smem + warp * 2 * kRepVStageBytes);
    // ldmatrix row address of this lane inside a stage, for channel tile 0: matrix j = lane/8 is (tokens 8(j/2).., 16-byte
    // column j%2), row lane%8; the column index is XORed with (token & 7) = lane%8
    const int lm_tok = (lane & 7) + 8 * (lane >> 4), lm_col = (lane >> 3) & 1;
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
    int page = t_begin / kPageSize + warp;
    int phys_next = 0;
    if (page < page_end) {
        issue_page(page, __ldg(pt + page), 0);
        if (page + kRepWarps < page_end) phys_next = __ldg(pt + page + kRepWarps);
    }
    cp_async_commit();
    for (int st = 0; page < page_end; page += kRepWarps, st ^= 1) {
        float sa[4] = {0.f, 0.f, 0.f, 0.f}, sb[4] = {0.f, 0.f, 0.f, 0.f};   // tokens 0..7 / 8..15 of the page
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            mma_bf16_16816(sa, qf[i].x, 0u, qf[i].y, 0u, a[i].x, a[i].y);
            mma_bf16_16816(sa, qf[i].z, 0u, qf[i].w, 0u, a[i].z, a[i].w);
            mma_bf16_16816(sb, qf[i].x, 0u, qf[i].y, 0u, c[i].x, c[i].y);
            mma_bf16_16816(sb, qf[i].z, 0u, qf[i].w, 0u, c[i].z, c[i].w);
        }
        // the fragments are consumed: put the next page of this warp in flight
        if (page + kRepWarps < page_end) {
            issue_page(page + kRepWarps, phys_next, st ^ 1);
            if (page + 2 * kRepWarps < page_end) phys_next = __ldg(pt + page + 2 * kRepWarps);
        }
        cp_async_commit();
        // sa[0], sa[1]: head g, tokens 2tig, 2tig+1 ; sb[0], sb[1]: tokens 8+2tig, 9+2tig.  Mask the tail of the last page.
        const int t0 = page * kPageSize + 2 * tig;
        const bool ok0 = t0 < t_end, ok1 = t0 + 1 < t_end, ok2 = t0 + 8 < t_end, ok3 = t0 + 9 < t_end;
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

    // ---- merge the warps of the CTA, write the chunk's partial ----
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
    for (int idx = threadIdx.x; idx < 8 * kHeadDim; idx += kRepThreads) {
        const int q = idx >> 7, ch = idx & (kHeadDim - 1);
        float ms = -INFINITY;
#pragma unroll
        for (int wv = 0; wv < kRepWarps; ++wv) ms = fmaxf(ms, s_o[wv][q][kHeadDim]);
        float num = 0.f, den = 0.f;
#pragma unroll
        for (int wv = 0; wv < kRepWarps; ++wv) {
            const float mw = s_o[wv][q][kHeadDim];
            const float wgt = (mw == -INFINITY) ? 0.f : fast_exp2(mw - ms);
            num += wgt * s_o[wv][q][ch];
            den += wgt * s_o[wv][q][kHeadDim + 1];
        }
        part[q * (kHeadDim + 2) + ch] = num;
        if (ch == 0) {
            part[q * (kHeadDim + 2) + kHeadDim] = ms;
            part[q * (kHeadDim + 2) + kHeadDim + 1] = den;
        }
    }
}

// out[b, hq, :] = sum_c 2^(m_c - m*) o_c / sum_c 2^(m_c - m*) l_c over the chunks of the unit; one block per unit,
// blockDim = (128 channels, G heads).  The chunk loops carry no dependent loads (the kernel is a latency chain otherwise).
__global__ void __launch_bounds__(kHeadDim * 8) rep_attn_merge_kernel(const RepAttnParams p) {
    const int unit = blockIdx.x, ch = threadIdx.x, q = threadIdx.y;
    const int b = unit / p.n_kv_heads, h = unit % p.n_kv_heads;
    const int G = p.n_q_heads / p.n_kv_heads;
    const float* part = p.part + (int64_t)unit * p.n_chunks * kRepPartFloats + q * (kHeadDim + 2);
    float ms = -INFINITY;
#pragma unroll 8
    for (int c = 0; c < p.n_chunks; ++c) ms = fmaxf(ms, __ldg(part + c * kRepPartFloats + kHeadDim));
    float num = 0.f, den = 0.f;
    if (ms != -INFINITY) {
#pragma unroll 8
        for (int c = 0; c < p.n_chunks; ++c) {
            const float* pc = part + c * kRepPartFloats;
            const float mc = __ldg(pc + kHeadDim);
            const bool live = mc != -INFINITY;              // an empty chunk wrote only its m
            const float wgt = live ? fast_exp2(mc - ms) : 0.f;
            const float oc = live ? __ldg(pc + ch) : 0.f, lc = live ? __ldg(pc + kHeadDim + 1) : 0.f;
            num += wgt * oc;
            den += wgt * lc;
        }
    }
    const int64_t row = (int64_t)b * p.n_q_heads + h * G + q;
    p.out[row * kHeadDim + ch] = den > 0.f ? num / den : 0.f;                           // no cached token: zeros
    if (p.lse && ch == 0) p.lse[row] = den > 0.f ? (ms + log2f(den)) * 0.6931471805599453f : -INFINITY;
}

}  // namespace herald
