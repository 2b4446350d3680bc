// Attention output of the representative query itself (NEXT-2 of DESIGN.md; section IV-B4: the fused
// selection kernel "maintains the FlashAttention statistics (m_g, l_g, o_g)" next to the raw scores, and PAPER.md:193:
// that output goes back to the layer's FFN).
//
//   o[b, hq, :] = softmax_t( sm_scale * q_rep[b, hq] . K[b, t, h] ) . V[b, t, h, :]   over every cached t < seq_lens[b]
//
// One query row per head: there is no dense contraction to give to tcgen05 (M = G <= 8), and the kernel is a second
// HBM stream, now over K AND V (512 B per token and KV head).  Scores come from the same mma.sync trick as the score
// scan (16 tokens x 16 channels x 8 heads per MMA, fed from 128-bit global loads); the P.V product is G x 128 FMAs per
// token on the CUDA cores with each lane owning 4 channels, p broadcast from shared memory.
//   grid = (chunks of kRepChunkTokens tokens, units); 8 warps stride over the pages of their chunk with an online
//   softmax per warp; warps merge in shared memory; one partial (m, l, o) per (unit, chunk) goes to the workspace and
//   rep_attn_merge_kernel combines the chunks of a unit.
#pragma once
#include "common.cuh"

namespace herald {

constexpr int kRepThreads = 256;
constexpr int kRepWarps = kRepThreads / 32;
constexpr int kRepChunkTokens = 2048;                 // tokens per CTA (128 pages)
constexpr int kRepPartFloats = 8 * (kHeadDim + 2);    // per (unit, chunk): 8 head slots x (128 channels, m, l)

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

__global__ void __launch_bounds__(kRepThreads, 2) rep_attn_kernel(const RepAttnParams p) {
    __shared__ __align__(16) float s_p[kRepWarps][16][8];       // this page's weights of each warp: [token][head]
    __shared__ __align__(16) float s_o[kRepWarps][8][kHeadDim + 4];   // per-warp results for the merge (rows of 528 B: float4 stores)
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

    uint4 qf[4];              // B operand of the score MMA: query head g (zeros for g >= G), channel-permuted like A
    {
        const __nv_bfloat16* qrow = p.q_rep + ((int64_t)b * p.n_q_heads + h * G + g) * kHeadDim + 8 * tig;
#pragma unroll
        for (int i = 0; i < 4; ++i) qf[i] = (g < G) ? ldg_u4(qrow + 32 * i) : make_uint4(0, 0, 0, 0);
    }
    float m_run[8], l_run[8], o[8][4];     // online softmax of this warp, per head; lane owns channels [4*lane, 4*lane+4)
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        m_run[q] = -INFINITY;
        l_run[q] = 0.f;
#pragma unroll
        for (int c = 0; c < 4; ++c) o[q][c] = 0.f;
    }

    const int32_t* pt = p.page_table + (int64_t)b * p.max_pages;
    const int page_end = (t_end + kPageSize - 1) / kPageSize;
    for (int page = t_begin / kPageSize + warp; page < page_end; page += kRepWarps) {
        const int phys = __ldg(pt + page);
        const int64_t tile = (int64_t)phys * p.page_stride + (int64_t)h * p.head_stride;
        // K fragments (as in the score scan) and the V rows of the page: lane reads 8 bytes (4 channels) of each of the 16 rows
        const __nv_bfloat16* r0 = p.k_pages + tile + (int64_t)g * p.token_stride + 8 * tig;
        const __nv_bfloat16* r1 = p.k_pages + tile + (int64_t)(g + 8) * p.token_stride + 8 * tig;
        uint4 a[4], c[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            a[i] = ldg_stream_u4(r0 + 32 * i);
            c[i] = ldg_stream_u4(r1 + 32 * i);
        }
        uint2 v[16];
#pragma unroll
        for (int t = 0; t < 16; ++t)
            v[t] = __ldg(reinterpret_cast<const uint2*>(p.v_pages + tile + (int64_t)t * p.token_stride + 4 * lane));
        float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            mma_bf16_16816(acc, a[i].x, c[i].x, a[i].y, c[i].y, qf[i].x, qf[i].y);
            mma_bf16_16816(acc, a[i].z, c[i].z, a[i].w, c[i].w, qf[i].z, qf[i].w);
        }
#pragma unroll
        for (int t = 0; t < 16; ++t)
            if (page * kPageSize + t >= t_end) v[t] = make_uint2(0u, 0u);   // tail slots of the last page: weight 0, but 0 x NaN
        // acc[0],acc[1]: token row g, heads 2*tig, 2*tig+1 ; acc[2],acc[3]: token row g+8.  Mask the tail of the last page.
        const int t0 = page * kPageSize;
        const bool ok0 = t0 + g < t_end, ok1 = t0 + g + 8 < t_end;
        float s0 = ok0 ? acc[0] * p.scale_log2 : -INFINITY, s1 = ok0 ? acc[1] * p.scale_log2 : -INFINITY;
        float s2 = ok1 ? acc[2] * p.scale_log2 : -INFINITY, s3 = ok1 ? acc[3] * p.scale_log2 : -INFINITY;
        // page maximum per head: over this lane's two rows, then over the 8 row groups (lanes with equal tig)
        float mx0 = fmaxf(s0, s2), mx1 = fmaxf(s1, s3);
#pragma unroll
        for (int off = 4; off < 32; off <<= 1) {
            mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, off));
            mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, off));
        }
        // every lane needs the maxima of all 8 head slots: lane tig' holds heads 2tig', 2tig'+1
        float m_new[8], alpha[8];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const float e0 = __shfl_sync(0xffffffffu, mx0, q), e1 = __shfl_sync(0xffffffffu, mx1, q);
            m_new[2 * q] = fmaxf(m_run[2 * q], e0);
            m_new[2 * q + 1] = fmaxf(m_run[2 * q + 1], e1);
        }
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            alpha[q] = (m_run[q] == -INFINITY) ? 0.f : fast_exp2(m_run[q] - m_new[q]);
            m_run[q] = m_new[q];
        }
        // weights of this lane's four (token, head) pairs -> shared memory (the page has a valid token, so m_new of a
        // real head is finite; head slots >= G carry zeros throughout)
        const float mh0 = m_new[2 * tig], mh1 = m_new[2 * tig + 1];
        __syncwarp();
        s_p[warp][g][2 * tig] = (2 * tig < G && ok0) ? fast_exp2(s0 - mh0) : 0.f;
        s_p[warp][g][2 * tig + 1] = (2 * tig + 1 < G && ok0) ? fast_exp2(s1 - mh1) : 0.f;
        s_p[warp][g + 8][2 * tig] = (2 * tig < G && ok1) ? fast_exp2(s2 - mh0) : 0.f;
        s_p[warp][g + 8][2 * tig + 1] = (2 * tig + 1 < G && ok1) ? fast_exp2(s3 - mh1) : 0.f;
        __syncwarp();
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            l_run[q] *= alpha[q];
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) o[q][cc] *= alpha[q];
        }
#pragma unroll
        for (int t = 0; t < 16; ++t) {
            const float4 pa = *reinterpret_cast<const float4*>(&s_p[warp][t][0]);
            const float4 pb = *reinterpret_cast<const float4*>(&s_p[warp][t][4]);
            const float pw[8] = {pa.x, pa.y, pa.z, pa.w, pb.x, pb.y, pb.z, pb.w};
            const float vf[4] = {__uint_as_float(v[t].x << 16), __uint_as_float(v[t].x & 0xffff0000u),
                                 __uint_as_float(v[t].y << 16), __uint_as_float(v[t].y & 0xffff0000u)};
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                l_run[q] += pw[q];
#pragma unroll
                for (int cc = 0; cc < 4; ++cc) o[q][cc] = fmaf(pw[q], vf[cc], o[q][cc]);
            }
        }
    }

    // ---- merge the warps of the CTA, write the chunk's partial ----
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        *reinterpret_cast<float4*>(&s_o[warp][q][4 * lane]) = make_float4(o[q][0], o[q][1], o[q][2], o[q][3]);
        if (lane == 0) {
            s_o[warp][q][kHeadDim] = m_run[q];
            s_o[warp][q][kHeadDim + 1] = l_run[q];
        }
    }
    __syncthreads();
    for (int idx = threadIdx.x; idx < 8 * kHeadDim; idx += kRepThreads) {
        const int q = idx >> 7, ch = idx & (kHeadDim - 1);
        float ms = -INFINITY;
        for (int wv = 0; wv < kRepWarps; ++wv) ms = fmaxf(ms, s_o[wv][q][kHeadDim]);
        float num = 0.f, den = 0.f;
        for (int wv = 0; wv < kRepWarps; ++wv) {
            const float mw = s_o[wv][q][kHeadDim];
            if (mw == -INFINITY) continue;
            const float wgt = fast_exp2(mw - ms);
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

// out[b, hq, :] = sum_c 2^(m_c - m*) o_c / sum_c 2^(m_c - m*) l_c over the chunks of the unit; one block per unit.
__global__ void __launch_bounds__(kHeadDim) rep_attn_merge_kernel(const RepAttnParams p) {
    const int unit = blockIdx.x, ch = threadIdx.x;
    const int b = unit / p.n_kv_heads, h = unit % p.n_kv_heads;
    const int G = p.n_q_heads / p.n_kv_heads;
    const float* part = p.part + (int64_t)unit * p.n_chunks * kRepPartFloats;
    for (int q = 0; q < G; ++q) {
        float ms = -INFINITY;
        for (int c = 0; c < p.n_chunks; ++c) ms = fmaxf(ms, part[c * kRepPartFloats + q * (kHeadDim + 2) + kHeadDim]);
        float num = 0.f, den = 0.f;
        for (int c = 0; c < p.n_chunks; ++c) {
            const float* pc = part + c * kRepPartFloats + q * (kHeadDim + 2);
            if (pc[kHeadDim] == -INFINITY) continue;
            const float wgt = fast_exp2(pc[kHeadDim] - ms);
            num += wgt * pc[ch];
            den += wgt * pc[kHeadDim + 1];
        }
        const int64_t row = (int64_t)b * p.n_q_heads + h * G + q;
        p.out[row * kHeadDim + ch] = den > 0.f ? num / den : 0.f;                       // no cached token: zeros
        if (p.lse && ch == 0) p.lse[row] = den > 0.f ? (ms + log2f(den)) * 0.6931471805599453f : -INFINITY;
    }
}

}  // namespace herald
