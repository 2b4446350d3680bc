// Denoising-step attention over critical KV + in-block KV (step a5 of DESIGN.md).
// v0: flash-style kernel on legacy mma.sync tensor-core tiles (bf16 x bf16 -> fp32) with split-KV and
// an LSE combine.  It is the correctness baseline that the tcgen05/TMEM kernel replaces.
//
// One unit = (sequence b, KV head h).  Its M = B*G query rows (row m = block row m/G, group head m%G)
// attend over N = pool_len[b][h] pool rows followed by the B in-block rows; no mask.
// grid = (M tiles of 64 rows, KV splits, units); 4 warps x 16 rows; K/V tiles of 64 keys are staged in
// shared memory with cp.async (double buffered, 16-byte chunks XOR-swizzled by row) and read with ldmatrix.
#pragma once
#include "common.cuh"

namespace herald {

constexpr int kAttnBM = 64, kAttnBN = 64, kAttnThreads = 128;
constexpr int kAttnSmemBytes = 2 * 2 * kAttnBN * kRowBytes;   // 2 stages x (K + V)

struct AttnParams {
    const __nv_bfloat16* pool_k;
    const __nv_bfloat16* pool_v;
    const int32_t* pool_len;
    const __nv_bfloat16* q_blk;
    const __nv_bfloat16* k_blk;
    const __nv_bfloat16* v_blk;
    float* out;
    float* lse;
    float* part_o;      // [units][n_splits][m_pad][128] unnormalised partial outputs
    float2* part_ml;    // [units][n_splits][m_pad]      (running max in log2 units, partial sum)
    int32_t n_q_heads, n_kv_heads, block_size, cap, n_splits, m_pad;
    float scale_log2;   // sm_scale * log2(e)
};

__device__ __forceinline__ void cp_async_16(uint32_t dst, const void* src, int src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N)); }

__device__ __forceinline__ void ldmatrix_x4(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void ldmatrix_x4_trans(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}

// (x, y) -> packed bf16 pair hi = bf16(x), bf16(y) and the packed residual lo = bf16(x - hi.x), bf16(y - hi.y)
__device__ __forceinline__ void split_bf16(float x, float y, uint32_t& hi, uint32_t& lo) {
    hi = pack_bf16(x, y);
    const float hx = __uint_as_float(hi << 16), hy = __uint_as_float(hi & 0xffff0000u);
    lo = pack_bf16(x - hx, y - hy);
}

__global__ void __launch_bounds__(kAttnThreads) attn_mma_kernel(const AttnParams p) {
    extern __shared__ __align__(128) uint8_t smem[];
    const int unit = blockIdx.z, split = blockIdx.y, mtile = blockIdx.x;
    const int b = unit / p.n_kv_heads, h = unit % p.n_kv_heads;
    const int G = p.n_q_heads / p.n_kv_heads, B = p.block_size, M = B * G;
    const int n_pool = max(0, min(p.pool_len[unit], p.cap));
    const int N = n_pool + B;
    const int n_tiles = (N + kAttnBN - 1) / kAttnBN;
    const int per = (n_tiles + p.n_splits - 1) / p.n_splits;
    const int t0 = split * per, t1 = min(n_tiles, t0 + per);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, t = lane & 3;
    const int rowA = mtile * kAttnBM + warp * 16 + g, rowB = rowA + 8;
    const int64_t part_base = ((int64_t)unit * p.n_splits + split) * p.m_pad;

    if (t0 >= t1) {   // empty split: tell the combine kernel to skip it
        if (t == 0) {
            if (rowA < p.m_pad) p.part_ml[part_base + rowA] = make_float2(-INFINITY, 0.f);
            if (rowB < p.m_pad) p.part_ml[part_base + rowB] = make_float2(-INFINITY, 0.f);
        }
        return;
    }

    // Q fragments (A operand), 8 k-steps of 16 channels
    uint32_t qa[8][4];
    {
        const __nv_bfloat16* qA = p.q_blk + (((int64_t)b * B + (rowA < M ? rowA / G : 0)) * p.n_q_heads + h * G + (rowA < M ? rowA % G : 0)) * kHeadDim;
        const __nv_bfloat16* qB = p.q_blk + (((int64_t)b * B + (rowB < M ? rowB / G : 0)) * p.n_q_heads + h * G + (rowB < M ? rowB % G : 0)) * kHeadDim;
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
            qa[ks][0] = rowA < M ? *reinterpret_cast<const uint32_t*>(qA + 16 * ks + 2 * t) : 0u;
            qa[ks][1] = rowB < M ? *reinterpret_cast<const uint32_t*>(qB + 16 * ks + 2 * t) : 0u;
            qa[ks][2] = rowA < M ? *reinterpret_cast<const uint32_t*>(qA + 16 * ks + 8 + 2 * t) : 0u;
            qa[ks][3] = rowB < M ? *reinterpret_cast<const uint32_t*>(qB + 16 * ks + 8 + 2 * t) : 0u;
        }
    }

    const uint32_t smem_base = smem_u32(smem);
    auto load_tile = [&](int tile, int stage) {
        const uint32_t ks = smem_base + stage * (2 * kAttnBN * kRowBytes);
        const uint32_t vs = ks + kAttnBN * kRowBytes;
        for (int c = tid; c < kAttnBN * 16; c += kAttnThreads) {
            const int r = c >> 4, ch = c & 15;
            const int kj = tile * kAttnBN + r;
            const bool valid = kj < N;
            int64_t off;
            const __nv_bfloat16 *ksrc, *vsrc;
            if (kj < n_pool) {
                off = ((int64_t)unit * p.cap + kj) * kHeadDim + ch * 8;
                ksrc = p.pool_k + off;
                vsrc = p.pool_v + off;
            } else {
                const int j = min(kj - n_pool, B - 1);
                off = (((int64_t)b * B + j) * p.n_kv_heads + h) * kHeadDim + ch * 8;
                ksrc = p.k_blk + off;
                vsrc = p.v_blk + off;
            }
            const uint32_t dst = r * kRowBytes + ((ch ^ (r & 7)) << 4);
            cp_async_16(ks + dst, ksrc, valid ? 16 : 0);
            cp_async_16(vs + dst, vsrc, valid ? 16 : 0);
        }
        cp_async_commit();
    };

    float o[16][4];
#pragma unroll
    for (int i = 0; i < 16; ++i) o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f;
    float mA = -INFINITY, mB = -INFINITY, lA = 0.f, lB = 0.f;

    load_tile(t0, 0);
    for (int tile = t0; tile < t1; ++tile) {
        const int stage = (tile - t0) & 1;
        if (tile + 1 < t1) {
            load_tile(tile + 1, stage ^ 1);
            cp_async_wait<1>();
        } else {
            cp_async_wait<0>();
        }
        __syncthreads();
        const uint32_t ks_base = smem_base + stage * (2 * kAttnBN * kRowBytes);
        const uint32_t vs_base = ks_base + kAttnBN * kRowBytes;

        float s[8][4];
#pragma unroll
        for (int nt = 0; nt < 8; ++nt) {
            s[nt][0] = s[nt][1] = s[nt][2] = s[nt][3] = 0.f;
            const int row = nt * 8 + (lane & 7);
#pragma unroll
            for (int kp = 0; kp < 4; ++kp) {
                const int chunk = 4 * kp + (lane >> 3);
                uint32_t r0, r1, r2, r3;
                ldmatrix_x4(ks_base + row * kRowBytes + ((chunk ^ (row & 7)) << 4), r0, r1, r2, r3);
                mma_bf16_16816(s[nt], qa[2 * kp][0], qa[2 * kp][1], qa[2 * kp][2], qa[2 * kp][3], r0, r1);
                mma_bf16_16816(s[nt], qa[2 * kp + 1][0], qa[2 * kp + 1][1], qa[2 * kp + 1][2], qa[2 * kp + 1][3], r2, r3);
            }
        }
        if (tile == n_tiles - 1) {
#pragma unroll
            for (int nt = 0; nt < 8; ++nt)
#pragma unroll
                for (int e = 0; e < 4; ++e)
                    if (tile * kAttnBN + nt * 8 + 2 * t + (e & 1) >= N) s[nt][e] = -INFINITY;
        }
        float mxA = -INFINITY, mxB = -INFINITY;
#pragma unroll
        for (int nt = 0; nt < 8; ++nt) {
            mxA = fmaxf(mxA, fmaxf(s[nt][0], s[nt][1]));
            mxB = fmaxf(mxB, fmaxf(s[nt][2], s[nt][3]));
        }
        mxA = fmaxf(mxA, __shfl_xor_sync(0xffffffffu, mxA, 1));
        mxB = fmaxf(mxB, __shfl_xor_sync(0xffffffffu, mxB, 1));
        mxA = fmaxf(mxA, __shfl_xor_sync(0xffffffffu, mxA, 2));
        mxB = fmaxf(mxB, __shfl_xor_sync(0xffffffffu, mxB, 2));
        const float mA_new = fmaxf(mA, mxA * p.scale_log2), mB_new = fmaxf(mB, mxB * p.scale_log2);
        const float alphaA = fast_exp2(mA - mA_new), alphaB = fast_exp2(mB - mB_new);
        mA = mA_new;
        mB = mB_new;
        float sumA = 0.f, sumB = 0.f;
#pragma unroll
        for (int nt = 0; nt < 8; ++nt) {
            s[nt][0] = fast_exp2(fmaf(s[nt][0], p.scale_log2, -mA));
            s[nt][1] = fast_exp2(fmaf(s[nt][1], p.scale_log2, -mA));
            s[nt][2] = fast_exp2(fmaf(s[nt][2], p.scale_log2, -mB));
            s[nt][3] = fast_exp2(fmaf(s[nt][3], p.scale_log2, -mB));
            sumA += s[nt][0] + s[nt][1];
            sumB += s[nt][2] + s[nt][3];
        }
        lA = lA * alphaA + sumA;
        lB = lB * alphaB + sumB;
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            o[i][0] *= alphaA;
            o[i][1] *= alphaA;
            o[i][2] *= alphaB;
            o[i][3] *= alphaB;
        }
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
            // P = P_hi + P_lo (two bf16 terms): keeps the softmax weights to ~2^-17 relative so that peaked
            // rows stay inside the 2e-3 output tolerance
            uint32_t a0, a1, a2, a3, l0, l1, l2, l3;
            split_bf16(s[2 * kk][0], s[2 * kk][1], a0, l0);
            split_bf16(s[2 * kk][2], s[2 * kk][3], a1, l1);
            split_bf16(s[2 * kk + 1][0], s[2 * kk + 1][1], a2, l2);
            split_bf16(s[2 * kk + 1][2], s[2 * kk + 1][3], a3, l3);
            const int mi = lane >> 3;
            const int row = 16 * kk + (mi & 1) * 8 + (lane & 7);
#pragma unroll
            for (int dp = 0; dp < 8; ++dp) {
                const int chunk = 2 * dp + (mi >> 1);
                uint32_t r0, r1, r2, r3;
                ldmatrix_x4_trans(vs_base + row * kRowBytes + ((chunk ^ (row & 7)) << 4), r0, r1, r2, r3);
                mma_bf16_16816(o[2 * dp], a0, a1, a2, a3, r0, r1);
                mma_bf16_16816(o[2 * dp + 1], a0, a1, a2, a3, r2, r3);
                mma_bf16_16816(o[2 * dp], l0, l1, l2, l3, r0, r1);
                mma_bf16_16816(o[2 * dp + 1], l0, l1, l2, l3, r2, r3);
            }
        }
        __syncthreads();
    }

    lA += __shfl_xor_sync(0xffffffffu, lA, 1);
    lB += __shfl_xor_sync(0xffffffffu, lB, 1);
    lA += __shfl_xor_sync(0xffffffffu, lA, 2);
    lB += __shfl_xor_sync(0xffffffffu, lB, 2);

    if (p.n_splits == 1) {
        const float invA = 1.f / lA, invB = 1.f / lB;
        if (rowA < M) {
            float* dst = p.out + (((int64_t)b * B + rowA / G) * p.n_q_heads + h * G + rowA % G) * kHeadDim;
#pragma unroll
            for (int i = 0; i < 16; ++i)
                *reinterpret_cast<float2*>(dst + 8 * i + 2 * t) = make_float2(o[i][0] * invA, o[i][1] * invA);
            if (p.lse && t == 0)
                p.lse[((int64_t)b * B + rowA / G) * p.n_q_heads + h * G + rowA % G] = (mA + log2f(lA)) * 0.6931471805599453f;
        }
        if (rowB < M) {
            float* dst = p.out + (((int64_t)b * B + rowB / G) * p.n_q_heads + h * G + rowB % G) * kHeadDim;
#pragma unroll
            for (int i = 0; i < 16; ++i)
                *reinterpret_cast<float2*>(dst + 8 * i + 2 * t) = make_float2(o[i][2] * invB, o[i][3] * invB);
            if (p.lse && t == 0)
                p.lse[((int64_t)b * B + rowB / G) * p.n_q_heads + h * G + rowB % G] = (mB + log2f(lB)) * 0.6931471805599453f;
        }
    } else {
        if (rowA < p.m_pad) {
            float* dst = p.part_o + (part_base + rowA) * kHeadDim;
#pragma unroll
            for (int i = 0; i < 16; ++i) *reinterpret_cast<float2*>(dst + 8 * i + 2 * t) = make_float2(o[i][0], o[i][1]);
            if (t == 0) p.part_ml[part_base + rowA] = make_float2(mA, lA);
        }
        if (rowB < p.m_pad) {
            float* dst = p.part_o + (part_base + rowB) * kHeadDim;
#pragma unroll
            for (int i = 0; i < 16; ++i) *reinterpret_cast<float2*>(dst + 8 * i + 2 * t) = make_float2(o[i][2], o[i][3]);
            if (t == 0) p.part_ml[part_base + rowB] = make_float2(mB, lB);
        }
    }
}

// Merge of the split-KV partials: out = sum_s 2^(m_s - m*) O_s / sum_s 2^(m_s - m*) l_s.
__global__ void __launch_bounds__(128) attn_combine_kernel(const AttnParams p) {
    const int unit = blockIdx.y, row = blockIdx.x;
    const int b = unit / p.n_kv_heads, h = unit % p.n_kv_heads;
    const int G = p.n_q_heads / p.n_kv_heads, B = p.block_size;
    const int d = threadIdx.x;
    float mstar = -INFINITY;
    for (int s = 0; s < p.n_splits; ++s)
        mstar = fmaxf(mstar, p.part_ml[((int64_t)unit * p.n_splits + s) * p.m_pad + row].x);
    float num = 0.f, den = 0.f;
    for (int s = 0; s < p.n_splits; ++s) {
        const int64_t base = ((int64_t)unit * p.n_splits + s) * p.m_pad + row;
        const float2 ml = p.part_ml[base];
        if (ml.x == -INFINITY) continue;
        const float w = fast_exp2(ml.x - mstar);
        den += w * ml.y;
        num += w * p.part_o[base * kHeadDim + d];
    }
    const int64_t orow = ((int64_t)b * B + row / G) * p.n_q_heads + h * G + row % G;
    p.out[orow * kHeadDim + d] = num / den;
    if (p.lse && d == 0) p.lse[orow] = (mstar + log2f(den)) * 0.6931471805599453f;
}

}  // namespace herald
