// Denoising-step attention over critical KV + in-block KV on the 5th-generation tensor cores
// (step a5 of DESIGN.md; "bidirectionally within the current block and causally to the
// cached KV", "denoises block n using the KV cache in the active sparse pool").
//
// One unit = (sequence b, KV head h).  Its M = B*G query rows (row m = block row m/G, group head m%G)
// attend over N = pool_len[b][h] pool rows followed by the B in-block rows; no mask.  The two products
// are real dense contractions (QK^T: [128 x d] x [d x 128], PV: [128 x 128] x [128 x d]) and run as
// tcgen05.mma (UMMA M=128, bf16 x bf16 -> fp32; P enters the PV product as a bf16 hi+lo pair) with the
// accumulators in TMEM:
//
//   grid  = (KV splits, M tiles of 128 rows, units), 352 threads, 1 CTA / SM
//   warps 8, 9  producers, one for K and one for V: whole 128-key pool tiles arrive by TMA (cp.async.bulk.tensor,
//               128B swizzle) into 3-stage rings; a K stage is released as soon as QK^T has read it, a V stage
//               after PV.  The ragged tail of the pool and the in-block rows are written with zero-filling
//               cp.async, so rows past the end are exact zeros.
//   warp 10     issues the MMAs (one lane): S[j&1] = Q K_j^T (operands in shared memory) into a double-buffered
//               TMEM tile, then O += P_{j-1} V_{j-1} with P read from TMEM; tcgen05.commit -> mbarrier
//   warps 0..7  softmax: thread (row, column half) reads 64 logits of its row from TMEM (tcgen05.ld),
//               exchanges the row maximum with its partner warp, exponentiates (ex2), accumulates the row sum,
//               splits P into a bf16 hi+lo pair and writes both back over S_j in TMEM (tcgen05.st).
//               The running maximum is only raised when it grows by more than 2^8 ("lazy rescale"):
//               O in TMEM is then rescaled in place, which is rare.
//   split-KV partials (unnormalised O, running max, row sum) go to the workspace and are merged by
//   attn_combine_kernel; with one split the epilogue normalises and writes `out` directly.
#pragma once
#include <cuda.h>

#include "common.cuh"

namespace herald {

constexpr int kTcBM = 128;                       // query rows per CTA (UMMA M)
constexpr int kTcBN = 128;                       // keys per tile (UMMA N of QK^T, K of PV)
constexpr int kTcStages = 3;                     // depth of the K ring and of the V ring
constexpr int kTcThreads = 352;                  // 8 softmax warps + K producer + V producer + MMA issuer
constexpr int kTcKWarp = 8, kTcVWarp = 9, kTcMmaWarp = 10;
constexpr int kTcHalfBytes = kTcBN * 128;        // one [128 rows x 64 el] swizzled half tile (16 KB)
constexpr int kTcTileBytes = 2 * kTcHalfBytes;   // a [128 x 128] bf16 tile = two halves (32 KB)
constexpr int kTcSmemQ = 0;
constexpr int kTcSmemK = kTcSmemQ + kTcTileBytes;                        // K ring
constexpr int kTcSmemV = kTcSmemK + kTcStages * kTcTileBytes;            // V ring
constexpr int kTcSmemMisc = kTcSmemV + kTcStages * kTcTileBytes;         // barriers, TMEM pointer, exchange buffers
constexpr int kTcMiscBytes = 2304;
constexpr int kTcSmemBytes = kTcSmemMisc + kTcMiscBytes;                 // 231,680 B of the 232,448 B a CTA may own
constexpr int kTcTmemCols = 512;                 // S0/P0 [0,128) S1/P1 [128,256) O [256,384)
constexpr float kTcRescaleThreshold = 8.f;       // log2 units

// barrier slots (8 bytes each) inside the misc area
enum { kBarKFull = 0, kBarKEmpty = kBarKFull + kTcStages, kBarVFull = kBarKEmpty + kTcStages, kBarVEmpty = kBarVFull + kTcStages,
       kBarSFull = kBarVEmpty + kTcStages, kBarPFull = kBarSFull + 2, kBarPvDone, kBarCount = kBarPvDone + 2 };
constexpr int kTcMiscTmemPtr = 192;              // uint32
constexpr int kTcMiscMax = 256;                  // float [2 buffers][2 halves][128 rows]
constexpr int kTcMiscSum = kTcMiscMax;           // float [2 halves][128 rows]; reuses the max buffer after the last tile
static_assert(kBarCount * 8 <= kTcMiscTmemPtr, "barriers overlap the TMEM pointer slot");

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

// ---- PTX wrappers -------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// Spins on try_wait; a wait that never completes (a protocol bug) traps instead of hanging the GPU.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    for (uint32_t spins = 0;; ++spins) {
        uint32_t done;
        asm volatile(
            "{\n\t"
            ".reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t"
            "}" : "=r"(done) : "r"(bar), "r"(parity) : "memory");
        if (done) return;
        if (spins > (1u << 26)) __trap();
    }
}
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void named_bar_sync(uint32_t id, uint32_t threads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}

__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
}

__device__ __forceinline__ void cp_async_16_zfill(uint32_t dst, const void* src, int src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// D[tmem] (+)= A[smem desc] * B[smem desc]
__device__ __forceinline__ void umma_ss(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t"
        "}" ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem desc]; A: row = TMEM lane, two 16-bit K elements per 32-bit column
__device__ __forceinline__ void umma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t"
        "}" ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}

// 32 lanes x 32 consecutive 32-bit columns: thread t of the warp gets columns [col, col+32) of TMEM lane (lane base + t)
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float (&v)[32]) {
    uint32_t r[32];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
          "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
          "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const float (&v)[32]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%32], "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31};"
        ::"r"(__float_as_uint(v[0])), "r"(__float_as_uint(v[1])), "r"(__float_as_uint(v[2])), "r"(__float_as_uint(v[3])),
          "r"(__float_as_uint(v[4])), "r"(__float_as_uint(v[5])), "r"(__float_as_uint(v[6])), "r"(__float_as_uint(v[7])),
          "r"(__float_as_uint(v[8])), "r"(__float_as_uint(v[9])), "r"(__float_as_uint(v[10])), "r"(__float_as_uint(v[11])),
          "r"(__float_as_uint(v[12])), "r"(__float_as_uint(v[13])), "r"(__float_as_uint(v[14])), "r"(__float_as_uint(v[15])),
          "r"(__float_as_uint(v[16])), "r"(__float_as_uint(v[17])), "r"(__float_as_uint(v[18])), "r"(__float_as_uint(v[19])),
          "r"(__float_as_uint(v[20])), "r"(__float_as_uint(v[21])), "r"(__float_as_uint(v[22])), "r"(__float_as_uint(v[23])),
          "r"(__float_as_uint(v[24])), "r"(__float_as_uint(v[25])), "r"(__float_as_uint(v[26])), "r"(__float_as_uint(v[27])),
          "r"(__float_as_uint(v[28])), "r"(__float_as_uint(v[29])), "r"(__float_as_uint(v[30])), "r"(__float_as_uint(v[31])),
          "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// (x, y) -> packed bf16 pair hi = (bf16(x), bf16(y)) and the packed residual lo = (bf16(x - hi.x), bf16(y - hi.y))
__device__ __forceinline__ void split_bf16(float x, float y, uint32_t& hi, uint32_t& lo) {
    hi = pack_bf16(x, y);
    const float hx = __uint_as_float(hi << 16), hy = __uint_as_float(hi & 0xffff0000u);
    lo = pack_bf16(x - hx, y - hy);
}

// Shared-memory matrix descriptor, 128-byte swizzle (layout type 2), descriptor version 1 (sm_100).
//   K-major operand : rows of 128 B (64 x 16-bit), 8-row groups `sbo` bytes apart, lbo unused (encoded 1)
//   MN-major operand: 64 contiguous MN elements per 128 B row, K rows 128 B apart, 8-row K groups `sbo`
//                     apart, next 64-element MN group `lbo` bytes away
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t smem_addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    return (uint64_t)((smem_addr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) | ((uint64_t)(sbo_bytes >> 4) << 32) |
           (1ull << 46) | (2ull << 61);
}
// Instruction descriptor of tcgen05.mma.kind::f16: fp32 accumulate, A/B formats (0 = f16, 1 = bf16),
// majors (0 = K, 1 = MN), N >> 3 at bit 17, M >> 4 at bit 24.
__device__ __forceinline__ constexpr uint32_t umma_idesc(int a_fmt, int b_fmt, int a_mn, int b_mn, int M, int N) {
    return (1u << 4) | ((uint32_t)a_fmt << 7) | ((uint32_t)b_fmt << 10) | ((uint32_t)a_mn << 15) | ((uint32_t)b_mn << 16) |
           ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

__global__ void __launch_bounds__(kTcThreads, 1)
attn_tc_kernel(const __grid_constant__ CUtensorMap tm_k, const __grid_constant__ CUtensorMap tm_v, const AttnParams p) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t sbase = smem_u32(smem_raw);
    uint8_t* sgen = smem_raw;
    if (sbase & 1023u) __trap();   // the 128B-swizzled tiles need a 1024 B aligned base

    const int split = blockIdx.x, mtile = blockIdx.y, unit = blockIdx.z;
    const int b = unit / p.n_kv_heads, h = unit % p.n_kv_heads;
    const int G = p.n_q_heads / p.n_kv_heads, B = p.block_size, M = B * G;
    const int n_pool = max(0, min(p.pool_len[unit], p.cap));
    const int N = n_pool + B;
    const int n_tiles = (N + kTcBN - 1) / kTcBN;
    const int n_full = n_pool / kTcBN;                       // tiles [0, n_full) are whole pool tiles -> TMA
    const int per = (n_tiles + p.n_splits - 1) / p.n_splits;
    const int t0 = split * per, t1 = min(n_tiles, t0 + per);
    const int nt = t1 - t0;                                  // tile j of this CTA is key tile t0 + j (ragged tiles last)
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int64_t part_base = ((int64_t)unit * p.n_splits + split) * p.m_pad + mtile * kTcBM;

    if (nt <= 0) {   // empty split: tell the combine kernel to skip it
        if (tid < kTcBM) p.part_ml[part_base + tid] = make_float2(-INFINITY, 0.f);
        return;
    }

    const uint32_t misc = sbase + kTcSmemMisc;
    auto bar = [&](int i) { return misc + 8u * i; };
    volatile uint32_t* tmem_ptr_gen = reinterpret_cast<volatile uint32_t*>(sgen + kTcSmemMisc + kTcMiscTmemPtr);
    float* ex_max = reinterpret_cast<float*>(sgen + kTcSmemMisc + kTcMiscMax);
    float* ex_sum = reinterpret_cast<float*>(sgen + kTcSmemMisc + kTcMiscSum);

    // ---- one-time setup ---------------------------------------------------------------------------
    if (warp == kTcMmaWarp) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(misc + kTcMiscTmemPtr), "n"(kTcTmemCols));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    if (warp == kTcKWarp && lane == 0) {
        for (int s = 0; s < kTcStages; ++s) {
            mbar_init(bar(kBarKFull + s), 1);
            mbar_init(bar(kBarKEmpty + s), 1);
            mbar_init(bar(kBarVFull + s), 1);
            mbar_init(bar(kBarVEmpty + s), 1);
        }
        for (int s = 0; s < 2; ++s) mbar_init(bar(kBarSFull + s), 1);
        mbar_init(bar(kBarPFull), 8);
        for (int s = 0; s < 2; ++s) mbar_init(bar(kBarPvDone + s), 1);   // PV_j commits to slot j&1 (see the epilogue wait)
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_k) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_v) : "memory");
    }
    // Q tile -> shared memory, UMMA K-major 128B-swizzled: rows past M are zero
    for (int c = tid; c < kTcBM * 16; c += kTcThreads) {
        const int r = c >> 4, ch = c & 15;
        const int m = mtile * kTcBM + r;
        uint4 v = make_uint4(0, 0, 0, 0);
        if (m < M) v = ldg_u4(p.q_blk + (((int64_t)b * B + m / G) * p.n_q_heads + h * G + m % G) * kHeadDim + ch * 8);
        *reinterpret_cast<uint4*>(sgen + kTcSmemQ + (ch >> 3) * kTcHalfBytes + r * 128 + (((ch & 7) ^ (r & 7)) << 4)) = v;
    }
    fence_proxy_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_ptr_gen;

    auto tile_cols = [&](int j) {   // key columns of this CTA's j-th tile that the MMAs touch (multiple of 16)
        const int valid = min(kTcBN, N - (t0 + j) * kTcBN);
        return (valid + 15) & ~15;
    };

    if (warp == kTcKWarp || warp == kTcVWarp) {
        // =========================== producers: one warp streams K tiles, one streams V tiles ===========================
        const bool is_k = warp == kTcKWarp;
        const CUtensorMap* map = is_k ? &tm_k : &tm_v;
        const __nv_bfloat16* pool = is_k ? p.pool_k : p.pool_v;
        const __nv_bfloat16* blk = is_k ? p.k_blk : p.v_blk;
        const int bar_full = is_k ? kBarKFull : kBarVFull, bar_empty = is_k ? kBarKEmpty : kBarVEmpty;
        const uint32_t ring = sbase + (is_k ? kTcSmemK : kTcSmemV);
        for (int j = 0; j < nt; ++j) {
            const int stage = j % kTcStages, t = t0 + j;
            if (j >= kTcStages) mbar_wait(bar(bar_empty + stage), ((j / kTcStages) - 1) & 1);
            const uint32_t dst = ring + stage * kTcTileBytes, full = bar(bar_full + stage);
            if (t < n_full) {
                if (lane == 0) {
                    mbar_arrive_expect_tx(full, kTcTileBytes);
                    tma_load_3d(dst, map, 0, t * kTcBN, unit, full);
                    tma_load_3d(dst + kTcHalfBytes, map, 64, t * kTcBN, unit, full);
                }
            } else {
                // ragged tile (pool tail and/or in-block rows): zero-filling 16-byte cp.async, rows past N are zeros
                const int rows = tile_cols(j);
                for (int c = lane; c < rows * 16; c += 32) {
                    const int r = c >> 4, ch = c & 15;
                    const int kj = t * kTcBN + r;
                    const __nv_bfloat16* src = pool;
                    int bytes = 0;
                    if (kj < n_pool) {
                        src = pool + ((int64_t)unit * p.cap + kj) * kHeadDim + ch * 8;
                        bytes = 16;
                    } else if (kj < N) {
                        src = blk + (((int64_t)b * B + (kj - n_pool)) * p.n_kv_heads + h) * kHeadDim + ch * 8;
                        bytes = 16;
                    }
                    cp_async_16_zfill(dst + (ch >> 3) * kTcHalfBytes + r * 128 + (((ch & 7) ^ (r & 7)) << 4), src, bytes);
                }
                cp_async_wait_all();
                fence_proxy_async_smem();
                __syncwarp();
                if (lane == 0) mbar_arrive(full);
            }
        }
    } else if (warp == kTcMmaWarp) {
        // =========================== MMA issuer ===========================
        constexpr uint32_t idesc_pv = umma_idesc(/*A bf16*/ 1, /*B bf16*/ 1, /*A K-major*/ 0, /*B MN-major*/ 1, kTcBM, kHeadDim);
        const uint32_t q_base = sbase + kTcSmemQ;
        auto issue_pv = [&](int j) {   // O (+)= (P_hi + P_lo)_j V_j, P read from TMEM (it overlays S_j)
            const int stage = j % kTcStages, sb = j & 1;
            mbar_wait(bar(kBarVFull + stage), (j / kTcStages) & 1);
            mbar_wait(bar(kBarPFull), j & 1);
            tc_fence_after();
            if (lane == 0) {
                const uint32_t v_base = sbase + kTcSmemV + stage * kTcTileBytes;
                const int ksteps = tile_cols(j) >> 4;
                for (int kk = 0; kk < ksteps; ++kk) {
                    const uint64_t bd = umma_desc_sw128(v_base + kk * 2048, kTcHalfBytes, 1024);
                    umma_ts(tmem + 256, tmem + sb * 128 + kk * 8, bd, idesc_pv, (j > 0 || kk > 0) ? 1u : 0u);
                    umma_ts(tmem + 256, tmem + sb * 128 + 64 + kk * 8, bd, idesc_pv, 1u);
                }
                umma_commit(bar(kBarPvDone + sb));
                umma_commit(bar(kBarVEmpty + stage));
            }
            __syncwarp();
        };
        for (int j = 0; j < nt; ++j) {
            const int stage = j % kTcStages, sb = j & 1;
            mbar_wait(bar(kBarKFull + stage), (j / kTcStages) & 1);
            tc_fence_after();
            if (lane == 0) {
                // S_j overwrites the TMEM columns of P_{j-2}: PV_{j-2} was issued earlier and the tensor pipe runs in order
                const uint32_t k_base = sbase + kTcSmemK + stage * kTcTileBytes;
                const uint32_t idesc_s = umma_idesc(1, 1, 0, 0, kTcBM, tile_cols(j));
#pragma unroll
                for (int ks = 0; ks < 8; ++ks) {
                    const uint32_t off = (ks >> 2) * kTcHalfBytes + (ks & 3) * 32;
                    umma_ss(tmem + sb * 128, umma_desc_sw128(q_base + off, 16, 1024), umma_desc_sw128(k_base + off, 16, 1024),
                            idesc_s, ks > 0 ? 1u : 0u);
                }
                umma_commit(bar(kBarSFull + sb));
                umma_commit(bar(kBarKEmpty + stage));
            }
            __syncwarp();
            if (j > 0) issue_pv(j - 1);
        }
        issue_pv(nt - 1);
    } else {
        // =========================== softmax warps ===========================
        const int quarter = warp & 3, hf = warp >> 2;
        const int row = quarter * 32 + lane;                 // row of the M tile == TMEM lane
        const uint32_t lane_base = tmem + ((uint32_t)(quarter * 32) << 16);
        float m_used = -INFINITY, l = 0.f;
        for (int j = 0; j < nt; ++j) {
            const int sb = j & 1;
            // S_j complete; the commit also covers PV_{j-2}, so the P columns overlaying this S buffer are free
            mbar_wait(bar(kBarSFull + sb), (j >> 1) & 1);
            tc_fence_after();
            float s[64];
            {
                float a[32], c[32];
                tmem_ld32(lane_base + sb * 128 + hf * 64, a);
                tmem_ld32(lane_base + sb * 128 + hf * 64 + 32, c);
#pragma unroll
                for (int i = 0; i < 32; ++i) { s[i] = a[i]; s[32 + i] = c[i]; }
            }
            const int valid = N - (t0 + j) * kTcBN;           // >= 1
            if (valid < kTcBN) {
#pragma unroll
                for (int i = 0; i < 64; ++i)
                    if (hf * 64 + i >= valid) s[i] = -INFINITY;
            }
            float mx = s[0];
#pragma unroll
            for (int i = 1; i < 64; ++i) mx = fmaxf(mx, s[i]);
            ex_max[(sb * 2 + hf) * 128 + row] = mx;
            named_bar_sync(1 + quarter, 64);                  // both column halves of these 32 rows have read S_j
            const float mrow = fmaxf(mx, ex_max[(sb * 2 + (hf ^ 1)) * 128 + row]) * p.scale_log2;
            float alpha = 1.f;
            bool need = false;
            if (j == 0) {
                m_used = mrow;
            } else if (mrow > m_used + kTcRescaleThreshold) {
                need = true;
                alpha = fast_exp2(m_used - mrow);
                m_used = mrow;
            }
            const bool any = __any_sync(0xffffffffu, need);
            float sum = 0.f;
#pragma unroll
            for (int i = 0; i < 64; ++i) {
                s[i] = fast_exp2(fmaf(s[i], p.scale_log2, -m_used));
                sum += s[i];
            }
            l = l * alpha + sum;
            if (any) {   // rare: the running maximum of some row grew by more than 2^8 -> rescale O in place
                mbar_wait(bar(kBarPvDone + ((j - 1) & 1)), ((j - 1) >> 1) & 1);   // PV_{j-1} finished; PV_j waits for our arrive
                tc_fence_after();
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    float o[32];
                    tmem_ld32(lane_base + 256 + hf * 64 + q * 32, o);
#pragma unroll
                    for (int i = 0; i < 32; ++i) o[i] *= alpha;
                    tmem_st32(lane_base + 256 + hf * 64 + q * 32, o);
                }
            }
            // P = P_hi + P_lo (bf16 pair, 16 significand bits: the PV product keeps the weights to ~2^-17 relative, so
            // peaked rows stay inside the 2e-3 output tolerance).  Both go to TMEM as the A operand of the PV MMA:
            // row = lane, two keys per 32-bit column; P_hi in columns [0,64) of the S buffer, P_lo in [64,128).
            {
                float hi[32], lo[32];
#pragma unroll
                for (int i = 0; i < 32; ++i) {
                    uint32_t h2, l2;
                    split_bf16(s[2 * i], s[2 * i + 1], h2, l2);
                    hi[i] = __uint_as_float(h2);
                    lo[i] = __uint_as_float(l2);
                }
                tmem_st32(lane_base + sb * 128 + hf * 32, hi);
                tmem_st32(lane_base + sb * 128 + 64 + hf * 32, lo);
            }
            tmem_wait_st();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(kBarPFull));
        }
        // ---- epilogue: O / l -> out (one split) or partials (split-KV) ----
        // A parity wait is only sound when the waiter is at most one phase behind.  The softmax warps do not wait for
        // every PV, but S_j's commit covers PV_{j-2}, so with one barrier per tile parity the lag is at most one phase.
        mbar_wait(bar(kBarPvDone + ((nt - 1) & 1)), ((nt - 1) >> 1) & 1);
        tc_fence_after();
        ex_sum[hf * 128 + row] = l;
        named_bar_sync(1 + quarter, 64);
        const float l_tot = l + ex_sum[(hf ^ 1) * 128 + row];
        const int m = mtile * kTcBM + row;
        const bool direct = p.n_splits == 1;
        const float scale = direct ? 1.f / l_tot : 1.f;
        float* dst = nullptr;
        if (direct) {
            if (m < M) dst = p.out + (((int64_t)b * B + m / G) * p.n_q_heads + h * G + m % G) * kHeadDim + hf * 64;
        } else {
            dst = p.part_o + (part_base + row) * kHeadDim + hf * 64;
        }
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            float o[32];
            tmem_ld32(lane_base + 256 + hf * 64 + q * 32, o);
            if (dst) {
#pragma unroll
                for (int i = 0; i < 32; i += 4)
                    *reinterpret_cast<float4*>(dst + q * 32 + i) = make_float4(o[i] * scale, o[i + 1] * scale, o[i + 2] * scale, o[i + 3] * scale);
            }
        }
        if (hf == 0) {
            if (direct) {
                if (p.lse && m < M)
                    p.lse[((int64_t)b * B + m / G) * p.n_q_heads + h * G + m % G] = (m_used + log2f(l_tot)) * 0.6931471805599453f;
            } else {
                p.part_ml[part_base + row] = make_float2(m_used, l_tot);
            }
        }
    }

    // ---- teardown ----
    tc_fence_before();
    __syncthreads();
    if (warp == kTcMmaWarp) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(kTcTmemCols));
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
