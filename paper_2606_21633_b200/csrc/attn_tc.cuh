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
//   grid  = (KV splits, M tiles of 128 rows, units), 320 threads, 1 CTA / SM
//   warp 8      producer: full 128-key pool tiles arrive by TMA (cp.async.bulk.tensor, 128B swizzle,
//               2-stage K/V ring); the ragged tail of the pool and the in-block rows are written with
//               zero-filling cp.async so that rows past the end are exact zeros
//   warp 9      issues the MMAs (one elected lane): S[j&1] = Q K_j^T into a double-buffered TMEM tile,
//               then O += P_{j-1} V_{j-1}; completion is signalled with tcgen05.commit -> mbarrier
//   warps 0..7  softmax: thread (row, column half) reads 64 logits of its row from TMEM (tcgen05.ld),
//               exchanges the row maximum with its partner warp, exponentiates (ex2), accumulates the
//               row sum, splits P into a bf16 hi+lo pair and stores both to shared memory in the UMMA K-major layout.
//               The running maximum is only raised when it grows by more than 2^8 ("lazy rescale"):
//               O in TMEM is then rescaled in place (tcgen05.ld / tcgen05.st), which is rare.
//   split-KV partials (unnormalised O, running max, row sum) go to the workspace and are merged by
//   attn_combine_kernel; with one split the epilogue normalises and writes `out` directly.
#pragma once
#include <cuda.h>

#include "common.cuh"

namespace herald {

constexpr int kTcBM = 128;                       // query rows per CTA (UMMA M)
constexpr int kTcBN = 128;                       // keys per tile (UMMA N of QK^T, K of PV)
constexpr int kTcStages = 2;                     // K/V ring depth
constexpr int kTcThreads = 320;                  // 8 softmax warps + producer + MMA issuer
constexpr int kTcProducerWarp = 8, kTcMmaWarp = 9;
constexpr int kTcHalfBytes = kTcBN * 128;        // one [128 rows x 64 el] swizzled half tile (16 KB)
constexpr int kTcTileBytes = 2 * kTcHalfBytes;   // a [128 x 128] 16-bit tile = two halves (32 KB)
constexpr int kTcSmemQ = 0;
constexpr int kTcSmemP = kTcSmemQ + kTcTileBytes;                        // P_hi, then P_lo (bf16 pair, see below)
constexpr int kTcSmemKV = kTcSmemP + 2 * kTcTileBytes;                   // stage s: K at +2s tiles, V at +(2s+1)
constexpr int kTcSmemMisc = kTcSmemKV + kTcStages * 2 * kTcTileBytes;    // barriers, TMEM pointer, exchange buffers
constexpr int kTcMiscBytes = 2304;
constexpr int kTcSmemBytes = kTcSmemMisc + kTcMiscBytes;                 // 231,680 B of the 232,448 B a CTA may own
constexpr int kTcTmemCols = 512;                 // S0 [0,128) S1 [128,256) O [256,384)
constexpr float kTcRescaleThreshold = 8.f;       // log2 units

// barrier slots (8 bytes each) inside the misc area
enum { kBarKvFull = 0, kBarKvEmpty = kBarKvFull + kTcStages, kBarSFull = kBarKvEmpty + kTcStages, kBarSFree = kBarSFull + 2,
       kBarPFull = kBarSFree + 2, kBarPvDone, kBarCount };
constexpr int kTcMiscTmemPtr = 128;              // uint32
constexpr int kTcMiscMax = 256;                  // float [2 buffers][2 halves][128 rows]
constexpr int kTcMiscSum = kTcMiscMax;           // float [2 halves][128 rows]; reuses the max buffer after the last tile

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
    const int nt = t1 - t0;                                  // tile j of this CTA is key tile t1-1-j (ragged tiles first)
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
    if (warp == kTcProducerWarp && lane == 0) {
        for (int s = 0; s < kTcStages; ++s) {
            mbar_init(bar(kBarKvFull + s), 1);
            mbar_init(bar(kBarKvEmpty + s), 1);
        }
        for (int s = 0; s < 2; ++s) {
            mbar_init(bar(kBarSFull + s), 1);
            mbar_init(bar(kBarSFree + s), 8);
        }
        mbar_init(bar(kBarPFull), 8);
        mbar_init(bar(kBarPvDone), 1);
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
        const int t = t1 - 1 - j;
        const int valid = min(kTcBN, N - t * kTcBN);
        return (valid + 15) & ~15;
    };

    if (warp == kTcProducerWarp) {
        // =========================== producer ===========================
        auto issue_tma = [&](int j) {
            const int t = t1 - 1 - j, stage = j % kTcStages;
            if (lane == 0) {
                const uint32_t kdst = sbase + kTcSmemKV + stage * 2 * kTcTileBytes, vdst = kdst + kTcTileBytes;
                const uint32_t full = bar(kBarKvFull + stage);
                mbar_arrive_expect_tx(full, 2 * kTcTileBytes);
                tma_load_3d(kdst, &tm_k, 0, t * kTcBN, unit, full);
                tma_load_3d(kdst + kTcHalfBytes, &tm_k, 64, t * kTcBN, unit, full);
                tma_load_3d(vdst, &tm_v, 0, t * kTcBN, unit, full);
                tma_load_3d(vdst + kTcHalfBytes, &tm_v, 64, t * kTcBN, unit, full);
            }
        };
        auto fill_manual = [&](int j) {
            const int t = t1 - 1 - j, stage = j % kTcStages;
            const uint32_t kdst = sbase + kTcSmemKV + stage * 2 * kTcTileBytes, vdst = kdst + kTcTileBytes;
            const int rows = tile_cols(j);
            for (int c = lane; c < rows * 16; c += 32) {
                const int r = c >> 4, ch = c & 15;
                const int kj = t * kTcBN + r;
                const __nv_bfloat16 *ksrc = p.pool_k, *vsrc = p.pool_v;
                int bytes = 0;
                if (kj < n_pool) {
                    const int64_t off = ((int64_t)unit * p.cap + kj) * kHeadDim + ch * 8;
                    ksrc = p.pool_k + off;
                    vsrc = p.pool_v + off;
                    bytes = 16;
                } else if (kj < N) {
                    const int64_t off = (((int64_t)b * B + (kj - n_pool)) * p.n_kv_heads + h) * kHeadDim + ch * 8;
                    ksrc = p.k_blk + off;
                    vsrc = p.v_blk + off;
                    bytes = 16;
                }
                const uint32_t dst = (ch >> 3) * kTcHalfBytes + r * 128 + (((ch & 7) ^ (r & 7)) << 4);
                cp_async_16_zfill(kdst + dst, ksrc, bytes);
                cp_async_16_zfill(vdst + dst, vsrc, bytes);
            }
            cp_async_wait_all();
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(kBarKvFull + stage));
        };
        const int first = min(nt, kTcStages);
        for (int j = 0; j < first; ++j)
            if (t1 - 1 - j < n_full) issue_tma(j);          // asynchronous tiles first, so they fly during the manual fills
        for (int j = 0; j < first; ++j)
            if (t1 - 1 - j >= n_full) fill_manual(j);
        for (int j = kTcStages; j < nt; ++j) {
            mbar_wait(bar(kBarKvEmpty + j % kTcStages), ((j / kTcStages) - 1) & 1);
            if (t1 - 1 - j < n_full) issue_tma(j);
            else fill_manual(j);
        }
    } else if (warp == kTcMmaWarp) {
        // =========================== MMA issuer ===========================
        constexpr uint32_t idesc_pv = umma_idesc(/*A bf16*/ 1, /*B bf16*/ 1, /*A K-major*/ 0, /*B MN-major*/ 1, kTcBM, kHeadDim);
        const uint32_t q_base = sbase + kTcSmemQ, p_base = sbase + kTcSmemP;
        auto issue_pv = [&](int j) {   // O (+)= P_j V_j
            const int stage = j % kTcStages;
            mbar_wait(bar(kBarPFull), j & 1);
            tc_fence_after();
            if (lane == 0) {
                const uint32_t v_base = sbase + kTcSmemKV + stage * 2 * kTcTileBytes + kTcTileBytes;
                const int ksteps = tile_cols(j) >> 4;
                for (int kk = 0; kk < ksteps; ++kk) {
                    const uint32_t a_off = (kk >> 2) * kTcHalfBytes + (kk & 3) * 32;
                    const uint64_t bd = umma_desc_sw128(v_base + kk * 2048, kTcHalfBytes, 1024);
                    umma_ss(tmem + 256, umma_desc_sw128(p_base + a_off, 16, 1024), bd, idesc_pv, (j > 0 || kk > 0) ? 1u : 0u);
                    umma_ss(tmem + 256, umma_desc_sw128(p_base + kTcTileBytes + a_off, 16, 1024), bd, idesc_pv, 1u);
                }
                umma_commit(bar(kBarPvDone));
                umma_commit(bar(kBarKvEmpty + stage));
            }
            __syncwarp();
        };
        for (int j = 0; j < nt; ++j) {
            const int stage = j % kTcStages, sb = j & 1;
            mbar_wait(bar(kBarKvFull + stage), (j / kTcStages) & 1);
            if (j >= 2) mbar_wait(bar(kBarSFree + sb), ((j >> 1) - 1) & 1);
            tc_fence_after();
            if (lane == 0) {
                const uint32_t k_base = sbase + kTcSmemKV + stage * 2 * kTcTileBytes;
                const uint32_t idesc_s = umma_idesc(1, 1, 0, 0, kTcBM, tile_cols(j));
#pragma unroll
                for (int ks = 0; ks < 8; ++ks) {
                    const uint32_t off = (ks >> 2) * kTcHalfBytes + (ks & 3) * 32;
                    umma_ss(tmem + sb * 128, umma_desc_sw128(q_base + off, 16, 1024), umma_desc_sw128(k_base + off, 16, 1024),
                            idesc_s, ks > 0 ? 1u : 0u);
                }
                umma_commit(bar(kBarSFull + sb));
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
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(kBarSFree + sb));
            const int t = t1 - 1 - j;
            const int valid = N - t * kTcBN;                  // >= 1
            if (valid < kTcBN) {
#pragma unroll
                for (int i = 0; i < 64; ++i)
                    if (hf * 64 + i >= valid) s[i] = -INFINITY;
            }
            float mx = s[0];
#pragma unroll
            for (int i = 1; i < 64; ++i) mx = fmaxf(mx, s[i]);
            ex_max[(sb * 2 + hf) * 128 + row] = mx;
            named_bar_sync(1 + quarter, 64);
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
            if (j > 0) {
                mbar_wait(bar(kBarPvDone), (j - 1) & 1);       // PV_{j-1} finished: P buffer free, O up to date
                tc_fence_after();
                if (any) {
#pragma unroll
                    for (int q = 0; q < 2; ++q) {
                        float o[32];
                        tmem_ld32(lane_base + 256 + hf * 64 + q * 32, o);
#pragma unroll
                        for (int i = 0; i < 32; ++i) o[i] *= alpha;
                        tmem_st32(lane_base + 256 + hf * 64 + q * 32, o);
                    }
                    tmem_wait_st();
                }
            }
            // P row (64 weights of this column half) -> shared memory, UMMA K-major 128B-swizzled, as the bf16 pair
            // P = P_hi + P_lo: the pair carries 16 significand bits, so the PV product keeps the weights to ~2^-17
            // relative and peaked rows stay inside the 2e-3 output tolerance.
            uint8_t* prow = sgen + kTcSmemP + hf * kTcHalfBytes + row * 128;
#pragma unroll
            for (int c8 = 0; c8 < 8; ++c8) {
                uint32_t hi[4], lo[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) split_bf16(s[8 * c8 + 2 * e], s[8 * c8 + 2 * e + 1], hi[e], lo[e]);
                const int off = (c8 ^ (row & 7)) << 4;
                *reinterpret_cast<uint4*>(prow + off) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
                *reinterpret_cast<uint4*>(prow + kTcTileBytes + off) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
            }
            fence_proxy_async_smem();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(kBarPFull));
        }
        // ---- epilogue: O / l -> out (one split) or partials (split-KV) ----
        mbar_wait(bar(kBarPvDone), (nt - 1) & 1);
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
