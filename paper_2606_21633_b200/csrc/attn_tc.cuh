// Denoising-step attention over critical KV + in-block KV on the 5th-generation tensor cores
// (step a5 of DESIGN.md; "bidirectionally within the current block and causally to the
// cached KV", "denoises block n using the KV cache in the active sparse pool").
//
// One unit = (sequence b, KV head h).  Its M = B*G query rows attend over N = pool_len[b][h] pool rows
// followed by the B in-block rows; no mask.  The two products are real dense contractions
// (QK^T: [128 x d] x [d x 128], PV: [128 x 128] x [128 x d]) and run as tcgen05.mma (UMMA M=128,
// fp32 accumulate in TMEM).  The softmax weights P enter the PV product as a bf16 hi+lo pair (16 significand
// bits, two MMAs per k-step): a single bf16 P breaks the 2e-3 output tolerance on peaked rows, and kind::f16
// rejects an fp16 A operand next to a bf16 B operand (tried on B200: illegal instruction).
//
//   grid    = (KV splits S, M tiles, units); the S CTAs of one (unit, M tile) form a thread-block cluster
//   M tile  = `ipt` block rows x G heads (row r = block row r/G, head r%G; at most 128 rows), so the Q tile
//             is one TMA box of q_blk; rows past ipt*G are zeros
//   TMEM    = three S/P tiles of 128 columns + O (128 columns): QK^T runs up to three tiles ahead of PV, so the softmax
//             warps never wait for the tensor pipe and the pipe never waits for one softmax
//   keys    = key tile t < n_pool_tiles holds pool rows [128t, 128t+128) (one TMA box of the pool), the last tile the B
//             in-block rows (one TMA box of k_blk / v_blk); softmax is invariant to the key order
//             (dense mode, herald_dense_attn: tile t holds tokens [128t, 128t+128) of the paged cache itself, one
//             TMA box per 16-token page)
//   warp 16   K producer (+ Q): tiles arrive by TMA (cp.async.bulk.tensor, 128B swizzle) into a 3-stage ring; a
//             stage is free as soon as QK^T has read it (the S-full barrier of that tile).  Rows past the valid keys of a
//             tile (stale pool rows, zero fill) give logits that the softmax masks.
//   warp 17   V producer, same, a stage is free after PV (its PV-done barrier).  Where the valid keys of a tile are not a
//             multiple of the MMA k-step (16), it zeroes the few V rows up to the next multiple after the box has landed
//             (P is 0 there, but 0 x NaN would poison O).
//   warp 18   issues S[j%3] = Q K_j^T (one elected lane; tcgen05.commit -> mbarrier) once PV_{j-3} has finished with those
//             TMEM columns; owns the TMEM allocation
//   warp 19   issues O += P_j V_j with P read from TMEM.  One warp per product: a tcgen05.mma costs its issuing warp ~45
//             cycles and every barrier poll or commit ~100, which for one warp doing both products (24 MMAs, 4 commits, 3
//             polls per tile) came to 2.25k cycles per tile against 1.56k of tensor-pipe time.
//   warps 0-15 softmax: thread (row, column quarter) reads 32 logits of its row from TMEM (tcgen05.ld), exponentiates
//             (ex2) against the row reference of the pass, accumulates the row sum, and writes P back over its own 32 S
//             columns (tcgen05.st).  The reference is fixed before the first exponential of a pass -- the maximum of the
//             pass's first tile, exchanged once among the four warps that hold the row -- so inside the loop no warp waits
//             for another and the four warps of a scheduler hide each other's TMEM and barrier round trips.  A logit may
//             rise 2^64 above the reference before P, l or O leave fp32; if one does (or if the fast pass's row statistics
//             fail, below), the block votes, takes the row maximum it has seen as the reference and goes through its tiles a
//             second time, which cannot fail.
//   precision modes.  EXACT: P = bf16 hi + lo (two MMAs per k-step).  FAST, tried first by blocks whose share of the keys is
//             >= 1536 long: P is ONE bf16 (8 PV MMAs per tile instead of 16).
//             Rounding a weight to 8 significant bits moves an output element by sum_i eps_i p_i v_i with |eps_i| <= 2^-8,
//             pseudo-random: standard deviation <= 2^-8 sqrt(sum_i p_i^2) rms(v) / sqrt(3).  The fast pass accumulates
//             sum_i e_i^2 per row next to the row sum and is ACCEPTED only if every row of the block has sum_i p_i^2 <= 1/64
//             (<= 2.8e-4 rms(v) per element, 7 sigma inside the 2e-3 bar; one key alone may then weigh at most 1/8; flat rows
//             over n keys have sum p^2 ~ e/n) and no logit rose past its 2^30 margin.  Otherwise the block goes through its
//             tiles once more with the pair and leaves a note in the workspace: two failures in a row make it start with
//             the pair for its next 16 launches.  Blocks with short key shares never try: among a few hundred keys a
//             5-sigma logit already breaks the criterion, and one redone block delays its launch.
//   merge     split-KV partials never leave the chip: tile row r is owned by CTA r / rows_own of the cluster; the
//             other CTAs write their unnormalised O rows and (max, sum) straight from registers into the owner's
//             shared memory (st.shared::cluster into the owner's K ring, which its last QK^T has released: every CTA
//             tells its peers so with a remote mbarrier arrive as soon as that MMA has completed, about a tile
//             period before the partials exist), then arrive on the owner's merge barrier (release.cluster).  The
//             owner merges with its own registers, normalises, stages the rows in shared memory and writes `out`
//             with fully coalesced 512-byte rows.  No cluster-wide barrier after the main loop, no staging copy.
#pragma once
#include <cuda.h>

#include <type_traits>

#include "common.cuh"

namespace herald {

constexpr int kTcBM = 128;                       // query rows per CTA (UMMA M)
constexpr int kTcBN = 128;                       // keys per tile (UMMA N of QK^T, K of PV)
constexpr int kTcStages = 3;                     // depth of the K ring and of the V ring
constexpr int kTcSBufs = 3;                      // S/P tiles in TMEM
constexpr int kTcSoftmaxWarps = 16;              // 4 row quarters (TMEM lane quarters) x 4 column quarters
constexpr int kTcKWarp = 16, kTcVWarp = 17, kTcMmaWarp = 18, kTcPvWarp = 19;   // warp 18 issues QK^T (and owns TMEM), warp 19 issues PV
constexpr int kTcThreads = 20 * 32;
static_assert(kTcStages == kTcSBufs, "a ring stage falls free on the S-full / PV-done barrier of the same index");
constexpr int kTcMaxSplits = 8;                  // portable cluster size
constexpr int kTcHalfBytes = kTcBN * 128;        // one [128 rows x 64 el] swizzled half tile (16 KB)
constexpr int kTcTileBytes = 2 * kTcHalfBytes;   // a [128 x 128] bf16 tile = two halves (32 KB)
constexpr int kTcSmemQ = 0;
constexpr int kTcSmemK = kTcSmemQ + kTcTileBytes;                        // K ring
constexpr int kTcSmemV = kTcSmemK + kTcStages * kTcTileBytes;            // V ring
constexpr int kTcSmemMisc = kTcSmemV + kTcStages * kTcTileBytes;         // barriers, TMEM pointer, exchange buffers
constexpr int kTcMiscBytes = 2304;
constexpr int kTcSmemBytes = kTcSmemMisc + kTcMiscBytes;                 // 231,680 B of the 232,448 B a CTA may own
constexpr int kTcTmemCols = 512;                 // S0/P0 [0,128) S1/P1 [128,256) S2/P2 [256,384) O [384,512)
constexpr int kTcTmemO = kTcSBufs * 128;
constexpr float kTcExactJump = 64.f;             // log2 units a logit may rise above the reference of a pass with the hi + lo pair (P, l, O stay inside fp32)
// fast pass ("precision modes" in the header comment)
constexpr int kTcFastMinKeys = 1536;             // a block tries the fast pass only if its share of the keys is at least this long
constexpr float kTcFastJump = 30.f;              // the same for the fast pass, which also sums squares of the weights
constexpr float kTcFastCmax = 1.f / 64.f;        // bound on sum_i p_i^2 of a row for single-bf16 weights
constexpr uint32_t kTcHintMagic = 0x45580000u;   // note word of a block: "EX" | failures in a row << 8 | launches still to start exact
constexpr uint32_t kTcHintBackoff = 16;          // after two failed fast passes in a row a block starts exact for this many launches
// merge buffers: received partial rows alias the K ring, the output staging rows alias the V ring (both dead once
// every CTA of the cluster has left its main loop)
constexpr int kTcRowFloats = kHeadDim + 4;       // 528-byte rows: 16-byte accesses of 8 consecutive rows hit 8 bank groups
constexpr int kTcRecvO = kTcSmemK;                                               // float [S-1 sources][rows_own][132]
constexpr int kTcRecvML = kTcRecvO + kTcBM * kTcRowFloats * 4;                   // float2 [S-1 sources][ml_stride]
constexpr int kTcStageO = kTcSmemV;                                              // float [rows_own][132]: the finished rows
static_assert(kTcRecvML + (kTcBM + 2 * kTcMaxSplits) * 8 <= kTcSmemV, "receive buffers must fit in the K ring");
static_assert(kTcBM * kTcRowFloats * 4 <= kTcStages * kTcTileBytes, "output staging must fit in the V ring");

// barrier slots (8 bytes each) inside the misc area
enum { kBarKFull = 0, kBarVFull = kBarKFull + kTcStages,
       kBarSFull = kBarVFull + kTcStages, kBarPFull = kBarSFull + kTcSBufs, kBarPvDone = kBarPFull + kTcSBufs,
       kBarPvIssued = kBarPvDone + kTcSBufs, kBarQFull = kBarPvIssued + kTcSBufs, kBarVTail, kBarMerge, kBarPeerReady, kBarAck, kBarQkDone, kBarCount };
constexpr int kTcMiscTmemPtr = 240;              // uint32
constexpr int kTcMiscReady = 244;                // uint32: the word the peers' "receive buffer ready" signals land on
constexpr int kTcMiscMax = 256;                  // bf16 [2 buffers][4 column quarters][128 rows]; float [4][128] for the row sums
static_assert(kBarCount <= 32, "one barrier per lane of the initialising warp");
static_assert(kBarCount * 8 <= kTcMiscTmemPtr, "barriers overlap the TMEM pointer slot");
static_assert(kTcMiscMax + 2 * 4 * 128 * 2 <= kTcMiscBytes, "exchange buffer overflows the misc area");

struct AttnParams {
    const int32_t* pool_len;
    const int32_t* unit_order;   // optional [units]: units by decreasing pool length (attn_plan_kernel); NULL = identity
    // dense mode (layers that keep their full KV): the keys of tile t >= 1 are tokens [128(t-1), 128t) of the
    // paged cache itself -- 8 pages, one TMA box each -- and pool_len is unused
    const int32_t* page_table;   // [batch][max_pages]; NULL = sparse mode (keys from the pool)
    const int32_t* seq_lens;     // [batch]
    int32_t max_pages, max_seq_len;
    float* out;
    float* lse;
    int32_t n_q_heads, n_kv_heads, block_size, cap, n_splits;
    int32_t pool_batch; // sequences that own pools / cache pages: query sequence b reads those of b % pool_batch (query groups
                        // that share the prefix; == batch otherwise)
    int32_t ipt;        // block rows per M tile (ipt * G <= 128)
    int32_t pool_box;   // rows of the pool tensor-map box: min(cap, 128)
    float scale_log2;   // sm_scale * log2(e)
    uint32_t* mode_hint; // [blocks of the grid] in the workspace, or NULL: see kTcHintExact
    int32_t precision;   // 0 = automatic, 1 = exact only, 2 = every block tries the fast pass first (herald_tuning_t.attn_precision)
#ifdef HERALD_ATTN_TRACE
    unsigned long long* trace;   // [CTAs][64] clock64 stamps (debug builds only)
#endif
};

#ifdef HERALD_ATTN_TRACE
#define HERALD_STAMP(slot) do { if (p.trace && (slot) < 56) p.trace[(((size_t)blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x) * 64 + (slot)] = clock64(); } while (0)
#define HERALD_GSTAMP(slot) do { if (p.trace) { unsigned long long gt_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt_)); p.trace[(((size_t)blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x) * 64 + (slot)] = gt_; } } while (0)
#else
#define HERALD_GSTAMP(slot) do { } while (0)
#define HERALD_STAMP(slot) do { } while (0)
#endif

// ---- PTX wrappers -------------------------------------------------------------------------------
__device__ __forceinline__ bool elect_one() {   // one lane of a converged warp
    uint32_t pred;
    asm volatile(
        "{\n\t"
        ".reg .pred P;\n\t"
        "elect.sync _|P, 0xffffffff;\n\t"
        "selp.u32 %0, 1, 0, P;\n\t"
        "}" : "=r"(pred));
    return pred != 0;
}
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
// the same wait with acquire semantics at cluster scope: the barrier is arrived on by other CTAs of the cluster
// (mbarrier.arrive.release.cluster) after they have written this CTA's shared memory
__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity) {
    for (uint32_t spins = 0;; ++spins) {
        uint32_t done;
        asm volatile(
            "{\n\t"
            ".reg .pred p;\n\t"
            "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t"
            "}" : "=r"(done) : "r"(bar), "r"(parity) : "memory");
        if (done) return;
        if (spins > (1u << 26)) __trap();
    }
}
// cluster barrier in two halves (every thread of every CTA of the cluster executes both): the arrive publishes the
// barrier initialisation, the wait comes right before the first remote operation so that its latency is hidden
__device__ __forceinline__ void cluster_arrive_all() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait_all() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ uint32_t map_to_cta(uint32_t smem_addr, uint32_t cta_rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_addr), "r"(cta_rank));
    return r;
}
// asynchronous stores into the shared memory of another CTA of the cluster; each one counts its bytes on the destination's
// mbarrier (complete_tx), so the sender needs neither a fence nor an arrive and the receiver sees the data once its wait
// on that barrier returns
__device__ __forceinline__ void st_async_f4(uint32_t addr, float a, float b, float c, float d, uint32_t bar_cluster) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.f32 [%0], {%1, %2, %3, %4}, [%5];"
                 ::"r"(addr), "f"(a), "f"(b), "f"(c), "f"(d), "r"(bar_cluster) : "memory");
}
__device__ __forceinline__ void st_async_u32(uint32_t addr, uint32_t v, uint32_t bar_cluster) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b32 [%0], %1, [%2];" ::"r"(addr), "r"(v), "r"(bar_cluster) : "memory");
}
__device__ __forceinline__ void st_async_f2(uint32_t addr, float a, float b, uint32_t bar_cluster) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f32 [%0], {%1, %2}, [%3];"
                 ::"r"(addr), "f"(a), "f"(b), "r"(bar_cluster) : "memory");
}
// bulk copy own shared memory -> a peer's shared memory; completes bytes on the peer's mbarrier
__device__ __forceinline__ void bulk_copy_to_peer(uint32_t dst_cluster, uint32_t src_cta, uint32_t bytes, uint32_t bar_cluster) {
    asm volatile("cp.async.bulk.shared::cluster.shared::cta.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst_cluster), "r"(src_cta), "r"(bytes), "r"(bar_cluster) : "memory");
}
__device__ __forceinline__ void mbar_arrive_remote(uint32_t bar_cluster) {
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(bar_cluster) : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
}
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2, int c3, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
        ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar) : "memory");
}

__device__ __forceinline__ void cp_async_16_zfill(uint32_t dst, const void* src, int src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// Shared-memory matrix descriptor, 128-byte swizzle (layout type 2), descriptor version 1 (sm_100), split in two
// 32-bit words so that stepping through a tile is one 32-bit add on the low word:
//   low  word: (address >> 4) in bits [0,14), (leading byte offset >> 4) in bits [16,30)
//   high word: (stride byte offset >> 4) in bits [0,14), version 1 at bit 14, swizzle mode 2 at bits [29,32)
//   K-major operand : rows of 128 B (64 x 16-bit), 8-row groups `sbo` bytes apart, lbo unused (encoded 1)
//   MN-major operand: 64 contiguous MN elements per 128 B row, K rows 128 B apart, 8-row K groups `sbo`
//                     apart, next 64-element MN group `lbo` bytes away
__device__ __forceinline__ constexpr uint32_t umma_desc_lo(uint32_t smem_addr, uint32_t lbo_bytes) {
    return ((smem_addr & 0x3FFFFu) >> 4) | ((lbo_bytes >> 4) << 16);
}
__device__ __forceinline__ constexpr uint32_t umma_desc_hi(uint32_t sbo_bytes) {
    return (sbo_bytes >> 4) | (1u << 14) | (2u << 29);
}
// Instruction descriptor of tcgen05.mma.kind::f16: fp32 accumulate, A/B formats (0 = f16, 1 = bf16),
// majors (0 = K, 1 = MN), N >> 3 at bit 17, M >> 4 at bit 24.
__device__ __forceinline__ constexpr uint32_t umma_idesc(int a_fmt, int b_fmt, int a_mn, int b_mn, int M, int N) {
    return (1u << 4) | ((uint32_t)a_fmt << 7) | ((uint32_t)b_fmt << 10) | ((uint32_t)a_mn << 15) | ((uint32_t)b_mn << 16) |
           ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

// D[tmem] (+)= A[smem desc] * B[smem desc]
template <bool kAccumulate>
__device__ __forceinline__ void umma_ss(uint32_t d_tmem, uint32_t a_lo, uint32_t a_hi, uint32_t b_lo, uint32_t b_hi, uint32_t idesc) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        ".reg .b64 da, db;\n\t"
        "mov.b64 da, {%1, %2};\n\t"
        "mov.b64 db, {%3, %4};\n\t"
        "setp.ne.b32 p, %6, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], da, db, %5, p;\n\t"
        "}" ::"r"(d_tmem), "r"(a_lo), "r"(a_hi), "r"(b_lo), "r"(b_hi), "r"(idesc), "n"(kAccumulate ? 1 : 0) : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem desc]; A: row = TMEM lane, two 16-bit K elements per 32-bit column
__device__ __forceinline__ void umma_ts(uint32_t d_tmem, uint32_t a_tmem, uint32_t b_lo, uint32_t b_hi, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        ".reg .b64 db;\n\t"
        "mov.b64 db, {%2, %3};\n\t"
        "setp.ne.b32 p, %5, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], db, %4, p;\n\t"
        "}" ::"r"(d_tmem), "r"(a_tmem), "r"(b_lo), "r"(b_hi), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}

// 32 lanes x 32 consecutive 32-bit columns: thread t of the warp gets columns [col, col+32) of TMEM lane (lane base + t).
// The load is asynchronous: tmem_wait_ld() before the registers are used.
__device__ __forceinline__ void tmem_ld32_async(uint32_t taddr, float* v) {
    uint32_t* r = reinterpret_cast<uint32_t*>(v);
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
          "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
          "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t* v) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%32], "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31};"
        ::"r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]),
          "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]), "r"(v[16]), "r"(v[17]), "r"(v[18]),
          "r"(v[19]), "r"(v[20]), "r"(v[21]), "r"(v[22]), "r"(v[23]), "r"(v[24]), "r"(v[25]), "r"(v[26]), "r"(v[27]),
          "r"(v[28]), "r"(v[29]), "r"(v[30]), "r"(v[31]), "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// (x, y) -> packed bf16 pair hi = (bf16(x), bf16(y)) and the packed residual lo = (bf16(x - hi.x), bf16(y - hi.y))
__device__ __forceinline__ void split_bf16(float x, float y, uint32_t& hi, uint32_t& lo) {
    hi = pack_bf16(x, y);
    const float hx = __uint_as_float(hi << 16), hy = __uint_as_float(hi & 0xffff0000u);
    lo = pack_bf16(x - hx, y - hy);
}
// packed fp32 pairs (sm_100: one FMA-pipe instruction for two lanes' worth of elements)
__device__ __forceinline__ void ffma2(float& d0, float& d1, float a0, float a1, float b, float c) {   // d = a * b + c
    asm("{\n\t.reg .b64 ra, rb, rc, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %4};\n\tmov.b64 rc, {%5, %5};\n\t"
        "fma.rn.f32x2 rd, ra, rb, rc;\n\tmov.b64 {%0, %1}, rd;\n\t}" : "=f"(d0), "=f"(d1) : "f"(a0), "f"(a1), "f"(b), "f"(c));
}
__device__ __forceinline__ void ffma2v(float& d0, float& d1, float a0, float a1, float b, float c0, float c1) {   // d = a * b + c
    asm("{\n\t.reg .b64 ra, rb, rc, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %4};\n\tmov.b64 rc, {%5, %6};\n\t"
        "fma.rn.f32x2 rd, ra, rb, rc;\n\tmov.b64 {%0, %1}, rd;\n\t}" : "=f"(d0), "=f"(d1) : "f"(a0), "f"(a1), "f"(b), "f"(c0), "f"(c1));
}
__device__ __forceinline__ void ffma2w(float& d0, float& d1, float a0, float a1, float b0, float b1, float c0, float c1) {   // d = a * b + c
    asm("{\n\t.reg .b64 ra, rb, rc, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\tmov.b64 rc, {%6, %7};\n\t"
        "fma.rn.f32x2 rd, ra, rb, rc;\n\tmov.b64 {%0, %1}, rd;\n\t}" : "=f"(d0), "=f"(d1) : "f"(a0), "f"(a1), "f"(b0), "f"(b1), "f"(c0), "f"(c1));
}
__device__ __forceinline__ void fadd2(float& d0, float& d1, float a0, float a1, float b0, float b1) {   // d = a + b
    asm("{\n\t.reg .b64 ra, rb, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\t"
        "add.rn.f32x2 rd, ra, rb;\n\tmov.b64 {%0, %1}, rd;\n\t}" : "=f"(d0), "=f"(d1) : "f"(a0), "f"(a1), "f"(b0), "f"(b1));
}
__device__ __forceinline__ float fmax3(float a, float b, float c) {
    float r;
    asm("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
    return r;
}

__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t* v) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x8.b32 [%8], {%0, %1, %2, %3, %4, %5, %6, %7};"
        ::"r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t* v) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%16], "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15};"
        ::"r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]),
          "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]), "r"(taddr) : "memory");
}

// kTryFast = false: the exact pass only (every register of the softmax warps is spoken for: the block-uniform state of the
// two-pass control costs the exact loop ~9 % when it is compiled in).  The launcher picks the instantiation from the
// longest key share a block of the grid can have.
template <bool kTryFast>
__global__ void __launch_bounds__(kTcThreads, 1)
attn_tc_kernel(const __grid_constant__ CUtensorMap tm_k, const __grid_constant__ CUtensorMap tm_v,
               const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_kb,
               const __grid_constant__ CUtensorMap tm_vb, const AttnParams p) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t sbase = smem_u32(smem_raw);
    uint8_t* sgen = smem_raw;
    if (sbase & 1023u) __trap();   // the 128B-swizzled tiles need a 1024 B aligned base

    const int split = blockIdx.x, mtile = blockIdx.y;        // split == rank of this CTA in its cluster
    const int S = p.n_splits;
    const int G = p.n_q_heads / p.n_kv_heads, B = p.block_size;
    const int i0 = mtile * p.ipt;                            // first block row of this M tile
    const int rows_valid = min(p.ipt, B - i0) * G;           // tile rows that are real queries
    const int rows_box = p.ipt * G;                          // tile rows the Q box writes (zeros past the block)
    const int rows_own = (rows_box + S - 1) / S;             // tile rows merged and written by each CTA of the cluster (zero rows past the box are nobody's)
    const int ml_stride = (rows_own + 1) & ~1;               // float2 per source, padded to 16 bytes
    const int n_own = max(0, min(rows_own, rows_box - split * rows_own));   // rows of the box this CTA merges
    const int merge_bytes = (S - 1) * n_own * (kTcRowFloats * 4 + 8);   // partial rows and (m, l) the other CTAs send to this one
    const int g_inv = (65536 + G - 1) / G;                   // (r * g_inv) >> 16 == r / G for r < 128, G <= 8
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) { HERALD_STAMP(0); HERALD_GSTAMP(60); }

    const uint32_t misc = sbase + kTcSmemMisc;
    auto bar = [&](int i) { return misc + 8u * i; };
    volatile uint32_t* tmem_ptr_gen = reinterpret_cast<volatile uint32_t*>(sgen + kTcSmemMisc + kTcMiscTmemPtr);
    __nv_bfloat16* ex_max = reinterpret_cast<__nv_bfloat16*>(sgen + kTcSmemMisc + kTcMiscMax);
    float* ex_sum = reinterpret_cast<float*>(sgen + kTcSmemMisc + kTcMiscMax);   // after the last tile

    // ---- one-time setup: nothing here waits on global memory ------------------------------------------
    if (warp == kTcMmaWarp) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(misc + kTcMiscTmemPtr), "n"(kTcTmemCols));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    } else if (warp == kTcKWarp) {
        // one barrier per lane: every count is 1 except P-full (one arrive per softmax warp)
        if (lane < kBarCount) {
            const bool is_p = lane >= kBarPFull && lane < kBarPFull + kTcSBufs;
            mbar_init(bar(lane), is_p ? kTcSoftmaxWarps : 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncwarp();
        if (lane == 0) {
            // the partial rows the other CTAs of the cluster will send (st.async, counted in bytes)
            if (merge_bytes > 0) mbar_arrive_expect_tx(bar(kBarMerge), (uint32_t)merge_bytes);
            // ... and the 4-byte "my receive buffer is ready" signals of the S - 1 peers (asynchronous stores as well: a remote
            // mbarrier arrive with release semantics compiles to a device-wide memory barrier)
            if (S > 1) mbar_arrive_expect_tx(bar(kBarPeerReady), (uint32_t)(S - 1) * 4u);
            if (S > 1) mbar_arrive_expect_tx(bar(kBarAck), (uint32_t)(S - 1) * 4u);
        }
        if (lane < 5) {
            const CUtensorMap* tm = lane == 0 ? &tm_q : lane == 1 ? &tm_k : lane == 2 ? &tm_v : lane == 3 ? &tm_kb : &tm_vb;
            asm volatile("prefetch.tensormap [%0];" ::"l"(tm) : "memory");
        }
    } else if (warp < kTcSoftmaxWarps) {
        // Q rows the TMA box does not write are zeros (all 16 chunks of a row, so the swizzle does not matter)
        for (int c = tid; c < (kTcBM - rows_box) * 16; c += kTcSoftmaxWarps * 32) {
            const int r = rows_box + (c >> 4), ch = c & 15;
            *reinterpret_cast<uint4*>(sgen + kTcSmemQ + (ch >> 3) * kTcHalfBytes + r * 128 + ((ch & 7) << 4)) = make_uint4(0, 0, 0, 0);
        }
        fence_proxy_async_smem();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_ptr_gen;
    if (S > 1) cluster_arrive_all();   // the barriers of this CTA are initialised: remote arrives may come from here on
    if (tid == 0) HERALD_STAMP(1);

    // Programmatic dependent launch: this grid may have been scheduled while the previous kernel of the stream was
    // still draining.  Everything above is on-chip; nothing is read from global memory before that kernel has
    // completed and flushed.  (Requesting pool tiles or reading the pool lengths ahead of the wait was measured: the early
    // requests queue in front of the Q tile and compete with the draining grid, 16.4 -> 16.7 us per C2 step.)
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (tid == 0) HERALD_GSTAMP(61);
    // blocks are dispatched in blockIdx order: with a plan (attn_plan_kernel) slot z holds the unit with the z-th longest
    // pool, so that the long units start first and the short ones fill the tail of a multi-wave grid
    const int unit = p.unit_order ? p.unit_order[blockIdx.z] : (int)blockIdx.z;
    const int b = unit / p.n_kv_heads, h = unit % p.n_kv_heads;
    if (warp == kTcKWarp) {
        // the Q tile is what the first MMA waits for longest: it is requested before the pool length is even read
        // (one box of q_blk [batch][B][H_q][128] = (64 channels, G heads, ipt block rows) per half)
        if (elect_one()) {
            mbar_arrive_expect_tx(bar(kBarQFull), (uint32_t)rows_box * 256u);
            tma_load_4d(sbase + kTcSmemQ, &tm_q, 0, h * G, i0, b, bar(kBarQFull));
            tma_load_4d(sbase + kTcSmemQ + kTcHalfBytes, &tm_q, 64, h * G, i0, b, bar(kBarQFull));
        }
        __syncwarp();
    }
    const int b_pool = b % p.pool_batch, unit_pool = b_pool * p.n_kv_heads + h;   // whose keys: the group's prefix owner
    const bool paged = p.page_table != nullptr;
    const int n_pool = paged ? max(0, min(p.seq_lens[b_pool], p.max_seq_len)) : max(0, min(p.pool_len[unit_pool], p.cap));
    const int n_pool_tiles = (n_pool + kTcBN - 1) / kTcBN;
    const int n_tiles = n_pool_tiles + 1;                    // key tile t < n_pool_tiles = pool rows [128t, 128t+128); the last tile = the in-block rows
    const int per = (n_tiles + S - 1) / S;
    const int t0 = split * per, t1 = min(n_tiles, t0 + per);
    const int nt = max(t1 - t0, 0);                          // tile j of this CTA is key tile t0 + j

    auto tile_valid = [&](int j) {  // valid keys of this CTA's j-th tile (>= 1)
        const int t = t0 + j;
        return t == n_pool_tiles ? B : min(kTcBN, n_pool - t * kTcBN);
    };
    auto tile_cols = [&](int j) {   // key columns of the tile that the MMAs touch (multiple of 16)
        return (tile_valid(j) + 15) & ~15;
    };

    // softmax threads: row of the M tile == TMEM lane, column quarter cq of every key tile
    const int quarter = warp & 3, cq = (warp >> 2) & 3;
    const int row = quarter * 32 + lane;
    const uint32_t lane_base = tmem + ((uint32_t)(quarter * 32) << 16);
    float m_used = -INFINITY, l_run = 0.f;   // running max (log2 units) and the sum of this thread's quarter row
    float q_run = 0.f;                       // fast pass: the sum of the squared weights of this thread's quarter row
    bool jumped = false;                     // this thread's rows fail the criteria of the pass
    float mx_all = -INFINITY;                // the largest logit this thread has seen (raw, before the scale)

    // One pass over the key tiles, or two (header comment, "softmax" and "precision modes"): if the pass fails its criteria,
    // every role goes through the same tiles once more.  Ring and TMEM barrier phases simply run on: tile j of the second pass
    // is pipeline step jb + j.
    int keys_here = 0;
    if (kTryFast)
        for (int j = 0; j < nt; ++j) keys_here += tile_valid(j);
    const int cta_lin = (blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
    bool fast = false;                       // block-uniform
    uint32_t hint = 0;
    if (kTryFast && nt > 0 && p.precision != 1 && (p.precision == 2 || keys_here >= kTcFastMinKeys)) {
        hint = p.mode_hint ? p.mode_hint[cta_lin] : 0u;
        if ((hint & 0xffff0000u) != kTcHintMagic || (hint & 0xffu) > kTcHintBackoff) hint = kTcHintMagic;   // uninitialised workspace: no history
        fast = p.precision == 2 || (hint & 0xffu) == 0;
    }
    const bool tried_fast = fast;
    int n_fixed = 0;                         // V tiles whose tail rows were zeroed so far (phase of kBarVTail; V producer)
    int jb_rt = 0;
#define HERALD_JB jb_rt
    for (int pass = 0; nt > 0; ++pass) {
        if (warp == kTcKWarp || warp == kTcVWarp) {
            // =========================== producers: one warp streams K tiles (and Q), one streams V tiles ===========================
            const bool is_k = warp == kTcKWarp;
            const CUtensorMap* map = is_k ? &tm_k : &tm_v;
            const CUtensorMap* map_blk = is_k ? &tm_kb : &tm_vb;
            // a K stage is free once QK^T has read it (= S of that tile is full), a V stage once PV has (= PV done): same index, same phase
            const int bar_full = is_k ? kBarKFull : kBarVFull, bar_empty = is_k ? kBarSFull : kBarPvDone;
            const uint32_t ring = sbase + (is_k ? kTcSmemK : kTcSmemV);
            uint8_t* ring_gen = sgen + (is_k ? kTcSmemK : kTcSmemV);
            // dense mode: the page ids of a tile are fetched one tile ahead, so that their round trip does not sit between a
            // ring slot falling free and its TMA requests
            auto tile_phys = [&](int jj) -> int {
                const int tt = t0 + jj;
                if (!paged || jj >= nt || tt == n_pool_tiles) return 0;
                const int n_pg = (tile_valid(jj) + kPageSize - 1) / kPageSize;
                return lane < n_pg ? __ldg(p.page_table + (int64_t)b_pool * p.max_pages + tt * (kTcBN / kPageSize) + lane) : 0;
            };
            int phys_next = tile_phys(0);
            for (int j = 0; j < nt; ++j) {
                const int jg = HERALD_JB + j, stage = jg % kTcStages, t = t0 + j;
                const int my_phys = phys_next;
                phys_next = tile_phys(j + 1);
                if (jg >= kTcStages) mbar_wait(bar(bar_empty + stage), ((jg / kTcStages) - 1) & 1);
                if (!is_k && jg == 0) named_bar_sync(9, 64);   // Q and K_0 are requested before any V tile
                const uint32_t dst = ring + stage * kTcTileBytes, full = bar(bar_full + stage);
                const int valid = tile_valid(j), cols = (valid + 15) & ~15;
                const bool fix = !is_k && cols != valid;      // V rows [valid, cols) must be zeros: land on kBarVTail first
                const uint32_t land = fix ? bar(kBarVTail) : full;
                if (elect_one()) {
                    if (t == n_pool_tiles) {   // in-block rows: box = (64 channels, 1 head, B rows, 1 sequence) per half
                        mbar_arrive_expect_tx(land, (uint32_t)B * 256u);
                        tma_load_4d(dst, map_blk, 0, h, 0, b, land);
                        tma_load_4d(dst + kTcHalfBytes, map_blk, 64, h, 0, b, land);
                    } else if (!paged) {   // pool rows: box = (64 channels, pool_box rows, 1 unit) per half; rows past cap are zero-filled
                        mbar_arrive_expect_tx(land, (uint32_t)p.pool_box * 256u);
                        tma_load_3d(dst, map, 0, t * kTcBN, unit_pool, land);
                        tma_load_3d(dst + kTcHalfBytes, map, 64, t * kTcBN, unit_pool, land);
                    }
                }
                __syncwarp();
                if (paged && t != n_pool_tiles) {
                    // dense mode: the 128 tokens of the tile are 8 pages of the cache; page i lands on tile rows [16i, 16i+16)
                    // (2 KB per half: a whole number of 1 KB swizzle atoms).  Pages past the sequence are not requested.
                    const int n_pg = (valid + kPageSize - 1) / kPageSize;
                    if (lane == 0) mbar_arrive_expect_tx(land, (uint32_t)n_pg * kPageSize * 256u);
                    __syncwarp();
                    if (lane < n_pg) {
                        tma_load_4d(dst + lane * (kPageSize * 128), map, 0, h, 0, my_phys, land);
                        tma_load_4d(dst + kTcHalfBytes + lane * (kPageSize * 128), map, 64, h, 0, my_phys, land);
                    }
                    __syncwarp();
                }
                if (is_k && jg == 0) named_bar_sync(9, 64);
                if (fix) {
                    mbar_wait(bar(kBarVTail), n_fixed & 1);
                    ++n_fixed;
                    for (int c = lane; c < (cols - valid) * 16; c += 32) {   // all 16 chunks of a row: the swizzle does not matter
                        const int r = valid + (c >> 4), ch = c & 15;
                        *reinterpret_cast<uint4*>(ring_gen + stage * kTcTileBytes + (ch >> 3) * kTcHalfBytes + r * 128 + ((ch & 7) << 4)) = make_uint4(0, 0, 0, 0);
                    }
                    fence_proxy_async_smem();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(full);
                }
            }
        } else if (warp == kTcMmaWarp) {
            // =========================== QK^T issuer ===========================
            // Two warps feed the tensor pipe, one per product: what an issuing warp does between its MMAs (barrier polls,
            // commits, descriptor set-up: about 1.1k cycles per tile next to 1.1k of issue) was longer than the pipe's own
            // 1.56k per tile while one warp did both.  S_j overwrites the TMEM columns PV_{j-3} reads its P from: this warp waits
            // until the other one has ISSUED that PV (tcgen05.fence::before_thread_sync + arrive there, wait +
            // fence::after_thread_sync here order the two groups of MMAs; the pipe executes them in that order) -- not until
            // it has completed, which put a whole PV between a block's P_j and its S_{j+3}.
            constexpr uint32_t hi_k = umma_desc_hi(1024);
            const uint32_t q_lo = umma_desc_lo(sbase + kTcSmemQ, 16);
            if (pass == 0) {
                mbar_wait(bar(kBarQFull), 0);
                if (lane == 0) HERALD_GSTAMP(57);
            }
#pragma unroll 1
            for (int j = 0; j < nt; ++j) {   // S_j = Q K_j^T into S buffer j % 3, which held P_{j-3}
                const int jg = HERALD_JB + j, stage = jg % kTcStages, sb = jg % kTcSBufs;
                if (jg >= kTcSBufs) mbar_wait(bar(kBarPvIssued + sb), ((jg / kTcSBufs) - 1) & 1);
                mbar_wait(bar(kBarKFull + stage), (jg / kTcStages) & 1);
                tc_fence_after();
                if (lane == 0) { HERALD_STAMP(8 + 4 * jg); if (jg == 0) HERALD_GSTAMP(58); }
                if (elect_one()) {
                    const uint32_t k_lo = umma_desc_lo(sbase + kTcSmemK + stage * kTcTileBytes, 16);
                    const uint32_t idesc_s = umma_idesc(1, 1, 0, 0, kTcBM, tile_cols(j));
                    const uint32_t s_base = tmem + sb * 128;
#pragma unroll
                    for (int ks = 0; ks < 8; ++ks) {
                        const uint32_t off = ((ks >> 2) * kTcHalfBytes + (ks & 3) * 32) >> 4;
                        if (ks == 0) umma_ss<false>(s_base, q_lo + off, hi_k, k_lo + off, hi_k, idesc_s);
                        else umma_ss<true>(s_base, q_lo + off, hi_k, k_lo + off, hi_k, idesc_s);
                    }
                    umma_commit(bar(kBarSFull + sb));                // S_j is complete; K stage j % 3 has been read
                    if (j == nt - 1) umma_commit(bar(kBarQkDone));   // every QK^T of this pass has read its K tile (phase = pass)
                }
                __syncwarp();
            }
        } else if (warp == kTcPvWarp) {
            // =========================== PV issuer ===========================
            constexpr uint32_t idesc_pv = umma_idesc(/*A bf16*/ 1, /*B bf16*/ 1, /*A K-major*/ 0, /*B MN-major*/ 1, kTcBM, kHeadDim);
            constexpr uint32_t hi_k = umma_desc_hi(1024);
#pragma unroll 1
            for (int j = 0; j < nt; ++j) {   // O (+)= (P_hi + P_lo)_j V_j, P read from TMEM (it overlays S_j)
                const int jg = HERALD_JB + j, stage = jg % kTcStages, sb = jg % kTcSBufs;
                mbar_wait(bar(kBarVFull + stage), (jg / kTcStages) & 1);
                mbar_wait(bar(kBarPFull + sb), (jg / kTcSBufs) & 1);
                tc_fence_after();
                if (lane == 0) HERALD_STAMP(8 + 4 * jg + 3);
                if (elect_one()) {
                    const uint32_t v_lo = umma_desc_lo(sbase + kTcSmemV + stage * kTcTileBytes, kTcHalfBytes);
                    const uint32_t p_base = tmem + sb * 128, o_base = tmem + kTcTmemO;
                    const int ksteps = tile_cols(j) >> 4;
                    const uint32_t acc0 = j > 0 ? 1u : 0u;
                    if (kTryFast && fast) {     // one bf16 per weight, at the head of each column quarter's own S columns
                        if (ksteps == 8) {
#pragma unroll
                            for (int kk = 0; kk < 8; ++kk)
                                umma_ts(o_base, p_base + (kk >> 1) * 32 + (kk & 1) * 8, v_lo + kk * 128, hi_k, idesc_pv, kk > 0 ? 1u : acc0);
                        } else {
                            for (int kk = 0; kk < ksteps; ++kk)
                                umma_ts(o_base, p_base + (kk >> 1) * 32 + (kk & 1) * 8, v_lo + kk * 128, hi_k, idesc_pv, kk > 0 ? 1u : acc0);
                        }
                    } else if (ksteps == 8) {
#pragma unroll
                        for (int kk = 0; kk < 8; ++kk) {
                            umma_ts(o_base, p_base + (kk >> 1) * 32 + (kk & 1) * 8, v_lo + kk * 128, hi_k, idesc_pv, kk > 0 ? 1u : acc0);
                            umma_ts(o_base, p_base + (kk >> 1) * 32 + (kk & 1) * 8 + 16, v_lo + kk * 128, hi_k, idesc_pv, 1u);
                        }
                    } else {
                        for (int kk = 0; kk < ksteps; ++kk) {
                            umma_ts(o_base, p_base + (kk >> 1) * 32 + (kk & 1) * 8, v_lo + kk * 128, hi_k, idesc_pv, kk > 0 ? 1u : acc0);
                            umma_ts(o_base, p_base + (kk >> 1) * 32 + (kk & 1) * 8 + 16, v_lo + kk * 128, hi_k, idesc_pv, 1u);
                        }
                    }
                    umma_commit(bar(kBarPvDone + sb));               // P_j and V stage j % 3 have been read
                    tc_fence_before();
                    mbar_arrive(bar(kBarPvIssued + sb));             // the QK^T issuer may queue S_{j+3} behind these MMAs
                }
                __syncwarp();
            }
        } else {
            // =========================== softmax warps ===========================
            // The warps run free of each other: the row reference is fixed before the first exponential of a pass (pass 0:
            // the maximum of the first tile, exchanged once among the four column quarters; pass 1: the row maximum that
            // pass 0 saw), so no thread waits for another one inside the loop and the four warps of a scheduler hide each
            // other's TMEM and barrier round trips.  Because they no longer meet, a thread may only overwrite S columns it
            // has read itself: its 32 weights go to its own 32 S columns, P_hi in the first 16, P_lo in the last 16.
            auto softmax_pass = [&](auto single_tag) {
                constexpr bool kSingle = decltype(single_tag)::value;   // one bf16 per weight (fast pass) or the hi + lo pair
                constexpr float kJump = kSingle ? kTcFastJump : kTcExactJump;
                for (int j = 0; j < nt; ++j) {
                    const int jg = jb_rt + j, sb = jg % kTcSBufs;
                    mbar_wait(bar(kBarSFull + sb), (jg / kTcSBufs) & 1);
                    tc_fence_after();
                    if (tid == 0) { HERALD_STAMP(8 + 4 * jg + 1); if (jg == 0) HERALD_GSTAMP(62); }
                    float s[32];
                    tmem_ld32_async(lane_base + sb * 128 + cq * 32, s);
                    tmem_wait_ld();
                    const int valid = tile_valid(j);
                    if (valid < kTcBN) {
#pragma unroll
                        for (int i = 0; i < 32; ++i)
                            if (cq * 32 + i >= valid) s[i] = -INFINITY;
                    }
                    float mx = fmax3(s[0], s[1], s[2]);
#pragma unroll
                    for (int i = 3; i + 1 < 32; i += 2) mx = fmax3(mx, s[i], s[i + 1]);
                    mx = fmaxf(mx, s[31]);
                    mx_all = fmaxf(mx_all, mx);
                    if (j == 0 && pass == 0) {
                        // the reference only has to be common to the four column quarters: it is exchanged rounded up to bf16
                        ex_max[cq * 128 + row] = __float2bfloat16_ru(mx);
                        named_bar_sync(1 + quarter, 128);             // the four warps that hold these 32 rows
                        float mrow = __bfloat162float(ex_max[row]);
#pragma unroll
                        for (int c = 1; c < 4; ++c) mrow = fmaxf(mrow, __bfloat162float(ex_max[c * 128 + row]));
                        m_used = mrow * p.scale_log2;
                    } else if (mx * p.scale_log2 > m_used + kJump) {
                        jumped = true;    // the reference cannot move without the other quarters: the block goes through its tiles again
                    }
                    // The exponentials (MUFU, 16 per clock and SM: the scarce unit) and the splitting arithmetic of earlier
                    // pairs share one unrolled loop so that the scheduler interleaves them.
                    // A operand of the PV MMA: row = lane, two keys per 32-bit column.  The weights leave for TMEM eight columns at
                    // a time, so that at most 16 of them sit in registers next to the logits still to be exponentiated.
                    float sum0 = 0.f, sum1 = 0.f, sq0 = 0.f, sq1 = 0.f;
#pragma unroll
                    for (int half = 0; half < 2; ++half) {
                        uint32_t hi[8], lo[kSingle ? 1 : 8];
#pragma unroll
                        for (int ii = 0; ii < 8; ++ii) {
                            const int i = half * 8 + ii;
                            float x0, x1;
                            ffma2(x0, x1, s[2 * i], s[2 * i + 1], p.scale_log2, -m_used);
                            const float e0 = fast_exp2(x0), e1 = fast_exp2(x1);
                            fadd2(sum0, sum1, sum0, sum1, e0, e1);
                            hi[ii] = pack_bf16(e0, e1);
                            if (kSingle) {
                                ffma2w(sq0, sq1, e0, e1, e0, e1, sq0, sq1);
                            } else {
                                float r0, r1;
                                ffma2v(r0, r1, __uint_as_float(hi[ii] << 16), __uint_as_float(hi[ii] & 0xffff0000u), -1.f, e0, e1);   // e - hi, exact
                                lo[ii] = pack_bf16(r0, r1);
                            }
                        }
                        tmem_st8(lane_base + sb * 128 + cq * 32 + half * 8, hi);
                        if (!kSingle) tmem_st8(lane_base + sb * 128 + cq * 32 + 16 + half * 8, lo);
                    }
                    l_run += sum0 + sum1;
                    if (kSingle) q_run += sq0 + sq1;
                    tmem_wait_st();
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar(kBarPFull + sb));
                    if (tid == 0) HERALD_STAMP(8 + 4 * jg + 2);
                }
            };
            l_run = 0.f, q_run = 0.f, jumped = false;
            if (kTryFast && fast) {
                softmax_pass(std::true_type{});
                // the verdict (the last PV is still running): row sums of e and e^2 over the four column quarters, exchanged as one
                // bf16 pair per thread (the sum rounded down, the sum of squares rounded up: the test stays on the safe side)
                uint32_t* ex_pair = reinterpret_cast<uint32_t*>(ex_max);
                const __nv_bfloat16 lb = __float2bfloat16_rd(l_run), qb = __float2bfloat16_ru(q_run);
                ex_pair[cq * 128 + row] = (uint32_t)__bfloat16_as_ushort(lb) | ((uint32_t)__bfloat16_as_ushort(qb) << 16);
                named_bar_sync(1 + quarter, 128);
                float l_row = 0.f, q_row = 0.f;
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const uint32_t v = ex_pair[c * 128 + row];
                    l_row += __uint_as_float(v << 16);
                    q_row += __uint_as_float(v & 0xffff0000u);
                }
                if (!(q_row <= kTcFastCmax * l_row * l_row)) jumped = true;
            } else {
                softmax_pass(std::false_type{});
            }
        }
        // ---- end of the first pass: one block-wide vote (every warp is here shortly after the last P was handed over) ----
        if (pass == 0) {
            fast = false;
            if (__syncthreads_or(warp < kTcSoftmaxWarps && jumped ? 1 : 0)) {
                // once more (the first PV of the pass overwrites O), with the hi + lo pair and the row maximum that this pass
                // saw as the reference: nothing can rise above it
                jb_rt += nt;
                if (warp < kTcSoftmaxWarps) {
                    ex_max[cq * 128 + row] = __float2bfloat16_ru(mx_all);
                    named_bar_sync(1 + quarter, 128);
                    float mrow = __bfloat162float(ex_max[row]);
#pragma unroll
                    for (int c = 1; c < 4; ++c) mrow = fmaxf(mrow, __bfloat162float(ex_max[c * 128 + row]));
                    m_used = mrow * p.scale_log2;
                }
                continue;
            }
        }
        break;
    }
    const int n_passes = jb_rt > 0 ? 2 : 1;
    if (kTryFast && tid == 0 && p.mode_hint && nt > 0) {
        // the note for this block's next launch.  One failed fast pass costs one redo and nothing more (on N(0,1)-like data a
        // row with a 6-sigma logit turns up in some block now and then, and a block that starts exact holds up its whole
        // launch); two in a row mean the data is peaked: exact for kTcHintBackoff launches, then one more try.
        if (tried_fast) {
            const uint32_t streak = n_passes == 2 ? min(((hint >> 8) & 0xffu) + 1u, 255u) : 0u;
            p.mode_hint[cta_lin] = kTcHintMagic | (streak << 8) | (streak >= 2 ? kTcHintBackoff : 0u);
        } else if (hint != 0 && (hint & 0xffu) != 0) {
            p.mode_hint[cta_lin] = hint - 1;
        }
    }
    if (warp < kTcSoftmaxWarps && nt > 0) {
        // A parity wait is only sound when the waiter is at most one phase behind: the slot of the last PV completes next
        // for a PV three pipeline steps later, which does not exist.
        const int jl = HERALD_JB + nt - 1;
#undef HERALD_JB
        mbar_wait(bar(kBarPvDone + (jl % kTcSBufs)), (jl / kTcSBufs) & 1);
        tc_fence_after();
        if (tid == 0) HERALD_STAMP(2);
    }

    // ---- merge of the split-KV partials inside the cluster, normalisation, output -----------------------
    // The K ring of a CTA is dead once its last QK^T has completed: it receives the other CTAs' partial rows.  The
    // K producer (idle by then) waits for that MMA and tells every peer with a remote arrive on its kBarPeerReady;
    // this happens about a tile period before any partial exists, so no sender ever waits for it in practice.
    if (warp == kTcKWarp && nt == 0) mbar_wait(bar(kBarQFull), 0);   // the Q box was requested: it must have landed before the CTA exits
    if (warp == kTcKWarp && S > 1) {
        if (nt > 0) mbar_wait(bar(kBarQkDone), (n_passes - 1) & 1);   // the last pass has read its last K tile
        cluster_wait_all();   // every CTA of the cluster has initialised its barriers (only this warp arrives on a peer's before it is told to)
        if (lane < S - 1) {
            const uint32_t peer = lane < split ? lane : lane + 1;
            st_async_u32(map_to_cta(misc + kTcMiscReady, peer), 1u, map_to_cta(bar(kBarPeerReady), peer));
        }
    }
    // the next kernel of the stream may be scheduled from here on: its blocks take the SMs as this grid's blocks exit
    asm volatile("griddepcontrol.launch_dependents;");
    const int owner = row / rows_own, row_l = row - owner * rows_own;
    float o[32];
    float l_tot = 0.f;
    if (warp < kTcSoftmaxWarps) {
        if (nt > 0) {
            ex_sum[cq * 128 + row] = l_run;
            tmem_ld32_async(lane_base + kTcTmemO + cq * 32, o);
            tmem_wait_ld();
            named_bar_sync(1 + quarter, 128);
            l_tot = (ex_sum[row] + ex_sum[128 + row]) + (ex_sum[256 + row] + ex_sum[384 + row]);
        } else {
#pragma unroll
            for (int i = 0; i < 32; ++i) o[i] = 0.f;
        }
        if (tid == 0) HERALD_STAMP(6);
        if (S > 1) {
            if (owner != split && row < rows_box) {
                float4* stg = reinterpret_cast<float4*>(sgen + kTcStageO + (row * kTcRowFloats + cq * 32) * 4);
#pragma unroll
                for (int i = 0; i < 8; ++i) stg[i] = make_float4(o[4 * i], o[4 * i + 1], o[4 * i + 2], o[4 * i + 3]);
                if (cq == 0) {
                    mbar_wait_cluster(bar(kBarPeerReady), 0);
                    const int src_slot = split < owner ? split : split - 1;
                    st_async_f2(map_to_cta(sbase + kTcRecvML + (src_slot * ml_stride + row_l) * 8, owner), nt > 0 ? m_used : -INFINITY, l_tot,
                                map_to_cta(bar(kBarMerge), owner));
                }
            }
            fence_proxy_async_smem();
            named_bar_sync(1 + quarter, 128);
            if (cq == 0 && lane == 0) {
                mbar_wait_cluster(bar(kBarPeerReady), 0);
                const int r0 = quarter * 32, r1 = min(r0 + 32, rows_box);
                for (int o2 = 0; o2 < S; ++o2) {
                    if (o2 == split) continue;
                    const int ra = max(r0, o2 * rows_own), rb = min(r1, (o2 + 1) * rows_own);
                    if (ra >= rb) continue;
                    const int src_slot = split < o2 ? split : split - 1;
                    bulk_copy_to_peer(map_to_cta(sbase + kTcRecvO + ((src_slot * rows_own + (ra - o2 * rows_own)) * kTcRowFloats) * 4, o2),
                                      sbase + kTcStageO + ra * kTcRowFloats * 4, (uint32_t)(rb - ra) * kTcRowFloats * 4, map_to_cta(bar(kBarMerge), o2));
                }
            }
        }
    }
    if (tid == 0) HERALD_STAMP(5);
    if (warp < kTcSoftmaxWarps && owner == split && row < rows_box) {
        if (merge_bytes > 0) mbar_wait_cluster(bar(kBarMerge), 0);   // every partial row addressed to this CTA has landed
        if (tid == 0) HERALD_STAMP(3);
        if (row < rows_valid) {
            const float* recv_o = reinterpret_cast<const float*>(sgen + kTcRecvO);
            const float2* recv_ml = reinterpret_cast<const float2*>(sgen + kTcRecvML);
            float mstar = nt > 0 ? m_used : -INFINITY;
#pragma unroll 1
            for (int s = 0; s < S - 1; ++s) mstar = fmaxf(mstar, recv_ml[s * ml_stride + row_l].x);
            const float w_self = nt > 0 ? fast_exp2(m_used - mstar) : 0.f;
            float den = w_self * l_tot;
#pragma unroll
            for (int i = 0; i < 32; ++i) o[i] *= w_self;
#pragma unroll 1
            for (int s = 0; s < S - 1; ++s) {
                const float2 ml = recv_ml[s * ml_stride + row_l];
                if (ml.x == -INFINITY) continue;                  // empty split: its rows carry nothing
                const float w = fast_exp2(ml.x - mstar);
                den += w * ml.y;
                const float4* src = reinterpret_cast<const float4*>(recv_o + (s * rows_own + row_l) * kTcRowFloats + cq * 32);
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const float4 v = src[i];
                    o[4 * i] += w * v.x; o[4 * i + 1] += w * v.y; o[4 * i + 2] += w * v.z; o[4 * i + 3] += w * v.w;
                }
            }
            const float inv = 1.f / den;
            // the V ring is dead (this thread has seen the last PV of the CTA complete): it stages the finished rows
            float4* dst = reinterpret_cast<float4*>(sgen + kTcStageO + (row * kTcRowFloats + cq * 32) * 4);
#pragma unroll
            for (int i = 0; i < 8; ++i) dst[i] = make_float4(o[4 * i] * inv, o[4 * i + 1] * inv, o[4 * i + 2] * inv, o[4 * i + 3] * inv);
            if (p.lse && cq == 0) {
                const int bi = (row * g_inv) >> 16;           // row / G
                const int64_t orow = ((int64_t)b * B + i0 + bi) * p.n_q_heads + h * G + (row - bi * G);
                p.lse[orow] = (mstar + log2f(den)) * 0.6931471805599453f;
            }
        }
        if (tid == 0) HERALD_STAMP(7);
    }
    __syncthreads();
    if (S > 1 && tid < S - 1) {   // every partial row addressed to this CTA has landed: its senders may let go of their staging rows
        const uint32_t peer = tid < split ? tid : tid + 1;
        st_async_u32(map_to_cta(misc + kTcMiscReady + 4, peer), 1u, map_to_cta(bar(kBarAck), peer));
    }
    {
        // coalesced copy of this CTA's finished rows: one warp writes one 512-byte row per instruction
        const float* stage = reinterpret_cast<const float*>(sgen + kTcStageO);
        const int r_begin = split * rows_own, r_end = min(min(kTcBM, r_begin + rows_own), rows_valid);
        for (int rl = warp; rl < r_end - r_begin; rl += kTcThreads / 32) {
            const int r = r_begin + rl, bi = (r * g_inv) >> 16;   // r / G
            const int64_t orow = ((int64_t)b * B + i0 + bi) * p.n_q_heads + h * G + (r - bi * G);
            *reinterpret_cast<float4*>(p.out + orow * kHeadDim + lane * 4) = *reinterpret_cast<const float4*>(stage + r * kTcRowFloats + lane * 4);
        }
    }
    // a CTA may not exit while a peer can still arrive on its barriers: every peer has announced its receive buffer by now
    // (the partial rows addressed to this CTA have landed: the merge waited for them)
    if (S > 1 && tid == 0) { mbar_wait_cluster(bar(kBarPeerReady), 0); mbar_wait_cluster(bar(kBarAck), 0); }
    if (tid == 0) { HERALD_STAMP(4); HERALD_GSTAMP(63); }

    // ---- teardown ----
    if (warp == kTcMmaWarp) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(kTcTmemCols));
    }
}

// Longest-pool-first order of the units for a ragged batch: order[rank] = unit, rank by (pool_len descending, unit ascending).
// One block; O(units^2 / threads) comparisons, units is a few hundred.
__global__ void __launch_bounds__(1024) attn_plan_kernel(const int32_t* __restrict__ pool_len, int cap, int units, int32_t* __restrict__ order) {
    for (int i = threadIdx.x; i < units; i += blockDim.x) {
        const int li = max(0, min(pool_len[i], cap));
        int rank = 0;
        for (int j = 0; j < units; ++j) {
            const int lj = max(0, min(pool_len[j], cap));
            rank += (lj > li) || (lj == li && j < i);
        }
        order[rank] = i;
    }
}

}  // namespace herald
