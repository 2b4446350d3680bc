/* herald.h -- C ABI of the B200-native HERALD per-block sparse-KV hot path.
 *
 * HERALD (arxiv/paper_2606_21633; text in PAPER.md) serves block-diffusion LLMs with a
 * sparse KV cache: once per block a single *representative query* scores the whole
 * prefix KV cache and a per-KV-head top-k picks the critical entries (PAPER.md:141-163
 * section IV-A2; section IV-B4), the selected K/V rows are gathered into
 * the idle one of two sparse KV pools (section IV-B1), and
 * the block's T-1 denoising steps attend over the active pool plus the block's own
 * bidirectional KV (section II-A).  Selection for block n+1 overlaps with the
 * denoising of block n on a second stream; the pools are swapped at the block boundary
 * (Fig. 11).  The paper runs selection/gather on the CPU;
 * here every stage is a CUDA kernel for sm_100a.
 *
 * Conventions
 *   - every entry point returns 0 (HERALD_OK) or a negative HERALD_ERR_* code; nothing
 *     throws or aborts; herald_last_error() returns a thread-local message.
 *   - the CALLER owns every buffer (caches, pools, indices, outputs, workspaces).  The
 *     library allocates nothing, frees nothing and never synchronises with the host;
 *     all work is enqueued on the stream(s) passed in and is CUDA-graph capturable
 *     (pools are "allocated at initialization and reused across blocks").
 *     Two exceptions, both host-side helpers: herald_pipeline_tune (a calibration that times block steps) and
 *     herald_pipeline_step_host (eager only: it orders itself after the previous call's download with an event).
 *   - one-time per-device setup (shared-memory opt-in, SM count) is kept per device ordinal; a host thread uses the
 *     device that is current when it calls.  batch * n_kv_heads must not exceed 65535.
 *   - pointers are DEVICE pointers unless the comment says "host"; all device pointers
 *     must be 16-byte aligned.  bf16 = IEEE bfloat16 bit patterns (uint16).
 *   - head_dim must be 128, page_size 16, G = n_q_heads / n_kv_heads an integer <= 8;
 *     anything else returns HERALD_ERR_UNSUPPORTED.
 *   - query head hq belongs to KV head hq / G (contiguous groups).
 *   - device-side integers (seq_lens, page_table, k_per_seq, pool_len) are trusted; they
 *     are never read back by the host.  Kernels clamp k to min(k, seq_len, pool_capacity).
 */
#ifndef HERALD_H
#define HERALD_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define HERALD_OK 0
#define HERALD_ERR_INVALID_ARG (-1)
#define HERALD_ERR_UNSUPPORTED (-2)
#define HERALD_ERR_WORKSPACE_TOO_SMALL (-3)
#define HERALD_ERR_CUDA (-4)

/* GQA aggregation of the G per-head scores of one cached position (reading 1). */
#define HERALD_AGG_MAX_LOGIT 0   /* a[t] = max_g s[g,t]                      (BASELINE.json north_star) */
#define HERALD_AGG_SOFTMAX_SUM 1 /* a[t] = sum_g exp(s[g,t]-m_g)/l_g             */

typedef void* herald_stream_t; /* a cudaStream_t  */
typedef void* herald_event_t;  /* a cudaEvent_t   */

/* Problem shape, host POD.  Notation follows PAPER.md:201: S = seq_len prefix entries, k the
 * per-KV-head budget, G query heads per KV head; B = block_size. */
typedef struct herald_shape {
    int32_t batch;             /* sequences                                                         */
    int32_t n_q_heads;         /* H_q                                                               */
    int32_t n_kv_heads;        /* H_kv                                                              */
    int32_t head_dim;          /* d, must be 128                                                    */
    int32_t page_size;         /* tokens per KV page, must be 16                                    */
    int32_t block_size;        /* B, tokens per diffusion block (1..64)                             */
    int32_t max_seq_len;       /* bound on seq_lens[]; row stride of the score plane; multiple of 16 */
    int32_t max_pages_per_seq; /* row stride of page_table                                          */
    int32_t pool_capacity;     /* rows per (sequence, KV head) in one pool buffer; stride of sel_idx */
    int32_t agg_mode;          /* HERALD_AGG_*                                                      */
    float sm_scale;            /* logit scale, d^-1/2 (reading 2)                         */
} herald_shape_t;

/* Paged full KV cache ("full KV pool"; paged).  Token t of sequence b
 * is slot t % page_size of physical page page_table[b][t / page_size].  Element (page p, slot s,
 * KV head h, channel c) is at  p*page_stride + s*token_stride + h*head_stride + c  (bf16 elements);
 * the 128 channels of a row are contiguous and every stride is a multiple of 8 elements.
 * The canonical layout [n_pages][16][H_kv][128] has strides (16*H_kv*128, H_kv*128, 128).
 * Slots past seq_lens[b] in the last page and page_table entries past the last page are never read. */
typedef struct herald_cache {
    const void* k_pages;
    const void* v_pages;
    int64_t page_stride, token_stride, head_stride;
    const int32_t* page_table; /* [batch][max_pages_per_seq] */
    const int32_t* seq_lens;   /* [batch]                    */
} herald_cache_t;

/* Launch-geometry overrides (tests, sweeps, profiling).  Every field 0 = the library chooses, which is what every
 * BASELINE number uses.  The library reads no environment variable; this struct is the only knob.  The values are copied
 * and apply to the following calls of the CALLING THREAD (workspace-size queries included); NULL restores the defaults.
 * Results do not depend on any of them (tests/test_gpu_parity.py runs the parity cases under forced geometries). */
#define HERALD_XQ_AUTO 0
#define HERALD_XQ_MMA_SYNC 1
#define HERALD_XQ_TCGEN05 2
#define HERALD_ATTN_AUTO 0
#define HERALD_ATTN_EXACT 1
#define HERALD_ATTN_FAST_FIRST 2
typedef struct herald_tuning {
    int32_t attn_splits;     /* KV splits (= cluster size) of the attention grid, 1..8                                   */
    int32_t attn_m_tiles;    /* M tiles per (sequence, KV head); only values above the minimum ceil(B*G/128) are honoured */
    int32_t attn_total_ctas; /* the attention grid is split over the keys until it reaches this many blocks (default: SMs) */
    int32_t attn_no_pdl;     /* non-zero: attention kernels are launched without programmatic stream serialization          */
    int32_t scan_ctas;       /* grid of every score scan (overrides herald_pipeline_t.scan_ctas)                          */
    int32_t scan_head_major; /* non-zero: the head-major scan even where the page-major one applies                       */
    int32_t xq_path;         /* herald_select_xq: HERALD_XQ_AUTO / _MMA_SYNC / _TCGEN05                                    */
    int32_t attn_precision;  /* HERALD_ATTN_AUTO: attention blocks with a long share of the keys try the single-bf16 pass first
                                (verified against the finished row statistics, redone exactly if they fail);
                                _EXACT: bf16 hi+lo weights everywhere; _FAST_FIRST: every block tries the fast pass first       */
} herald_tuning_t;
int herald_set_tuning(const herald_tuning_t* tuning);

/* Message for the last error returned on this thread ("" if none).  Host only. */
const char* herald_last_error(void);

/* Budget rows k = min(L, ceil(L * permille / 1000)) in integer arithmetic (reading 5;
 * BASELINE.json: 5 % of 4096 -> 205, of 32768 -> 1639).  Host only; returns -1 on bad arguments. */
int32_t herald_budget_rows(int32_t seq_len, int32_t permille);

/* Workspace sizes in bytes for herald_select / herald_sparse_attn with this shape.  Host only;
 * return 0 on an invalid shape.  (SURVEY.md section 8(b) lists one herald_workspace_bytes: it is two queries because the
 * two stages run concurrently on the two streams of the pipeline and therefore need two distinct workspaces; the NEXT
 * entries have their own herald_*_workspace_bytes beside them.) */
size_t herald_select_workspace_bytes(const herald_shape_t* shape);
size_t herald_attn_workspace_bytes(const herald_shape_t* shape);

/* Number of thread blocks (one per SM) herald_sparse_attn launches for this shape: KV splits x M tiles x
 * batch x n_kv_heads.  A caller that overlaps selection with denoising gives the retrieval
 * stream the SMs this leaves free (herald_pipeline_t.scan_ctas).  Host only; 0 on an invalid shape. */
int32_t herald_attn_grid_ctas(const herald_shape_t* shape);

/* Representative-query selection (Eq.(1)).
 * For every sequence b and KV head h:
 *   s[g,t]  = sm_scale * q_rep[b, h*G+g, :] . K[b, t, h, :]      for all t < seq_lens[b]   (fp32 accumulate)
 *   a[t]    = aggregate_g s[g,t]                                 (shape->agg_mode)
 *   sel     = the k = min(k_per_seq[b], seq_lens[b], pool_capacity) positions of largest a[t];
 *             ties -> lower position; written in ASCENDING position order.
 *   q_rep      bf16 [batch][H_q][128]
 *   k_per_seq  int32 [batch]
 *   sel_idx    int32 [batch][H_kv][pool_capacity]  (entries past sel_cnt are left untouched)
 *   sel_cnt    int32 [batch][H_kv]
 *   scores_out optional fp32 [batch][H_kv][max_seq_len]: receives a[t] for t < seq_lens[b]; if NULL
 *              the plane lives in the workspace.
 *   ws         >= herald_select_workspace_bytes(shape) bytes, 256-byte aligned.
 * Errors: INVALID_ARG (null / misaligned pointer, bad shape), UNSUPPORTED, WORKSPACE_TOO_SMALL, CUDA. */
int herald_select(const herald_shape_t* shape, const herald_cache_t* cache, const void* q_rep,
                  const int32_t* k_per_seq, int32_t* sel_idx, int32_t* sel_cnt, float* scores_out,
                  void* ws, size_t ws_bytes, herald_stream_t stream);

/* herald_select for callers that may not allocate device memory (code under CUDA-graph capture, serving loops, harnesses
 * that forbid cudaMalloc): the same selection, with the workspace -- level-1 histograms and the score plane -- in a
 * file-scope __device__ array of HERALD_SELECT_STATIC_BYTES inside the library instead of a caller's buffer.  The library
 * allocates nothing here either: every GPU that loads it holds the array until the process exits.
 *   Arguments, output layout and errors are herald_select's, without scores_out / ws / ws_bytes.
 *   Limit: herald_select_workspace_bytes(shape) <= HERALD_SELECT_STATIC_BYTES (mode 0: about batch * H_kv * (max_seq_len + 4096)
 *   * 4 bytes -- BASELINE C1, C2 and C3 fit, C4 and C5 do not); a larger shape returns HERALD_ERR_WORKSPACE_TOO_SMALL and
 *   enqueues nothing.
 *   Every call on a device shares the one array, which keeps the previous call's contents (the call clears the histograms
 *   itself).  Two herald_select_static calls that overlap on the GPU (different streams, or graphs replayed side by side)
 *   race on it: keep them on one stream.  Calls that bring their own workspace (herald_select, herald_pipeline_step) do
 *   not touch the array and may run beside it. */
#define HERALD_SELECT_STATIC_BYTES (16u << 20)
size_t herald_select_static_max_bytes(void);      /* host-only: HERALD_SELECT_STATIC_BYTES */
int herald_select_static(const herald_shape_t* shape, const herald_cache_t* cache, const void* q_rep,
                         const int32_t* k_per_seq, int32_t* sel_idx, int32_t* sel_cnt, herald_stream_t stream);

/* Selection scored by x queries per sequence instead of one (PAPER.md:137 Fig. 8, :143, :161: the selection kernel as
 * the query count goes from B = 32 down to 1).  The paper does not say how the x
 * queries' scores combine into one ranking (reading 25): this entry takes the maximum,
 *   a[t] = sm_scale * max over j < x, g < G of  q_x[b, j, h*G+g, :] . K[b, t, h, :]
 * i.e. herald_select's max-logit aggregation over all x*G score rows; x = 1 is herald_select with agg_mode 0.  K is
 * read once whatever x is; FLOPs grow with x.
 *   q_x   bf16 [batch][x][H_q][128], device;  1 <= x, x*G <= 256;  shape->agg_mode must be HERALD_AGG_MAX_LOGIT.
 * Every other argument, the output layout, the workspace size and the error behaviour are herald_select's. */
int herald_select_xq(const herald_shape_t* shape, const herald_cache_t* cache, const void* q_x, int32_t x,
                     const int32_t* k_per_seq, int32_t* sel_idx, int32_t* sel_cnt, float* scores_out,
                     void* ws, size_t ws_bytes, herald_stream_t stream);

/* Gather of the selected entries into a sparse KV pool (pools PAPER.md:175):
 *   pool_k[b][h][j][:] = K[b, sel_idx[b][h][j], h, :]   for j < sel_cnt[b][h]   (bit copies; same for V)
 *   pool_k, pool_v  bf16 [batch][H_kv][pool_capacity][128] -- the IDLE buffer; rows j >= sel_cnt untouched. */
int herald_gather(const herald_shape_t* shape, const herald_cache_t* cache, const int32_t* sel_idx,
                  const int32_t* sel_cnt, void* pool_k, void* pool_v, herald_stream_t stream);

/* One denoising step's attention over critical KV + in-block KV:
 *   out[b][i][hq][:] = softmax_j( sm_scale * q_blk[b][i][hq][:] . K'_j ) . V'_j ,   h = hq / G,
 *   K' = pool_k[b][h][0 .. pool_len[b][h]) followed by k_blk[b][0..B)[h]  (no mask; V' likewise).
 *   pool_k/pool_v bf16 [batch][H_kv][pool_capacity][128] (the ACTIVE buffer); pool_len int32 [batch][H_kv]
 *   q_blk bf16 [batch][B][H_q][128]; k_blk, v_blk bf16 [batch][B][H_kv][128]
 *   out fp32 [batch][B][H_q][128]; lse optional fp32 [batch][B][H_q] = log sum_j exp(logit_j).
 *   ws >= herald_attn_workspace_bytes(shape), 256-byte aligned.  bf16 tensor-core products, fp32 softmax and accumulation.
 *   The softmax weights enter the PV product as a bf16 pair hi + lo (2^-17 relative).  A thread block whose share of the
 *   keys is long (>= 1536) first tries a single bf16 per weight, accepts the result only if every one of its rows has
 *   sum_i p_i^2 <= 1/64 on the FINISHED row (then the rounding moves an output by ~1e-4 |v|), and otherwise redoes its tiles
 *   exactly.  The workspace keeps one note per block from launch to launch ("failed: start exact");
 *   its content never changes a result, so it needs no initialisation. */
int herald_sparse_attn(const herald_shape_t* shape, const void* pool_k, const void* pool_v,
                       const int32_t* pool_len, const void* q_blk, const void* k_blk, const void* v_blk,
                       float* out, float* lse, void* ws, size_t ws_bytes, herald_stream_t stream);

/* The same attention for n_groups query groups that share the prefix (the step after the draft is formed
 * runs "as a 2B-token forward pass ... the denoising group and the draft group use different custom attention masks: both
 * groups attend to the KV cache of the completed prefix but not to each other"): ONE launch in which group g, sequence b
 * attends over the pools of sequence b and over its OWN in-block rows,
 *   out[g][b][i][hq][:] = softmax_j( sm_scale * q_blk[g][b][i][hq][:] . K'_j ) . V'_j,
 *   K' = pool_k[b][h][0 .. pool_len[b][h]) followed by k_blk[g][b][0..B)[h].
 *   q_blk bf16 [n_groups][batch][B][H_q][128]; k_blk, v_blk bf16 [n_groups][batch][B][H_kv][128]
 *   out fp32 [n_groups][batch][B][H_q][128]; lse optional fp32 [n_groups][batch][B][H_q]; pools and pool_len as above.
 *   ws >= n_groups * herald_attn_workspace_bytes(shape), 256-byte aligned.  n_groups = 1 is herald_sparse_attn. */
int herald_sparse_attn_groups(const herald_shape_t* shape, int32_t n_groups, const void* pool_k, const void* pool_v,
                              const int32_t* pool_len, const void* q_blk, const void* k_blk, const void* v_blk,
                              float* out, float* lse, void* ws, size_t ws_bytes, herald_stream_t stream);

/* Dense attention of the block queries over the FULL paged cache + in-block KV, for layers that keep their whole KV
 * ("the first two layers ... retain the full KV cache"; = herald_sparse_attn at a 100 % budget without
 * the gather):
 *   out[b][i][hq][:] = softmax_j( sm_scale * q_blk[b][i][hq][:] . K'_j ) . V'_j ,   h = hq / G,
 *   K' = K[b, 0 .. seq_lens[b]), h, :] read through the page table, followed by k_blk[b][0..B)[h]  (no mask).
 * Same tensor-core kernel; the key tiles are TMA boxes of the cache pages themselves.  Arguments as herald_sparse_attn;
 * ws >= herald_attn_workspace_bytes(shape). */
int herald_dense_attn(const herald_shape_t* shape, const herald_cache_t* cache, const void* q_blk, const void* k_blk,
                      const void* v_blk, float* out, float* lse, void* ws, size_t ws_bytes, herald_stream_t stream);

/* Attention output of the representative query itself (the fused selection kernel keeps the
 * FlashAttention statistics (m_g, l_g, o_g); o_g returns to the layer's FFN):
 *   out[b][hq][:] = softmax_t( sm_scale * q_rep[b][hq][:] . K[b,t,h,:] ) . V[b,t,h,:]  over all t < seq_lens[b], h = hq / G
 *   q_rep bf16 [batch][H_q][128]; out fp32 [batch][H_q][128]; lse optional fp32 [batch][H_q] (= log sum_t exp(logit_t)).
 *   A sequence without cached tokens gives zeros (lse = -inf).  ws >= herald_rep_attn_workspace_bytes(shape), 256-byte aligned.
 * A second HBM stream over K and V (512 B per token and KV head); fp32 accumulation. */
size_t herald_rep_attn_workspace_bytes(const herald_shape_t* shape);
int herald_rep_attn(const herald_shape_t* shape, const herald_cache_t* cache, const void* q_rep, float* out, float* lse,
                    void* ws, size_t ws_bytes, herald_stream_t stream);

/* The fused retrieval kernel (section IV-B4: the selection kernel "maintains the FlashAttention
 * statistics (m_g, l_g, o_g)" next to the raw scores): ONE pass over K and V gives both what herald_select gives
 * (scores, sel_idx, sel_cnt, either aggregation) and what herald_rep_attn gives (rep_out [batch][H_q][128] fp32,
 * optional rep_lse [batch][H_q]).  K is read once instead of twice.  With HERALD_AGG_SOFTMAX_SUM the pass keeps the
 * per-head logits in the workspace and one more kernel, after the statistics are final, forms sum_g exp(s - lse_g).  Arguments as in those two entries; ws >= herald_select_rep_workspace_bytes(shape), 256-byte aligned. */
size_t herald_select_rep_workspace_bytes(const herald_shape_t* shape);
int herald_select_rep(const herald_shape_t* shape, const herald_cache_t* cache, const void* q_rep, const int32_t* k_per_seq,
                      int32_t* sel_idx, int32_t* sel_cnt, float* scores_out, float* rep_out, float* rep_lse,
                      void* ws, size_t ws_bytes, herald_stream_t stream);

/* Block-boundary cache operations.
 * herald_cache_write_block: K[b, write_pos[b] + i, h, :] = k_new[b][i][h][:] for i < block_size (same for V), through
 *   the page table -- appends the rows of a block (the draft KV, "appended temporarily" to the full KV pool,
 *   PAPER.md:189) or replaces rows already there (the true KV "replacing the draft").  The pages must be
 *   mapped; seq_lens is the caller's to advance.  write_pos int32 [batch] (device); k_new / v_new bf16
 *   [batch][B][H_kv][128].  Bit copies.  The cache pages are written: pass them non-const in `cache`.
 * herald_pool_append_block: pool[b][h][pool_len[b][h] + i][:] = k_new[b][i][h][:], then pool_len[b][h] += B (clamped to
 *   pool_capacity): the completed block joins block n+1's pool (reading 10). */
int herald_cache_write_block(const herald_shape_t* shape, const herald_cache_t* cache, const int32_t* write_pos,
                             const void* k_new, const void* v_new, herald_stream_t stream);
int herald_pool_append_block(const herald_shape_t* shape, void* pool_k, void* pool_v, int32_t* pool_len,
                             const void* k_new, const void* v_new, herald_stream_t stream);

/* Per-layer state of the dual-stream block step.  Host POD holding device pointers. */
typedef struct herald_layer {
    herald_cache_t cache;      /* this layer's full KV pool                                                   */
    const void* q_rep;         /* bf16 [batch][H_q][128]: representative query of the NEXT block              */
    const int32_t* k_per_seq;  /* int32 [batch]                                                               */
    const void* q_blk;         /* bf16 [n_steps][batch][B][H_q][128]: denoise step s reads slice s            */
    const void* k_blk;         /* bf16 [n_steps][batch][B][H_kv][128]                                         */
    const void* v_blk;         /* bf16 [n_steps][batch][B][H_kv][128]                                         */
    float* out;                /* fp32 [n_steps][batch][B][H_q][128]                                          */
    void* pool_k[2];           /* double-buffered sparse KV pools, each [batch][H_kv][cap][128] */
    void* pool_v[2];
    int32_t* pool_len[2];      /* int32 [batch][H_kv] per buffer                                              */
    int32_t dense;             /* non-zero: the layer keeps its full KV and attends over the cache itself (PAPER.md:181:
                                  "the first two layers always perform exact attention"): no selection, no gather,
                                  q_rep / k_per_seq / pool_* unused (may be NULL)                               */
} herald_layer_t;

/* One block step of the dual-stream pipeline (Fig. 11):
 *   main stream     : for s in [0, n_steps): for each layer: herald_sparse_attn on pools[active]
 *                     (herald_dense_attn on the cache for a layer with `dense` set; the retrieval stream skips it)
 *   retrieval stream: starts once `start_after_step` main-stream steps have been enqueued-and-finished
 *                     (0 = immediately, the north-star default; 2 = the paper's "waits only for the
 *                     first two steps"); for each layer: herald_select -> herald_gather into
 *                     pools[1-active], sel_cnt written to pool_len[1-active]
 *   join            : main stream waits for the retrieval stream; `active` is flipped (pool swap).
 * No host synchronisation.  `layers` is a host array.  Events are caller-created cudaEvent_t. */
typedef struct herald_pipeline {
    herald_shape_t shape;
    int32_t n_layers;
    int32_t n_steps;          /* T-1 attention steps per block (reading 13) */
    int32_t start_after_step; /* 0 .. n_steps                                           */
    int32_t active;           /* index of the ACTIVE pool buffer; flipped on success    */
    int32_t scan_ctas;        /* grid of the retrieval stream's score scan (1024-thread blocks, one per SM; each takes
                                 1/scan_ctas of the cache); 0 = the SMs the attention grid leaves free, at least an eighth of the
                                 device (herald_pipeline_tune measures the alternatives).  The scan is a long
                                 bandwidth-bound kernel and the attention blocks need whole SMs:
                                   <= the SMs the attention grid leaves free: the scan streams K beside the denoising
                                      steps without ever taking their SMs (denoising-bound shapes);
                                   a multiple of the SM count: short blocks in several waves, time-sliced with the
                                      attention launches (selection-bound shapes; "bound by the slower
                                      stream", Fig. 14)                                              */
    int32_t scan_head_permille; /* 0..1000: that many thousandths of the (first sparse layer's) score scan run with one block per
                                 SM BEFORE the main stream's next denoising step starts (the main stream waits for them), the rest
                                 with scan_ctas blocks beside the steps.  The retrieval stream needs a fixed amount of SM time
                                 (an SM draws ~100 GB/s from L2/HBM with the scan's access pattern); when the SMs the attention grid leaves free cannot deliver it
                                 inside the denoising window, a head start costs less than a retrieval stream that outlasts the
                                 window.  0 = everything beside the steps (max-logit aggregation only;
                                 ignored with HERALD_AGG_SOFTMAX_SUM) */
    herald_layer_t* layers;   /* host array [n_layers]                                  */
    int32_t* sel_idx;         /* int32 [batch][H_kv][pool_capacity] scratch (retrieval stream) */
    void* ws_select;
    size_t ws_select_bytes;
    void* ws_attn;            /* >= herald_attn_workspace_bytes(); with n_layers times that, a multi-wave attention grid over   */
    size_t ws_attn_bytes;     /* ragged pools is dispatched longest pool first (one slice per layer holds the unit order)      */
    herald_stream_t main_stream;
    herald_stream_t retrieval_stream;
    herald_event_t ev_fork; /* recorded on the main stream, waited on by the retrieval stream */
    herald_event_t ev_join; /* recorded on the retrieval stream, waited on by the main stream */
} herald_pipeline_t;

int herald_pipeline_step(herald_pipeline_t* pipe);

/* Calibration of the schedule of a pipeline (how the retrieval stream shares the device with the denoising steps): runs
 * block steps -- each a complete, valid step, so the pools stay consistent -- for a handful of
 * (scan_ctas, start_after_step, scan_head_permille) candidates: two eager warm-up steps, then the step captured into a CUDA
 * graph and replayed `reps` times between two CUDA events on the main stream (eager steps if the capture fails), and leaves
 * the fastest candidate in *pipe.  This is the ONE entry of the library that creates (and destroys) events and graphs and
 * synchronises with the host; call it once outside any timed region or graph
 * capture.  table (optional, host): receives up to table_cap measured candidates, *n_table how many.  Host only. */
typedef struct herald_schedule {
    int32_t scan_ctas, start_after_step, scan_head_permille;
    float ms_per_step;
} herald_schedule_t;
int herald_pipeline_tune(herald_pipeline_t* pipe, int32_t reps, herald_schedule_t* table, int32_t table_cap, int32_t* n_table);

/* Optional timing hooks for the retrieval stream (measurement only, no effect on results): caller-created
 * events recorded on the retrieval stream around the stages of the LAST layer's selection inside
 * herald_pipeline_step; a plain herald_select records scan_begin / scan_end / topk_end on its own stream as well
 * (this is how bench.py times the scan kernel by itself).  Any member may be NULL.  scan = score scan (+ aggregation in mode 1),
 * topk = radix select, gather = pool fill.  Pass NULL to herald_pipeline_set_profile to switch off. */
typedef struct herald_profile {
    herald_event_t scan_begin, scan_end, topk_end, gather_end;
} herald_profile_t;

/* Stores `prof` (host pointer, must outlive the following pipeline steps) for this thread.  Host only. */
int herald_pipeline_set_profile(const herald_profile_t* prof);

/* Test hook (no effect on results): the following herald_pipeline_step calls of this thread put a kernel that idles for
 * `main_us` microseconds on the main stream right after the retrieval stream has been forked, and one that idles for
 * `retrieval_us` at the head of the retrieval stream's work.  PAPER.md:191: the schedule "affects only the selection and never
 * the generated output": the pools swap only at the block boundary -- so outputs and pools must not depend
 * on either delay (tests/test_gpu_full_size.py).  0, 0 switches the hook off; at most 1 s each.  Host only. */
int herald_pipeline_set_debug_delay(uint32_t main_us, uint32_t retrieval_us);

/* Host-buffer variant used for end-to-end timing: per block, the step's inputs come from (pinned)
 * HOST memory and its outputs return to HOST memory, all asynchronously on the pipeline's streams:
 *   H2D  host_q_rep[l] -> layers[l].q_rep ; host_q_blk/k_blk/v_blk[l] -> layers[l].q_blk/k_blk/v_blk
 *   herald_pipeline_step
 *   D2H  layers[l].out -> host_out[l]
 * Each host_* is a host array of n_layers host pointers with the same extents as the device tensors.
 * The KV cache stays resident in HBM (it is the state, not a per-step input).  Uploads run on the main stream and
 * downloads on the retrieval stream, so that the upload of a block overlaps the download of the previous one; the next
 * call orders its attention after the download that last read its output buffer by itself (see dev_out_alt).  The caller synchronises BOTH streams before reading
 * host_out (or before touching the host input buffers again) -- and copy_stream / upload_stream if given. */
typedef struct herald_host_io {
    const void* const* host_q_rep;
    const void* const* host_q_blk;
    const void* const* host_k_blk;
    const void* const* host_v_blk;
    void* const* host_out;
    /* optional double buffering of the device outputs: dev_out_alt[l] is a second fp32 [n_steps][batch][B][H_q][128] device buffer per
     * layer.  Blocks then alternate between layers[l].out and dev_out_alt[l] (by pipe->active), so that the attention of a block
     * runs beside the download of the previous block instead of behind it; ev_download[2] are caller-created events the library
     * records after each download.  NULL = single buffering (the attention waits for the previous download). */
    void* const* dev_out_alt;
    herald_event_t ev_download[2];
    herald_stream_t copy_stream; /* optional third stream for the downloads; NULL = the retrieval stream (the next block's selection
                                    then queues behind the download of this block) */
    /* optional double buffering of the device INPUTS: dev_*_alt[l] are second device buffers with the extents of layers[l].q_rep /
     * q_blk / k_blk / v_blk (dev_q_rep_alt[l] may be NULL for a dense layer).  Blocks alternate between the two sets; the uploads of
     * a block then run on upload_stream beside the previous block's attention instead of in front of their own.  ev_upload[2]
     * (recorded on upload_stream after a block's uploads) and ev_compute[2] (recorded on the main stream after a block step: its
     * input set may be overwritten) are caller-created.  dev_q_blk_alt == NULL = single buffering, uploads on the main stream. */
    void* const* dev_q_rep_alt;
    void* const* dev_q_blk_alt;
    void* const* dev_k_blk_alt;
    void* const* dev_v_blk_alt;
    herald_stream_t upload_stream;
    herald_event_t ev_upload[2];
    herald_event_t ev_compute[2];
} herald_host_io_t;

/* host_q_rep[l] may be NULL for a layer with `dense` set.  Every pointer is validated before anything is enqueued.
 * Not capturable into a CUDA graph (see Conventions). */
int herald_pipeline_step_host(herald_pipeline_t* pipe, const herald_host_io_t* io);

#ifdef HERALD_ATTN_TRACE
/* Debug builds only (-DHERALD_ATTN_TRACE; not part of the release ABI): the attention kernel writes clock64 / globaltimer
 * stamps of its phases to dev_buf ([blocks of the grid][64] uint64, device memory) on every following launch; NULL stops. */
int herald_debug_set_attn_trace(void* dev_buf);
#endif

#ifdef __cplusplus
}
#endif
#endif /* HERALD_H */
