// Host side of the C ABI declared in include/herald.h: argument checks, workspace carving,
// launches, and the dual-stream block step.  No allocation, no host synchronisation.
#include "../../include/herald.h"

#include <cstdarg>
#include <cstdio>
#include <cstring>

#include "attn_tc.cuh"
#include <functional>
#include "common.cuh"
#include "cache_ops.cuh"
#include "gather.cuh"
#include "rep_attn.cuh"
#include "scan_xq.cuh"
#include "scan_xq_tc.cuh"
#include "scan.cuh"
#include "topk.cuh"

namespace herald {

static thread_local char g_err[512] = "";
static thread_local const herald_profile_t* g_prof = nullptr;   // timing hooks (herald_pipeline_set_profile)
static thread_local bool g_prof_armed = false;                    // inside a pipeline step: only the last sparse layer is timed
static thread_local bool g_in_pipeline = false;
static thread_local uint32_t g_delay_main_us = 0, g_delay_retrieval_us = 0;   // test hook (herald_pipeline_set_debug_delay)
#ifdef HERALD_ATTN_TRACE
static unsigned long long* g_attn_trace = nullptr;               // debug builds only: device buffer [CTAs][64]
#endif                   // true only inside the last layer's retrieval

static int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

static int cuda_fail(cudaError_t e, const char* what) {
    return fail(HERALD_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// launch-geometry overrides of this thread (herald_set_tuning); all zero = automatic
static thread_local herald_tuning_t g_tune = {0, 0, 0, 0, 0, 0, 0, 0};

static int check_shape(const herald_shape_t* s) {
    if (!s) return fail(HERALD_ERR_INVALID_ARG, "shape is NULL");
    if (s->batch < 0 || s->n_q_heads <= 0 || s->n_kv_heads <= 0 || s->block_size <= 0 || s->max_seq_len < 0 ||
        s->max_pages_per_seq < 0 || s->pool_capacity < 0)
        return fail(HERALD_ERR_INVALID_ARG, "negative or zero extent in shape");
    if (s->head_dim != kHeadDim) return fail(HERALD_ERR_UNSUPPORTED, "head_dim must be 128 (got %d)", s->head_dim);
    if (s->page_size != kPageSize) return fail(HERALD_ERR_UNSUPPORTED, "page_size must be 16 (got %d)", s->page_size);
    if (s->n_q_heads % s->n_kv_heads) return fail(HERALD_ERR_INVALID_ARG, "n_q_heads %% n_kv_heads != 0");
    if (s->n_q_heads / s->n_kv_heads > 8) return fail(HERALD_ERR_UNSUPPORTED, "G = n_q_heads/n_kv_heads must be <= 8");
    if (s->block_size > 64) return fail(HERALD_ERR_UNSUPPORTED, "block_size must be <= 64");
    if (s->max_seq_len % kPageSize) return fail(HERALD_ERR_INVALID_ARG, "max_seq_len must be a multiple of 16");
    if ((int64_t)s->max_pages_per_seq * kPageSize < s->max_seq_len)
        return fail(HERALD_ERR_INVALID_ARG, "max_pages_per_seq * 16 < max_seq_len");
    if (s->agg_mode != HERALD_AGG_MAX_LOGIT && s->agg_mode != HERALD_AGG_SOFTMAX_SUM)
        return fail(HERALD_ERR_INVALID_ARG, "agg_mode must be 0 or 1");
    if (!(s->sm_scale > 0.f)) return fail(HERALD_ERR_INVALID_ARG, "sm_scale must be > 0");
    if ((int64_t)s->batch * s->n_kv_heads > 65535)
        return fail(HERALD_ERR_UNSUPPORTED, "batch * n_kv_heads = %lld exceeds 65535 (a grid dimension of the gather and attention kernels)",
                    (long long)s->batch * s->n_kv_heads);
    return HERALD_OK;
}

static int check_cache(const herald_cache_t* c, bool need_v) {
    if (!c) return fail(HERALD_ERR_INVALID_ARG, "cache is NULL");
    if (!c->k_pages || (need_v && !c->v_pages) || !c->page_table || !c->seq_lens)
        return fail(HERALD_ERR_INVALID_ARG, "cache has a NULL pointer");
    if (!aligned16(c->k_pages) || (need_v && !aligned16(c->v_pages)))
        return fail(HERALD_ERR_INVALID_ARG, "cache pages must be 16-byte aligned");
    if (c->page_stride % 8 || c->token_stride % 8 || c->head_stride % 8 || c->head_stride < kHeadDim)
        return fail(HERALD_ERR_INVALID_ARG, "cache strides must be multiples of 8 elements, head_stride >= 128");
    return HERALD_OK;
}

// Test hook: one thread that sleeps until the global timer has advanced by `ns` (an artificial delay on a stream).
__global__ void delay_kernel(unsigned long long ns) {
    unsigned long long t0, t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    do {
        __nanosleep(1000);
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    } while (t - t0 < ns);
}

// ---- select workspace layout ------------------------------------------------------------------
struct SelectWs {
    size_t hist1, scores, raw, stats, total;
    int scan_ctas;
};

// One-time setup is per DEVICE (cudaFuncSetAttribute applies to the current device; so does the SM count): small tables
// indexed by the device ordinal.  Races between host threads are benign (the same values are written twice).
constexpr int kMaxDevices = 64;
static int current_device() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) dev = 0;
    return dev;
}
static int sm_count() {
    static int n[kMaxDevices] = {0};
    const int dev = current_device();
    if (n[dev] == 0) {
        int v = 0;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v <= 0) v = 148;   // B200
        n[dev] = v;
    }
    return n[dev];
}
// opt a kernel into `bytes` of dynamic shared memory once per device; `done` is that kernel's table
template <typename Kernel>
static cudaError_t ensure_smem(Kernel kernel, int bytes, bool (&done)[kMaxDevices]) {
    const int dev = current_device();
    if (done[dev]) return cudaSuccess;
    const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) done[dev] = true;
    return e;
}

// grid of the score scan (0 = one block per SM); set by herald_pipeline_step around its select calls
static thread_local int g_scan_ctas = 0;

// Grid of the scan: one 1024-thread CTA per SM it may occupy, or several waves of them.
static int scan_ctas_for(const herald_shape_t* s) {
    (void)s;
    int n = g_tune.scan_ctas;
    if (n <= 0) n = g_scan_ctas > 0 ? g_scan_ctas : sm_count();
    if (n > kScanMaxCtas) n = kScanMaxCtas;
    return n;
}

static SelectWs select_ws_layout(const herald_shape_t* s) {
    SelectWs w{};
    const size_t units = (size_t)s->batch * s->n_kv_heads;
    const int G = s->n_q_heads / s->n_kv_heads;
    w.scan_ctas = scan_ctas_for(s);
    size_t off = 0;
    w.hist1 = off;
    off = align_up(off + units * kBins1 * sizeof(uint32_t), 256);
    w.scores = off;
    off = align_up(off + units * (size_t)s->max_seq_len * sizeof(float), 256);
    w.raw = off;
    w.stats = off;
    if (s->agg_mode == HERALD_AGG_SOFTMAX_SUM) {
        off = align_up(off + units * G * (size_t)s->max_seq_len * sizeof(float), 256);
        w.stats = off;
        off = align_up(off + units * G * (size_t)kScanMaxCtas * sizeof(float2), 256);   // any grid size fits
    }
    w.total = off;
    return w;
}

// ---- attention launch geometry ----------------------------------------------------------------
struct AttnGeom {
    int m_tiles, ipt, n_splits;
    size_t hint_off, total;
};

static AttnGeom attn_geom(const herald_shape_t* s, bool dense = false) {
    AttnGeom a{};
    const int G = s->n_q_heads / s->n_kv_heads;
    const int units = s->batch * s->n_kv_heads;
    // an M tile is `ipt` whole block rows x G heads (<= 128 rows), balanced over the tiles
    const int rows_cap = kTcBM / G;
    a.m_tiles = (s->block_size + rows_cap - 1) / rows_cap;
    const int forced_mt = g_tune.attn_m_tiles;
    if (forced_mt > a.m_tiles && forced_mt <= s->block_size) a.m_tiles = forced_mt;
    a.ipt = (s->block_size + a.m_tiles - 1) / a.m_tiles;
    // one CTA per SM: split the keys of a unit over a cluster until the grid covers the 148 SMs once
    const int max_keys = dense ? s->max_seq_len : s->pool_capacity;
    const int max_tiles = 1 + (max_keys + kTcBN - 1) / kTcBN;   // the in-block rows are a key tile of their own
    const int target = g_tune.attn_total_ctas > 0 ? g_tune.attn_total_ctas : sm_count();
    int splits = units > 0 ? target / (units * a.m_tiles) : 1;
    const int forced = g_tune.attn_splits;
    if (forced > 0) splits = forced;
    if (splits > max_tiles) splits = max_tiles;
    if (splits > kTcMaxSplits) splits = kTcMaxSplits;
    if (splits < 1) splits = 1;
    a.n_splits = splits;
    // split-KV partials are merged on chip (DSMEM); the workspace holds the longest-first unit order of a layer and one
    // precision note per block of the largest grid the shape can get (attn_tc.cuh, "precision modes")
    a.hint_off = align_up((size_t)(units > 0 ? units : 1) * sizeof(int32_t), 256);
    a.total = a.hint_off + align_up((size_t)(units > 0 ? units : 1) * 4 * kTcMaxSplits * sizeof(int32_t), 256);
    return a;
}

// ---- TMA tensor maps (driver entry point resolved at run time; libcuda is not linked) -------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* ptr = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(ptr);
    }
    return fn;
}

// Encoding a tensor map costs about a microsecond of host time and the same maps come back every denoising step
// (5 per launch, ~50 per layer and block), so encodings are kept per thread in a small hash table keyed by
// (base pointer, extents).  Callers copy the map out at once: a later insertion may evict any slot.
struct MapKey {
    const void* ptr;
    int32_t d[4];
    bool operator==(const MapKey& o) const { return ptr == o.ptr && d[0] == o.d[0] && d[1] == o.d[1] && d[2] == o.d[2] && d[3] == o.d[3]; }
};
struct MapSlot {
    MapKey key;
    CUtensorMap map;
    bool used;
};
constexpr int kMapSlots = 512;       // power of two; ~70 KB of thread-local storage per thread that launches attention
constexpr int kMapProbe = 8;
static thread_local MapSlot g_maps[kMapSlots];

static uint32_t map_hash(const MapKey& k) {
    uint64_t h = reinterpret_cast<uintptr_t>(k.ptr) * 0x9E3779B97F4A7C15ull;
    h ^= (uint64_t)(uint32_t)k.d[3] * 0xC2B2AE3D27D4EB4Full + (uint64_t)(uint32_t)k.d[0] * 31u + (uint32_t)k.d[1];
    return (uint32_t)(h >> 40) & (kMapSlots - 1);
}
static bool cached_map(const MapKey& key, CUtensorMap* out) {
    const uint32_t h = map_hash(key);
    for (int i = 0; i < kMapProbe; ++i) {
        const MapSlot& s = g_maps[(h + i) & (kMapSlots - 1)];
        if (s.used && s.key == key) {
            *out = s.map;
            return true;
        }
    }
    return false;
}
static void store_map(const MapKey& key, const CUtensorMap& map) {
    const uint32_t h = map_hash(key);
    MapSlot* s = &g_maps[h];                      // full neighbourhood: evict the home slot
    for (int i = 0; i < kMapProbe; ++i) {
        MapSlot* c = &g_maps[(h + i) & (kMapSlots - 1)];
        if (!c->used) {
            s = c;
            break;
        }
    }
    s->key = key;
    s->map = map;
    s->used = true;
}

// bf16 pool [units][cap][128] as a 3-D tensor (d, row, unit); box = 64 channels x 128 rows, 128-byte swizzle:
// the box lands in shared memory exactly in the UMMA canonical layout (K-major for K, MN-major for V).
static int make_pool_map(CUtensorMap* out, const void* pool, int units, int cap) {
    const MapKey key{pool, {units, cap, 0, 3}};
    if (cached_map(key, out)) return HERALD_OK;
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return fail(HERALD_ERR_CUDA, "cuTensorMapEncodeTiled is not available from the driver");
    CUtensorMap* map = out;
    const cuuint64_t rows = cap > 0 ? cap : 1;
    const cuuint64_t dims[3] = {(cuuint64_t)kHeadDim, rows, (cuuint64_t)units};
    const cuuint64_t strides[2] = {(cuuint64_t)kRowBytes, rows * kRowBytes};
    const cuuint32_t box[3] = {64u, (cuuint32_t)(rows < (cuuint64_t)kTcBN ? rows : kTcBN), 1u};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    const CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(pool), dims, strides, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(HERALD_ERR_CUDA, "cuTensorMapEncodeTiled(pool) failed with CUresult %d", (int)r);
    store_map(key, *map);
    return HERALD_OK;
}

// bf16 q_blk [batch][B][H_q][128] as a 4-D tensor (d, head, block row, sequence); box = 64 channels x G heads x ipt
// block rows: one box is one half of the Q tile of an (unit, M tile), rows ordered (block row, head), zero-filled past B.
// bf16 k_blk / v_blk [batch][B][H_kv][128] as a 4-D tensor (d, head, block row, sequence); box = 64 channels x 1 head x
// B block rows: one half of the in-block key tile of a unit.
static int make_blk_map(CUtensorMap* out, const void* blk, const herald_shape_t* s) {
    const MapKey key{blk, {s->batch, s->block_size, s->n_kv_heads, 5}};
    if (cached_map(key, out)) return HERALD_OK;
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return fail(HERALD_ERR_CUDA, "cuTensorMapEncodeTiled is not available from the driver");
    CUtensorMap* map = out;
    const cuuint64_t dims[4] = {(cuuint64_t)kHeadDim, (cuuint64_t)s->n_kv_heads, (cuuint64_t)s->block_size, (cuuint64_t)s->batch};
    const cuuint64_t strides[3] = {(cuuint64_t)kRowBytes, (cuuint64_t)s->n_kv_heads * kRowBytes,
                                   (cuuint64_t)s->block_size * s->n_kv_heads * kRowBytes};
    const cuuint32_t box[4] = {64u, 1u, (cuuint32_t)s->block_size, 1u};
    const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
    const CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(blk), dims, strides, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(HERALD_ERR_CUDA, "cuTensorMapEncodeTiled(k_blk/v_blk) failed with CUresult %d", (int)r);
    store_map(key, *map);
    return HERALD_OK;
}

// Paged bf16 cache [n_pages][16][H_kv][128] (any strides) as a 4-D tensor (d, head, slot, page); box = 64 channels x 1 head x
// 16 slots x 1 page: the 16 rows of one head of one page, one half.  The page extent is unknown to the ABI (page ids are
// trusted): the map is given 2^24 pages.
static int make_paged_map(CUtensorMap* out, const void* pages, const herald_cache_t* c, int n_kv_heads) {
    const MapKey key{pages, {(int32_t)c->page_stride, (int32_t)c->token_stride, (int32_t)c->head_stride, 6 | (n_kv_heads << 8)}};
    if (cached_map(key, out)) return HERALD_OK;
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return fail(HERALD_ERR_CUDA, "cuTensorMapEncodeTiled is not available from the driver");
    CUtensorMap* map = out;
    const cuuint64_t dims[4] = {(cuuint64_t)kHeadDim, (cuuint64_t)n_kv_heads, (cuuint64_t)kPageSize, (cuuint64_t)1 << 24};
    const cuuint64_t strides[3] = {(cuuint64_t)c->head_stride * 2, (cuuint64_t)c->token_stride * 2, (cuuint64_t)c->page_stride * 2};
    const cuuint32_t box[4] = {64u, 1u, (cuuint32_t)kPageSize, 1u};
    const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
    const CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(pages), dims, strides, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(HERALD_ERR_CUDA, "cuTensorMapEncodeTiled(paged cache) failed with CUresult %d", (int)r);
    store_map(key, *map);
    return HERALD_OK;
}

static int make_q_map(CUtensorMap* out, const void* q_blk, const herald_shape_t* s, int ipt) {
    const MapKey key{q_blk, {s->batch, s->block_size, s->n_q_heads, 4 | (ipt << 8) | (s->n_kv_heads << 16)}};
    if (cached_map(key, out)) return HERALD_OK;
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return fail(HERALD_ERR_CUDA, "cuTensorMapEncodeTiled is not available from the driver");
    CUtensorMap* map = out;
    const int G = s->n_q_heads / s->n_kv_heads;
    const cuuint64_t dims[4] = {(cuuint64_t)kHeadDim, (cuuint64_t)s->n_q_heads, (cuuint64_t)s->block_size, (cuuint64_t)s->batch};
    const cuuint64_t strides[3] = {(cuuint64_t)kRowBytes, (cuuint64_t)s->n_q_heads * kRowBytes,
                                   (cuuint64_t)s->block_size * s->n_q_heads * kRowBytes};
    const cuuint32_t box[4] = {64u, (cuuint32_t)G, (cuuint32_t)ipt, 1u};
    const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
    const CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(q_blk), dims, strides, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(HERALD_ERR_CUDA, "cuTensorMapEncodeTiled(q_blk) failed with CUresult %d", (int)r);
    store_map(key, *map);
    return HERALD_OK;
}

// q_x [batch][x][H_q][128]: box = (64 channels, G heads, x queries, 1 sequence): the x*G score rows of one KV head
static int make_qx_map(CUtensorMap* out, const void* q_x, const herald_shape_t* s, int x) {
    const MapKey key{q_x, {s->batch, x, s->n_q_heads, 7 | (s->n_kv_heads << 16)}};
    if (cached_map(key, out)) return HERALD_OK;
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return fail(HERALD_ERR_CUDA, "cuTensorMapEncodeTiled is not available from the driver");
    const int G = s->n_q_heads / s->n_kv_heads;
    const cuuint64_t dims[4] = {(cuuint64_t)kHeadDim, (cuuint64_t)s->n_q_heads, (cuuint64_t)x, (cuuint64_t)s->batch};
    const cuuint64_t strides[3] = {(cuuint64_t)kRowBytes, (cuuint64_t)s->n_q_heads * kRowBytes, (cuuint64_t)x * s->n_q_heads * kRowBytes};
    const cuuint32_t box[4] = {64u, (cuuint32_t)G, (cuuint32_t)x, 1u};
    const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
    const CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(q_x), dims, strides, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(HERALD_ERR_CUDA, "cuTensorMapEncodeTiled(q_x) failed with CUresult %d", (int)r);
    store_map(key, *out);
    return HERALD_OK;
}

}  // namespace herald

using namespace herald;

extern "C" {

const char* herald_last_error(void) { return g_err; }

int32_t herald_budget_rows(int32_t seq_len, int32_t permille) {
    if (seq_len < 0 || permille < 0 || permille > 1000) return -1;
    const int64_t k = ((int64_t)seq_len * permille + 999) / 1000;
    return (int32_t)(k < seq_len ? k : seq_len);
}

size_t herald_select_workspace_bytes(const herald_shape_t* shape) {
    if (check_shape(shape) != HERALD_OK) return 0;
    return select_ws_layout(shape).total;
}

size_t herald_attn_workspace_bytes(const herald_shape_t* shape) {
    if (check_shape(shape) != HERALD_OK) return 0;
    return attn_geom(shape).total;
}

int32_t herald_attn_grid_ctas(const herald_shape_t* shape) {
    if (check_shape(shape) != HERALD_OK) return 0;
    const AttnGeom a = attn_geom(shape);
    return a.n_splits * a.m_tiles * shape->batch * shape->n_kv_heads;
}

// Top-k of every unit from the score plane and its level-1 histogram (shared by herald_select and herald_select_xq).
static int launch_topk(const herald_shape_t* shape, const herald_cache_t* cache, const float* scores, const uint32_t* hist1,
                       const int32_t* k_per_seq, int32_t* sel_idx, int32_t* sel_cnt, cudaStream_t stream, bool programmatic = false) {
    const int units = shape->batch * shape->n_kv_heads;
    cudaError_t e;
    TopkParams tp{};
    tp.scores = scores;
    tp.hist1 = hist1;
    tp.seq_lens = cache->seq_lens;
    tp.k_per_seq = k_per_seq;
    tp.sel_idx = sel_idx;
    tp.sel_cnt = sel_cnt;
    tp.n_kv_heads = shape->n_kv_heads;
    tp.max_seq_len = shape->max_seq_len;
    tp.cap = shape->pool_capacity;
    static bool topk_attr[kMaxDevices] = {false};
    e = ensure_smem(topk_kernel, kTopkMaxSmemBytes, topk_attr);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(topk)");
    // shared memory of the one-pass path: a bit per position and room for 1/8 of the positions in the threshold bin
    // (N(0,1)-like scores put 1-5 % of them there); what does not fit takes the multi-pass path
    tp.bitmap_words = (shape->max_seq_len + 31) / 32;
    if (tp.bitmap_words > kTopkMaxBitmapWords) tp.bitmap_words = kTopkMaxBitmapWords;
    tp.cand_cap = shape->max_seq_len / 8;
    if (tp.cand_cap < 2048) tp.cand_cap = 2048;
    if (tp.cand_cap > kTopkMaxCandCap) tp.cand_cap = kTopkMaxCandCap;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(units);
    cfg.blockDim = dim3(kTopkThreads);
    cfg.dynamicSmemBytes = (size_t)tp.cand_cap * 8 + 2 * (size_t)tp.bitmap_words * 4;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = programmatic ? 1 : 0;
    e = cudaLaunchKernelEx(&cfg, topk_kernel, tp);
    if (e != cudaSuccess) return cuda_fail(e, "topk launch");
    return HERALD_OK;
}

// herald_select in phases.  The pipeline runs the score scan in two launches (herald_pipeline_t.scan_head_permille): a head part
// over the first `head` thousandths of the cache on every SM, before the denoising steps start, and the rest on the SMs
// the attention grid leaves free, beside them; the level-1 histogram accumulates over both (global atomics).
enum { kSelectAll = 0, kSelectHead = 1, kSelectTail = 2 };
static int select_impl(const herald_shape_t* shape, const herald_cache_t* cache, const void* q_rep,
                  const int32_t* k_per_seq, int32_t* sel_idx, int32_t* sel_cnt, float* scores_out, void* ws,
                  size_t ws_bytes, herald_stream_t stream_, int phase, int head_permille) {
    int rc = check_shape(shape);
    if (rc) return rc;
    rc = check_cache(cache, false);
    if (rc) return rc;
    if (!q_rep || !k_per_seq || !sel_idx || !sel_cnt || !ws) return fail(HERALD_ERR_INVALID_ARG, "herald_select: NULL pointer");
    if (!aligned16(q_rep) || !aligned16(sel_idx) || !aligned16(scores_out) || (reinterpret_cast<uintptr_t>(ws) & 255u))
        return fail(HERALD_ERR_INVALID_ARG, "herald_select: misaligned pointer (16 B; workspace 256 B)");
    const SelectWs w = select_ws_layout(shape);
    if (ws_bytes < w.total) return fail(HERALD_ERR_WORKSPACE_TOO_SMALL, "herald_select: workspace %zu < %zu", ws_bytes, w.total);
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const int units = shape->batch * shape->n_kv_heads;
    if (units == 0) return HERALD_OK;
    g_err[0] = 0;

    uint8_t* wsb = static_cast<uint8_t*>(ws);
    uint32_t* hist1 = reinterpret_cast<uint32_t*>(wsb + w.hist1);
    float* scores = scores_out ? scores_out : reinterpret_cast<float*>(wsb + w.scores);
    cudaError_t e = cudaSuccess;
    if (phase != kSelectTail) {
        e = cudaMemsetAsync(hist1, 0, (size_t)units * kBins1 * sizeof(uint32_t), stream);
        if (e != cudaSuccess) return cuda_fail(e, "memset hist1");
    }
    const herald_profile_t* prof = (g_prof_armed || !g_in_pipeline) ? g_prof : nullptr;   // a plain herald_select is timed too
    if (prof && prof->scan_begin && phase != kSelectTail) cudaEventRecord(static_cast<cudaEvent_t>(prof->scan_begin), stream);

    if (shape->max_seq_len > 0) {
        ScanParams sp{};
        sp.k_pages = static_cast<const __nv_bfloat16*>(cache->k_pages);
        sp.page_stride = cache->page_stride;
        sp.token_stride = cache->token_stride;
        sp.head_stride = cache->head_stride;
        sp.page_table = cache->page_table;
        sp.seq_lens = cache->seq_lens;
        sp.q_rep = static_cast<const __nv_bfloat16*>(q_rep);
        sp.scores = scores;
        sp.raw = reinterpret_cast<float*>(wsb + w.raw);
        sp.stats_part = reinterpret_cast<float2*>(wsb + w.stats);
        sp.hist1 = hist1;
        sp.batch = shape->batch;
        sp.n_q_heads = shape->n_q_heads;
        sp.n_kv_heads = shape->n_kv_heads;
        sp.max_seq_len = shape->max_seq_len;
        sp.max_pages = shape->max_pages_per_seq;
        sp.sm_scale = shape->sm_scale;
        sp.part_lo = phase == kSelectTail ? head_permille : 0;
        sp.part_hi = phase == kSelectHead ? head_permille : 1000;
        // the head part runs alone on the device: one block per SM whatever the overlapped part is given
        const int scan_ctas = phase == kSelectHead ? (g_tune.scan_ctas > 0 ? g_tune.scan_ctas : sm_count()) : scan_ctas_for(shape);
        dim3 grid(scan_ctas);
        const int Hkv = shape->n_kv_heads;
        if (shape->agg_mode == HERALD_AGG_MAX_LOGIT && Hkv <= 8 && kScanWarps % Hkv == 0 && !g_tune.scan_head_major) {
            // page-major order: the warps next to each other read the head tiles of one page (whole pages for DRAM)
            const size_t smem = (size_t)Hkv * kBins1 * sizeof(uint32_t);
            static bool pm_attr[kMaxDevices] = {false}, pm_wide_attr[kMaxDevices] = {false};
            // A scan on less than half of the SMs (beside the attention) is bound by what one SM can draw, not by HBM: it takes
            // 32-byte loads (rows must be 32-byte aligned; the contract asks for 16) and prefetches the next page into L2 (pages
            // must be token-major and whole: the prefetched range [page, page + 16 token rows) then belongs to the page).
            const bool few = 2 * scan_ctas <= sm_count() && (kScanPmWideThreads / 32) % Hkv == 0;
            const bool wide = few && reinterpret_cast<uintptr_t>(sp.k_pages) % 32 == 0 && sp.page_stride % 16 == 0 && sp.token_stride % 16 == 0 &&
                              sp.head_stride % 16 == 0;
            // (the range ends with the last row the scan itself reads from the page, so it never leaves the caller's allocation)
            const int64_t page_span = ((kPageSize - 1) * sp.token_stride + (Hkv - 1) * sp.head_stride + kHeadDim) * 2;   // bytes
            if (wide && sp.token_stride >= (int64_t)Hkv * sp.head_stride && sp.head_stride >= kHeadDim &&
                sp.page_stride >= kPageSize * sp.token_stride && page_span <= (1 << 20))
                sp.l2_prefetch = (int32_t)page_span;
            e = wide ? ensure_smem(scan_pm_kernel<true, kScanPmWideThreads>, 8 * kBins1 * (int)sizeof(uint32_t), pm_wide_attr)
                     : ensure_smem(scan_pm_kernel<false, kScanThreads>, 8 * kBins1 * (int)sizeof(uint32_t), pm_attr);
            if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(scan)");
            if (wide) scan_pm_kernel<true, kScanPmWideThreads><<<grid, kScanPmWideThreads, smem, stream>>>(sp);
            else scan_pm_kernel<false, kScanThreads><<<grid, kScanThreads, smem, stream>>>(sp);
        } else if (shape->agg_mode == HERALD_AGG_MAX_LOGIT) {
            scan_kernel<0><<<grid, kScanThreads, 0, stream>>>(sp);
        } else {
            scan_kernel<1><<<grid, kScanThreads, 0, stream>>>(sp);
            AggParams ap{};
            ap.raw = sp.raw;
            ap.stats_part = sp.stats_part;
            ap.n_parts = scan_ctas;
            ap.batch = shape->batch;
            ap.seq_lens = cache->seq_lens;
            ap.scores = scores;
            ap.hist1 = hist1;
            ap.n_q_heads = shape->n_q_heads;
            ap.n_kv_heads = shape->n_kv_heads;
            ap.max_seq_len = shape->max_seq_len;
            int chunks = (shape->max_seq_len + 256 * 8 - 1) / (256 * 8);
            if (chunks < 1) chunks = 1;
            dim3 agrid(chunks, shape->n_kv_heads, shape->batch);
            aggregate_softmax_kernel<<<agrid, 256, 0, stream>>>(ap);
        }
        e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(e, "scan launch");
    }

    if (phase == kSelectHead) return HERALD_OK;
    if (prof && prof->scan_end) cudaEventRecord(static_cast<cudaEvent_t>(prof->scan_end), stream);
    rc = launch_topk(shape, cache, scores, hist1, k_per_seq, sel_idx, sel_cnt, stream);
    if (rc) return rc;
    if (prof && prof->topk_end) cudaEventRecord(static_cast<cudaEvent_t>(prof->topk_end), stream);
    return HERALD_OK;
}

int herald_select(const herald_shape_t* shape, const herald_cache_t* cache, const void* q_rep,
                  const int32_t* k_per_seq, int32_t* sel_idx, int32_t* sel_cnt, float* scores_out, void* ws,
                  size_t ws_bytes, herald_stream_t stream_) {
    return select_impl(shape, cache, q_rep, k_per_seq, sel_idx, sel_cnt, scores_out, ws, ws_bytes, stream_, kSelectAll, 0);
}

// ---- herald_select with its workspace inside the library (callers that may not allocate) -------------------------------
// The array's name is a device symbol: host code may not pass it to a kernel, it asks the runtime for its device address,
// once per device and with that device current.
static __device__ __align__(256) uint8_t g_select_scratch[HERALD_SELECT_STATIC_BYTES];

static int select_scratch_ptr(void** out) {
    static void* ptr[kMaxDevices] = {nullptr};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    if (dev < 0 || dev >= kMaxDevices) return fail(HERALD_ERR_UNSUPPORTED, "herald_select_static: device %d >= %d", dev, kMaxDevices);
    if (!ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_select_scratch);
        if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(select scratch)");
        if (!p || (reinterpret_cast<uintptr_t>(p) & 255u)) return fail(HERALD_ERR_CUDA, "herald_select_static: scratch symbol at %p", p);
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return HERALD_OK;
}

size_t herald_select_static_max_bytes(void) { return HERALD_SELECT_STATIC_BYTES; }

int herald_select_static(const herald_shape_t* shape, const herald_cache_t* cache, const void* q_rep,
                         const int32_t* k_per_seq, int32_t* sel_idx, int32_t* sel_cnt, herald_stream_t stream_) {
    int rc = check_shape(shape);
    if (rc) return rc;
    const size_t need = select_ws_layout(shape).total;
    if (need > (size_t)HERALD_SELECT_STATIC_BYTES)
        return fail(HERALD_ERR_WORKSPACE_TOO_SMALL,
                    "herald_select_static: this shape needs %zu bytes of scratch, the library holds %zu (batch * H_kv * (max_seq_len + %d) * 4 "
                    "must fit, mode 0); use herald_select with a caller-owned workspace", need, (size_t)HERALD_SELECT_STATIC_BYTES, kBins1);
    void* ws = nullptr;
    rc = select_scratch_ptr(&ws);
    if (rc) return rc;
    // the level-1 histograms must start at zero and the array keeps the last call's contents: select_impl clears them on the
    // stream before the scan, as it does for a caller's workspace; the score plane is fully rewritten for t < seq_lens[b]
    return select_impl(shape, cache, q_rep, k_per_seq, sel_idx, sel_cnt, nullptr, ws, (size_t)HERALD_SELECT_STATIC_BYTES, stream_, kSelectAll, 0);
}

int herald_select_xq(const herald_shape_t* shape, const herald_cache_t* cache, const void* q_x, int32_t x,
                     const int32_t* k_per_seq, int32_t* sel_idx, int32_t* sel_cnt, float* scores_out, void* ws,
                     size_t ws_bytes, herald_stream_t stream_) {
    int rc = check_shape(shape);
    if (rc) return rc;
    rc = check_cache(cache, false);
    if (rc) return rc;
    if (!q_x || !k_per_seq || !sel_idx || !sel_cnt || !ws) return fail(HERALD_ERR_INVALID_ARG, "herald_select_xq: NULL pointer");
    if (!aligned16(q_x) || !aligned16(sel_idx) || !aligned16(scores_out) || (reinterpret_cast<uintptr_t>(ws) & 255u))
        return fail(HERALD_ERR_INVALID_ARG, "herald_select_xq: misaligned pointer (16 B; workspace 256 B)");
    const int G = shape->n_q_heads / shape->n_kv_heads;
    if (x < 1 || (int64_t)x * G > 8 * kXqMaxTiles)
        return fail(HERALD_ERR_INVALID_ARG, "herald_select_xq: x = %d queries x G = %d heads must give 1..%d score rows per KV head", x, G, 8 * kXqMaxTiles);
    if (shape->agg_mode != HERALD_AGG_MAX_LOGIT)
        return fail(HERALD_ERR_INVALID_ARG, "herald_select_xq: only agg_mode HERALD_AGG_MAX_LOGIT is defined for x queries");
    const SelectWs w = select_ws_layout(shape);
    if (ws_bytes < w.total) return fail(HERALD_ERR_WORKSPACE_TOO_SMALL, "herald_select_xq: workspace %zu < %zu", ws_bytes, w.total);
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const int units = shape->batch * shape->n_kv_heads;
    if (units == 0) return HERALD_OK;
    g_err[0] = 0;

    uint8_t* wsb = static_cast<uint8_t*>(ws);
    uint32_t* hist1 = reinterpret_cast<uint32_t*>(wsb + w.hist1);
    float* scores = scores_out ? scores_out : reinterpret_cast<float*>(wsb + w.scores);
    cudaError_t e = cudaMemsetAsync(hist1, 0, (size_t)units * kBins1 * sizeof(uint32_t), stream);
    if (e != cudaSuccess) return cuda_fail(e, "memset hist1");
    if (shape->max_seq_len > 0) {
        // a dense contraction from ~32 score rows per KV head on: tcgen05 (scan_xq_tc.cuh); below that the rows fit a few
        // mma.sync tiles and the kernel is an HBM stream either way (scan_xq.cuh).  HERALD_XQ_TC = 0 / 1 forces one.
        const int rows = x * G;
        if (g_tune.xq_path == HERALD_XQ_TCGEN05 || (g_tune.xq_path != HERALD_XQ_MMA_SYNC && rows >= 32)) {
            CUtensorMap tm_k, tm_q;
            rc = make_paged_map(&tm_k, cache->k_pages, cache, shape->n_kv_heads);
            if (rc) return rc;
            rc = make_qx_map(&tm_q, q_x, shape, x);
            if (rc) return rc;
            ScanXqTcParams tp{};
            tp.page_table = cache->page_table;
            tp.seq_lens = cache->seq_lens;
            tp.scores = scores;
            tp.hist1 = hist1;
            tp.batch = shape->batch;
            tp.n_q_heads = shape->n_q_heads;
            tp.n_kv_heads = shape->n_kv_heads;
            tp.max_seq_len = shape->max_seq_len;
            tp.max_pages = shape->max_pages_per_seq;
            tp.x = x;
            tp.sm_scale = shape->sm_scale;
            const int xt_ctas = scan_ctas_for(shape);
            tp.set_size = (xt_ctas >= shape->n_kv_heads && !g_tune.scan_head_major) ? shape->n_kv_heads : 1;
            static bool xt_attr[kMaxDevices] = {false};
            e = ensure_smem(scan_xq_tc_kernel, kXtSmemBytes + 1024, xt_attr);
            if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(scan_xq_tc)");
            scan_xq_tc_kernel<<<xt_ctas, kXtThreads, kXtSmemBytes + 1024, stream>>>(tm_k, tm_q, tp);
        } else {
            ScanXqParams sp{};
            sp.k_pages = static_cast<const __nv_bfloat16*>(cache->k_pages);
            sp.page_stride = cache->page_stride;
            sp.token_stride = cache->token_stride;
            sp.head_stride = cache->head_stride;
            sp.page_table = cache->page_table;
            sp.seq_lens = cache->seq_lens;
            sp.q_x = static_cast<const __nv_bfloat16*>(q_x);
            sp.scores = scores;
            sp.hist1 = hist1;
            sp.batch = shape->batch;
            sp.n_q_heads = shape->n_q_heads;
            sp.n_kv_heads = shape->n_kv_heads;
            sp.max_seq_len = shape->max_seq_len;
            sp.max_pages = shape->max_pages_per_seq;
            sp.x = x;
            sp.sm_scale = shape->sm_scale;
            static bool xq_attr[kMaxDevices] = {false};
            e = ensure_smem(scan_xq_kernel, kXqMaxSmemBytes, xq_attr);
            if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(scan_xq)");
            const int n_tiles = (x * G + 7) / 8;
            scan_xq_kernel<<<scan_ctas_for(shape), kScanThreads, (size_t)n_tiles * kXqTileBytes, stream>>>(sp);
        }
        e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(e, "scan_xq launch");
    }
    return launch_topk(shape, cache, scores, hist1, k_per_seq, sel_idx, sel_cnt, stream);
}

int herald_gather(const herald_shape_t* shape, const herald_cache_t* cache, const int32_t* sel_idx,
                  const int32_t* sel_cnt, void* pool_k, void* pool_v, herald_stream_t stream_) {
    int rc = check_shape(shape);
    if (rc) return rc;
    rc = check_cache(cache, true);
    if (rc) return rc;
    if (!sel_idx || !sel_cnt || !pool_k || !pool_v) return fail(HERALD_ERR_INVALID_ARG, "herald_gather: NULL pointer");
    if (!aligned16(pool_k) || !aligned16(pool_v) || !aligned16(sel_idx))
        return fail(HERALD_ERR_INVALID_ARG, "herald_gather: misaligned pointer");
    const int units = shape->batch * shape->n_kv_heads;
    if (units == 0 || shape->pool_capacity == 0) return HERALD_OK;
    g_err[0] = 0;
    GatherParams gp{};
    gp.k_pages = static_cast<const __nv_bfloat16*>(cache->k_pages);
    gp.v_pages = static_cast<const __nv_bfloat16*>(cache->v_pages);
    gp.page_stride = cache->page_stride;
    gp.token_stride = cache->token_stride;
    gp.head_stride = cache->head_stride;
    gp.page_table = cache->page_table;
    gp.sel_idx = sel_idx;
    gp.sel_cnt = sel_cnt;
    gp.pool_k = static_cast<__nv_bfloat16*>(pool_k);
    gp.pool_v = static_cast<__nv_bfloat16*>(pool_v);
    gp.n_kv_heads = shape->n_kv_heads;
    gp.max_pages = shape->max_pages_per_seq;
    gp.cap = shape->pool_capacity;
    const int rows_per_cta = (kGatherThreads / 32) * kGatherRowsPerWarp;
    int gx = (shape->pool_capacity + rows_per_cta - 1) / rows_per_cta;
    if (gx > 4096) gx = 4096;
    dim3 grid(gx, units);
    gather_kernel<<<grid, kGatherThreads, 0, static_cast<cudaStream_t>(stream_)>>>(gp);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "gather launch");
    return HERALD_OK;
}

static int sparse_attn_impl(const herald_shape_t* shape, const void* pool_k, const void* pool_v, const int32_t* pool_len,
                            const void* q_blk, const void* k_blk, const void* v_blk, float* out, float* lse, void* ws,
                            size_t ws_bytes, herald_stream_t stream_, const int32_t* unit_order,
                            const herald_cache_t* dense_cache = nullptr, int pool_batch = 0) {
    const bool dense = dense_cache != nullptr;
    if (pool_batch <= 0) pool_batch = shape->batch;           // every query sequence has its own pools / pages
    const int units_pool = pool_batch * shape->n_kv_heads;
    int rc = check_shape(shape);
    if (rc) return rc;
    if (!pool_k || !pool_v || (!dense && !pool_len) || !q_blk || !k_blk || !v_blk || !out || !ws)
        return fail(HERALD_ERR_INVALID_ARG, "herald_sparse_attn / herald_dense_attn: NULL pointer");
    if (!aligned16(pool_k) || !aligned16(pool_v) || !aligned16(q_blk) || !aligned16(k_blk) || !aligned16(v_blk) ||
        !aligned16(out) || (reinterpret_cast<uintptr_t>(ws) & 255u))
        return fail(HERALD_ERR_INVALID_ARG, "herald_sparse_attn: misaligned pointer (16 B; workspace 256 B)");
    const AttnGeom a = attn_geom(shape, dense);
    if (ws_bytes < a.total) return fail(HERALD_ERR_WORKSPACE_TOO_SMALL, "herald_sparse_attn: workspace %zu < %zu", ws_bytes, a.total);
    const int units = shape->batch * shape->n_kv_heads;
    if (units == 0) return HERALD_OK;
    g_err[0] = 0;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);

    static bool attn_attr[kMaxDevices] = {false}, attn_fast_attr[kMaxDevices] = {false};
    {
        cudaError_t e = ensure_smem(attn_tc_kernel<false>, kTcSmemBytes, attn_attr);
        if (e == cudaSuccess) e = ensure_smem(attn_tc_kernel<true>, kTcSmemBytes, attn_fast_attr);
        if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(attn)");
    }
    CUtensorMap tm_k, tm_v, tm_q, tm_kb, tm_vb;
    rc = dense ? make_paged_map(&tm_k, pool_k, dense_cache, shape->n_kv_heads) : make_pool_map(&tm_k, pool_k, units_pool, shape->pool_capacity);
    if (rc) return rc;
    rc = dense ? make_paged_map(&tm_v, pool_v, dense_cache, shape->n_kv_heads) : make_pool_map(&tm_v, pool_v, units_pool, shape->pool_capacity);
    if (rc) return rc;
    rc = make_q_map(&tm_q, q_blk, shape, a.ipt);
    if (rc) return rc;
    rc = make_blk_map(&tm_kb, k_blk, shape);
    if (rc) return rc;
    rc = make_blk_map(&tm_vb, v_blk, shape);
    if (rc) return rc;
    AttnParams ap{};
    ap.pool_len = pool_len;
    ap.unit_order = unit_order;
    ap.page_table = dense ? dense_cache->page_table : nullptr;
    ap.seq_lens = dense ? dense_cache->seq_lens : nullptr;
    ap.max_pages = shape->max_pages_per_seq;
    ap.max_seq_len = shape->max_seq_len;
    ap.out = out;
    ap.lse = lse;
    ap.n_q_heads = shape->n_q_heads;
    ap.n_kv_heads = shape->n_kv_heads;
    ap.block_size = shape->block_size;
    ap.cap = shape->pool_capacity;
    ap.n_splits = a.n_splits;
    ap.pool_batch = pool_batch;
    ap.ipt = a.ipt;
    ap.pool_box = shape->pool_capacity < kTcBN ? (shape->pool_capacity > 0 ? shape->pool_capacity : 1) : kTcBN;
    ap.scale_log2 = shape->sm_scale * 1.4426950408889634f;
    ap.mode_hint = (size_t)a.n_splits * a.m_tiles * units * sizeof(int32_t) <= a.total - a.hint_off
                       ? reinterpret_cast<uint32_t*>(static_cast<uint8_t*>(ws) + a.hint_off) : nullptr;
    ap.precision = g_tune.attn_precision;
#ifdef HERALD_ATTN_TRACE
    ap.trace = g_attn_trace;
#endif
    // the n_splits CTAs of one (unit, M tile) are one thread-block cluster: the split-KV merge runs over DSMEM
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(a.n_splits, a.m_tiles, units);
    cfg.blockDim = dim3(kTcThreads);
    cfg.dynamicSmemBytes = kTcSmemBytes;
    cfg.stream = stream;
    cudaLaunchAttribute attr[2];
    int n_attr = 0;
    if (a.n_splits > 1) {
        attr[n_attr].id = cudaLaunchAttributeClusterDimension;
        attr[n_attr].val.clusterDim.x = a.n_splits;
        attr[n_attr].val.clusterDim.y = 1;
        attr[n_attr].val.clusterDim.z = 1;
        ++n_attr;
    }
    if (!g_tune.attn_no_pdl) {
        // consecutive denoising steps: the next grid is scheduled while this one runs its merge and takes each SM as
        // it is released (the kernel itself waits, griddepcontrol.wait, before its first global read)
        attr[n_attr].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[n_attr].val.programmaticStreamSerializationAllowed = 1;
        ++n_attr;
    }
    cfg.attrs = attr;
    cfg.numAttrs = n_attr;
    // the instantiation with the fast first pass only where some block can have a key share long enough to try it
    const int max_keys = (dense ? shape->max_seq_len : shape->pool_capacity) + shape->block_size;
    // (and only for shapes whose step is bound by the tensor pipe / softmax issue: an M tile of 64 rows streams its pool at the HBM rate)
    const bool try_fast = g_tune.attn_precision == HERALD_ATTN_FAST_FIRST ||
                          (g_tune.attn_precision == HERALD_ATTN_AUTO && a.ipt * (shape->n_q_heads / shape->n_kv_heads) >= 96 &&
                           (max_keys + a.n_splits - 1) / a.n_splits + kTcBN >= kTcFastMinKeys);
    cudaError_t e = try_fast ? cudaLaunchKernelEx(&cfg, attn_tc_kernel<true>, tm_k, tm_v, tm_q, tm_kb, tm_vb, ap)
                             : cudaLaunchKernelEx(&cfg, attn_tc_kernel<false>, tm_k, tm_v, tm_q, tm_kb, tm_vb, ap);
    if (e != cudaSuccess) return cuda_fail(e, "attention launch");
    return HERALD_OK;
}

int herald_sparse_attn(const herald_shape_t* shape, const void* pool_k, const void* pool_v, const int32_t* pool_len,
                       const void* q_blk, const void* k_blk, const void* v_blk, float* out, float* lse, void* ws,
                       size_t ws_bytes, herald_stream_t stream_) {
    return sparse_attn_impl(shape, pool_k, pool_v, pool_len, q_blk, k_blk, v_blk, out, lse, ws, ws_bytes, stream_, nullptr);
}

int herald_sparse_attn_groups(const herald_shape_t* shape, int32_t n_groups, const void* pool_k, const void* pool_v,
                              const int32_t* pool_len, const void* q_blk, const void* k_blk, const void* v_blk, float* out,
                              float* lse, void* ws, size_t ws_bytes, herald_stream_t stream) {
    int rc = check_shape(shape);
    if (rc) return rc;
    if (n_groups < 1 || (int64_t)n_groups * shape->batch > (1 << 20))
        return fail(HERALD_ERR_INVALID_ARG, "herald_sparse_attn_groups: n_groups = %d", n_groups);
    herald_shape_t grouped = *shape;                          // the query side sees n_groups * batch sequences,
    grouped.batch = shape->batch * n_groups;                  // sequence b of group g reads the pools of sequence b
    return sparse_attn_impl(&grouped, pool_k, pool_v, pool_len, q_blk, k_blk, v_blk, out, lse, ws, ws_bytes, stream, nullptr,
                            nullptr, shape->batch);
}

int herald_dense_attn(const herald_shape_t* shape, const herald_cache_t* cache, const void* q_blk, const void* k_blk,
                      const void* v_blk, float* out, float* lse, void* ws, size_t ws_bytes, herald_stream_t stream_) {
    int rc = check_shape(shape);
    if (rc) return rc;
    rc = check_cache(cache, true);
    if (rc) return rc;
    return sparse_attn_impl(shape, cache->k_pages, cache->v_pages, nullptr, q_blk, k_blk, v_blk, out, lse, ws, ws_bytes, stream_, nullptr, cache);
}

int herald_cache_write_block(const herald_shape_t* shape, const herald_cache_t* cache, const int32_t* write_pos,
                             const void* k_new, const void* v_new, herald_stream_t stream_) {
    int rc = check_shape(shape);
    if (rc) return rc;
    rc = check_cache(cache, true);
    if (rc) return rc;
    if (!write_pos || !k_new || !v_new) return fail(HERALD_ERR_INVALID_ARG, "herald_cache_write_block: NULL pointer");
    if (!aligned16(k_new) || !aligned16(v_new)) return fail(HERALD_ERR_INVALID_ARG, "herald_cache_write_block: misaligned pointer");
    const int rows = shape->batch * shape->block_size * shape->n_kv_heads;
    if (rows == 0) return HERALD_OK;
    g_err[0] = 0;
    CacheWriteParams cp{};
    cp.k_pages = static_cast<__nv_bfloat16*>(const_cast<void*>(cache->k_pages));
    cp.v_pages = static_cast<__nv_bfloat16*>(const_cast<void*>(cache->v_pages));
    cp.page_stride = cache->page_stride;
    cp.token_stride = cache->token_stride;
    cp.head_stride = cache->head_stride;
    cp.page_table = cache->page_table;
    cp.write_pos = write_pos;
    cp.k_new = static_cast<const __nv_bfloat16*>(k_new);
    cp.v_new = static_cast<const __nv_bfloat16*>(v_new);
    cp.batch = shape->batch;
    cp.block_size = shape->block_size;
    cp.n_kv_heads = shape->n_kv_heads;
    cp.max_pages = shape->max_pages_per_seq;
    int grid = (rows + 15) / 16;
    if (grid > 4 * sm_count()) grid = 4 * sm_count();
    cache_write_block_kernel<<<grid, 256, 0, static_cast<cudaStream_t>(stream_)>>>(cp);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "cache_write_block launch");
    return HERALD_OK;
}

int herald_pool_append_block(const herald_shape_t* shape, void* pool_k, void* pool_v, int32_t* pool_len, const void* k_new,
                             const void* v_new, herald_stream_t stream_) {
    int rc = check_shape(shape);
    if (rc) return rc;
    if (!pool_k || !pool_v || !pool_len || !k_new || !v_new) return fail(HERALD_ERR_INVALID_ARG, "herald_pool_append_block: NULL pointer");
    if (!aligned16(pool_k) || !aligned16(pool_v) || !aligned16(k_new) || !aligned16(v_new))
        return fail(HERALD_ERR_INVALID_ARG, "herald_pool_append_block: misaligned pointer");
    const int units = shape->batch * shape->n_kv_heads;
    if (units == 0 || shape->pool_capacity == 0) return HERALD_OK;
    g_err[0] = 0;
    PoolAppendParams pp{};
    pp.pool_k = static_cast<__nv_bfloat16*>(pool_k);
    pp.pool_v = static_cast<__nv_bfloat16*>(pool_v);
    pp.pool_len = pool_len;
    pp.k_new = static_cast<const __nv_bfloat16*>(k_new);
    pp.v_new = static_cast<const __nv_bfloat16*>(v_new);
    pp.batch = shape->batch;
    pp.block_size = shape->block_size;
    pp.n_kv_heads = shape->n_kv_heads;
    pp.cap = shape->pool_capacity;
    pool_append_block_kernel<<<units, 256, 0, static_cast<cudaStream_t>(stream_)>>>(pp);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "pool_append_block launch");
    return HERALD_OK;
}

// herald_rep_attn takes hg KV heads of a page together: the largest of 8, 4, 2, 1 that divides H_kv
static int rep_head_group(const herald_shape_t* s) {
    for (int hg = 8; hg > 1; hg >>= 1)
        if (s->n_kv_heads % hg == 0) return hg;
    return 1;
}

size_t herald_rep_attn_workspace_bytes(const herald_shape_t* shape) {
    if (check_shape(shape) != HERALD_OK) return 0;
    const size_t hg = rep_head_group(shape), groups = (size_t)shape->batch * (shape->n_kv_heads / hg);
    return align_up((kRepMaxCtas + groups) * hg * kRepPartFloats * sizeof(float), 256);   // slot = cta + group, hg head partials each
}

// The K+V pass of herald_rep_attn; with `scores` it also writes the max-logit selection scores (herald_select_rep).
// `between` (herald_select_rep: the top-k, launched programmatically) runs after the pass and before the merge is enqueued;
// the merge then starts beside it and does not wait for it.
static int rep_attn_launch(const herald_shape_t* shape, const herald_cache_t* cache, const void* q_rep, float* out, float* lse,
                           void* ws, float* scores, uint32_t* hist1, float* raw, cudaStream_t stream,
                           const std::function<int()>& between, bool has_between) {
    RepAttnParams rp{};
    rp.scores = scores;
    rp.hist1 = hist1;
    rp.raw = raw;
    rp.sm_scale = shape->sm_scale;
    rp.merge_waits = has_between ? 0 : 1;
    rp.k_pages = static_cast<const __nv_bfloat16*>(cache->k_pages);
    rp.v_pages = static_cast<const __nv_bfloat16*>(cache->v_pages);
    rp.page_stride = cache->page_stride;
    rp.token_stride = cache->token_stride;
    rp.head_stride = cache->head_stride;
    rp.page_table = cache->page_table;
    rp.seq_lens = cache->seq_lens;
    rp.q_rep = static_cast<const __nv_bfloat16*>(q_rep);
    rp.hg = rep_head_group(shape);
    rp.part = static_cast<float*>(ws);
    rp.batch = shape->batch;
    rp.out = out;
    rp.lse = lse;
    rp.n_q_heads = shape->n_q_heads;
    rp.n_kv_heads = shape->n_kv_heads;
    rp.max_seq_len = shape->max_seq_len;
    rp.max_pages = shape->max_pages_per_seq;
    rp.scale_log2 = shape->sm_scale * 1.4426950408889634f;
    const int n_ctas = std::min(2 * sm_count(), kRepMaxCtas);   // persistent: two CTAs per SM
    static bool rep_attr[kMaxDevices] = {false};   // over the 48 KB default: opt in once per device
    {
        const cudaError_t ea = ensure_smem(rep_attn_kernel, kRepSmemBytes, rep_attr);
        if (ea != cudaSuccess) return cuda_fail(ea, "cudaFuncSetAttribute(rep_attn)");
    }
    rep_attn_kernel<<<n_ctas, kRepThreads, kRepSmemBytes, stream>>>(rp);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "rep_attn launch");
    if (has_between) {
        const int rc = between();
        if (rc) return rc;
    }
    // the merge is launched programmatically behind the main grid: its blocks are scheduled as the main CTAs retire,
    // find their partial list (inputs only) and wait (griddepcontrol.wait) for the grid to complete
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(shape->batch * shape->n_q_heads);
    cfg.blockDim = dim3(kHeadDim, kRepMergeSlices);
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    e = cudaLaunchKernelEx(&cfg, rep_attn_merge_kernel, rp, n_ctas);
    if (e != cudaSuccess) return cuda_fail(e, "rep_attn launch");
    return HERALD_OK;
}

int herald_rep_attn(const herald_shape_t* shape, const herald_cache_t* cache, const void* q_rep, float* out, float* lse,
                    void* ws, size_t ws_bytes, herald_stream_t stream_) {
    int rc = check_shape(shape);
    if (rc) return rc;
    rc = check_cache(cache, true);
    if (rc) return rc;
    if (!q_rep || !out || !ws) return fail(HERALD_ERR_INVALID_ARG, "herald_rep_attn: NULL pointer");
    if (!aligned16(q_rep) || !aligned16(out) || (reinterpret_cast<uintptr_t>(ws) & 255u))
        return fail(HERALD_ERR_INVALID_ARG, "herald_rep_attn: misaligned pointer (16 B; workspace 256 B)");
    const size_t need = herald_rep_attn_workspace_bytes(shape);
    if (ws_bytes < need) return fail(HERALD_ERR_WORKSPACE_TOO_SMALL, "herald_rep_attn: workspace %zu < %zu", ws_bytes, need);
    if (shape->batch * shape->n_kv_heads == 0) return HERALD_OK;
    g_err[0] = 0;
    return rep_attn_launch(shape, cache, q_rep, out, lse, ws, nullptr, nullptr, nullptr, static_cast<cudaStream_t>(stream_), [] { return 0; }, false);
}

size_t herald_select_rep_workspace_bytes(const herald_shape_t* shape) {
    if (check_shape(shape) != HERALD_OK) return 0;
    // select workspace, rep_attn partials, and a log-sum-exp per query head (mode 1 needs it even when the caller does not)
    return align_up(select_ws_layout(shape).total, 256) + herald_rep_attn_workspace_bytes(shape) +
           align_up((size_t)(shape->batch > 0 ? shape->batch : 1) * shape->n_q_heads * sizeof(float), 256);
}

int herald_select_rep(const herald_shape_t* shape, const herald_cache_t* cache, const void* q_rep, const int32_t* k_per_seq,
                      int32_t* sel_idx, int32_t* sel_cnt, float* scores_out, float* rep_out, float* rep_lse, void* ws,
                      size_t ws_bytes, herald_stream_t stream_) {
    int rc = check_shape(shape);
    if (rc) return rc;
    rc = check_cache(cache, true);
    if (rc) return rc;
    if (!q_rep || !k_per_seq || !sel_idx || !sel_cnt || !rep_out || !ws) return fail(HERALD_ERR_INVALID_ARG, "herald_select_rep: NULL pointer");
    if (!aligned16(q_rep) || !aligned16(sel_idx) || !aligned16(scores_out) || !aligned16(rep_out) || (reinterpret_cast<uintptr_t>(ws) & 255u))
        return fail(HERALD_ERR_INVALID_ARG, "herald_select_rep: misaligned pointer (16 B; workspace 256 B)");
    const size_t need = herald_select_rep_workspace_bytes(shape);
    if (ws_bytes < need) return fail(HERALD_ERR_WORKSPACE_TOO_SMALL, "herald_select_rep: workspace %zu < %zu", ws_bytes, need);
    const int units = shape->batch * shape->n_kv_heads;
    if (units == 0) return HERALD_OK;
    g_err[0] = 0;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const SelectWs w = select_ws_layout(shape);
    uint8_t* wsb = static_cast<uint8_t*>(ws);
    uint32_t* hist1 = reinterpret_cast<uint32_t*>(wsb + w.hist1);
    float* scores = scores_out ? scores_out : reinterpret_cast<float*>(wsb + w.scores);
    cudaError_t e = cudaMemsetAsync(hist1, 0, (size_t)units * kBins1 * sizeof(uint32_t), stream);
    if (e != cudaSuccess) return cuda_fail(e, "memset hist1");
    uint8_t* ws_rep = wsb + align_up(w.total, 256);
    if (shape->agg_mode == HERALD_AGG_MAX_LOGIT) {
        // pass (scores + histogram + partials) -> top-k, launched programmatically behind the pass -> merge, beside the top-k
        return rep_attn_launch(shape, cache, q_rep, rep_out, rep_lse, ws_rep, scores, hist1, nullptr, stream,
                               [&] { return launch_topk(shape, cache, scores, hist1, k_per_seq, sel_idx, sel_cnt, stream, true); }, true);
    }
    // softmax-sum aggregation: a[t] = sum_g exp(s[g,t] - m_g) / l_g needs the finished (m_g, l_g), i.e. the
    // log-sum-exp the merge produces.  The pass keeps the per-head logits; after the merge one more kernel turns them into
    // the score plane and its histogram; then the top-k.
    float* lse_buf = rep_lse ? rep_lse : reinterpret_cast<float*>(ws_rep + herald_rep_attn_workspace_bytes(shape));
    float* raw = reinterpret_cast<float*>(wsb + w.raw);
    rc = rep_attn_launch(shape, cache, q_rep, rep_out, lse_buf, ws_rep, nullptr, nullptr, raw, stream, [] { return 0; }, false);
    if (rc) return rc;
    if (shape->max_seq_len > 0) {
        AggParams ap{};
        ap.raw = raw;
        ap.lse = lse_buf;
        ap.batch = shape->batch;
        ap.seq_lens = cache->seq_lens;
        ap.scores = scores;
        ap.hist1 = hist1;
        ap.n_q_heads = shape->n_q_heads;
        ap.n_kv_heads = shape->n_kv_heads;
        ap.max_seq_len = shape->max_seq_len;
        int chunks = (shape->max_seq_len + 256 * 8 - 1) / (256 * 8);
        if (chunks < 1) chunks = 1;
        aggregate_softmax_kernel<<<dim3(chunks, shape->n_kv_heads, shape->batch), 256, 0, stream>>>(ap);
        e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(e, "aggregate launch");
    }
    return launch_topk(shape, cache, scores, hist1, k_per_seq, sel_idx, sel_cnt, stream);
}

// Longest-pool-first unit order of one layer into `order` (device, [units]); enqueued on `stream`.
static int attn_plan(const herald_shape_t* shape, const int32_t* pool_len, int32_t* order, cudaStream_t stream) {
    const int units = shape->batch * shape->n_kv_heads;
    if (units == 0) return HERALD_OK;
    attn_plan_kernel<<<1, 1024, 0, stream>>>(pool_len, shape->pool_capacity, units, order);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "attention plan launch");
    return HERALD_OK;
}

// Grid of the overlapped score scan when the caller leaves herald_pipeline_t.scan_ctas at 0: the SMs the attention grid
// leaves free, at least an eighth of the device (a scan grid larger than that takes SMs the next attention launch needs and
// was measured slower than running the two streams one after the other).
static int default_scan_ctas(const herald_shape_t* sh) {
    const int n_sm = sm_count(), attn = herald_attn_grid_ctas(sh);
    if (attn <= 0) return n_sm;
    const int rem = attn % n_sm;                         // blocks of the attention grid's last wave
    const int spare = rem == 0 ? 0 : n_sm - rem, floor8 = n_sm / 8 > 0 ? n_sm / 8 : 1;
    return spare > floor8 ? spare : floor8;
}

static int check_pipeline(const herald_pipeline_t* p) {
    if (!p) return fail(HERALD_ERR_INVALID_ARG, "pipeline is NULL");
    int rc = check_shape(&p->shape);
    if (rc) return rc;
    if (p->n_layers <= 0 || !p->layers) return fail(HERALD_ERR_INVALID_ARG, "pipeline: no layers");
    if (p->n_steps < 0 || p->start_after_step < 0 || p->start_after_step > p->n_steps)
        return fail(HERALD_ERR_INVALID_ARG, "pipeline: bad n_steps / start_after_step");
    if (p->active != 0 && p->active != 1) return fail(HERALD_ERR_INVALID_ARG, "pipeline: active must be 0 or 1");
    if (p->scan_ctas < 0) return fail(HERALD_ERR_INVALID_ARG, "pipeline: scan_ctas must be >= 0");
    if (p->scan_head_permille < 0 || p->scan_head_permille > 1000)
        return fail(HERALD_ERR_INVALID_ARG, "pipeline: scan_head_permille must be 0..1000");
    if (!p->sel_idx || !p->ws_select || !p->ws_attn || !p->ev_fork || !p->ev_join)
        return fail(HERALD_ERR_INVALID_ARG, "pipeline: NULL scratch / workspace / event");
    if (p->main_stream == p->retrieval_stream)
        return fail(HERALD_ERR_INVALID_ARG, "pipeline: main and retrieval streams must differ");
    for (int l = 0; l < p->n_layers; ++l) {       // nothing is enqueued unless every layer is complete
        const herald_layer_t* ly = &p->layers[l];
        if (!ly->q_blk || !ly->k_blk || !ly->v_blk || !ly->out) return fail(HERALD_ERR_INVALID_ARG, "pipeline: layer %d has a NULL block tensor", l);
        int rc2 = check_cache(&ly->cache, true);
        if (rc2) return rc2;
        if (!ly->dense && (!ly->q_rep || !ly->k_per_seq || !ly->pool_k[0] || !ly->pool_k[1] || !ly->pool_v[0] || !ly->pool_v[1] ||
                           !ly->pool_len[0] || !ly->pool_len[1]))
            return fail(HERALD_ERR_INVALID_ARG, "pipeline: sparse layer %d has a NULL q_rep / k_per_seq / pool pointer", l);
    }
    return HERALD_OK;
}

int herald_pipeline_step(herald_pipeline_t* p) {
    int rc = check_pipeline(p);
    if (rc) return rc;
    cudaStream_t s_main = static_cast<cudaStream_t>(p->main_stream);
    cudaStream_t s_ret = static_cast<cudaStream_t>(p->retrieval_stream);
    cudaEvent_t ev_fork = static_cast<cudaEvent_t>(p->ev_fork), ev_join = static_cast<cudaEvent_t>(p->ev_join);
    const herald_shape_t* sh = &p->shape;
    const int act = p->active, idle = 1 - act;
    const size_t q_step = (size_t)sh->batch * sh->block_size * sh->n_q_heads * kHeadDim;
    const size_t kv_step = (size_t)sh->batch * sh->block_size * sh->n_kv_heads * kHeadDim;
    cudaError_t e;
    const int scan_ctas = p->scan_ctas > 0 ? p->scan_ctas : default_scan_ctas(sh);
    // head part of the first sparse layer's scan: on every SM, and the main stream waits for it (max-logit aggregation only)
    const int head = sh->agg_mode == HERALD_AGG_MAX_LOGIT ? p->scan_head_permille : 0;
    bool head_pending = false;

    auto retrieval = [&]() -> int {
        e = cudaEventRecord(ev_fork, s_main);
        if (e != cudaSuccess) return cuda_fail(e, "record fork");
        e = cudaStreamWaitEvent(s_ret, ev_fork, 0);
        if (e != cudaSuccess) return cuda_fail(e, "wait fork");
        if (g_delay_retrieval_us) delay_kernel<<<1, 1, 0, s_ret>>>((unsigned long long)g_delay_retrieval_us * 1000ull);
        int last_sparse = -1;
        for (int l = 0; l < p->n_layers; ++l)
            if (!p->layers[l].dense) last_sparse = l;
        for (int l = 0; l < p->n_layers; ++l) {
            herald_layer_t* ly = &p->layers[l];
            if (ly->dense) continue;                      // keeps its full KV: nothing to select
            g_prof_armed = (l == last_sparse);
            g_in_pipeline = true;
            g_scan_ctas = scan_ctas;
            int r;
            if (head > 0 && !head_pending) {
                r = select_impl(sh, &ly->cache, ly->q_rep, ly->k_per_seq, p->sel_idx, ly->pool_len[idle], nullptr, p->ws_select,
                                p->ws_select_bytes, s_ret, kSelectHead, head);
                if (r == HERALD_OK) {
                    // the main stream resumes here; the wait is enqueued now because the join records the same event again below
                    e = cudaEventRecord(ev_join, s_ret);
                    if (e == cudaSuccess) e = cudaStreamWaitEvent(s_main, ev_join, 0);
                    if (e != cudaSuccess) r = cuda_fail(e, "record / wait scan head");
                    head_pending = true;
                }
                if (r == HERALD_OK)
                    r = select_impl(sh, &ly->cache, ly->q_rep, ly->k_per_seq, p->sel_idx, ly->pool_len[idle], nullptr, p->ws_select,
                                    p->ws_select_bytes, s_ret, kSelectTail, head);
            } else {
                r = herald_select(sh, &ly->cache, ly->q_rep, ly->k_per_seq, p->sel_idx, ly->pool_len[idle], nullptr,
                                  p->ws_select, p->ws_select_bytes, s_ret);
            }
            g_prof_armed = false;
            g_in_pipeline = false;
            g_scan_ctas = 0;
            if (r) return r;
            r = herald_gather(sh, &ly->cache, p->sel_idx, ly->pool_len[idle], ly->pool_k[idle], ly->pool_v[idle], s_ret);
            if (r) return r;
            if (l == last_sparse && g_prof && g_prof->gather_end)
                cudaEventRecord(static_cast<cudaEvent_t>(g_prof->gather_end), s_ret);
        }
        e = cudaEventRecord(ev_join, s_ret);
        if (e != cudaSuccess) return cuda_fail(e, "record join");
        return HERALD_OK;
    };

    // A multi-wave attention grid (more blocks than SMs) over ragged pools is dispatched longest pool first: one tiny plan
    // kernel per layer and block writes the unit order into that layer's slice of the attention workspace.
    const size_t ws_layer = attn_geom(sh).total;
    const bool planned = herald_attn_grid_ctas(sh) > sm_count() && p->ws_attn_bytes >= ws_layer * (size_t)p->n_layers && p->n_steps > 0;
    if (planned) {
        for (int l = 0; l < p->n_layers; ++l) {
            if (p->layers[l].dense) continue;
            rc = attn_plan(sh, p->layers[l].pool_len[act], reinterpret_cast<int32_t*>(static_cast<uint8_t*>(p->ws_attn) + ws_layer * l), s_main);
            if (rc) return rc;
        }
    }
    bool forked = false;
    for (int s = 0; s <= p->n_steps; ++s) {
        if (s == p->start_after_step && !forked) {
            rc = retrieval();
            if (rc) return rc;
            forked = true;
            if (g_delay_main_us) delay_kernel<<<1, 1, 0, s_main>>>((unsigned long long)g_delay_main_us * 1000ull);
        }
        if (s == p->n_steps) break;
        for (int l = 0; l < p->n_layers; ++l) {
            herald_layer_t* ly = &p->layers[l];
            if (ly->dense) {      // exact attention over the whole paged cache
                rc = sparse_attn_impl(sh, ly->cache.k_pages, ly->cache.v_pages, nullptr,
                                      static_cast<const __nv_bfloat16*>(ly->q_blk) + s * q_step,
                                      static_cast<const __nv_bfloat16*>(ly->k_blk) + s * kv_step,
                                      static_cast<const __nv_bfloat16*>(ly->v_blk) + s * kv_step,
                                      ly->out + s * q_step, nullptr, p->ws_attn, p->ws_attn_bytes, s_main, nullptr, &ly->cache);
                if (rc) return rc;
                continue;
            }
            rc = sparse_attn_impl(sh, ly->pool_k[act], ly->pool_v[act], ly->pool_len[act],
                                  static_cast<const __nv_bfloat16*>(ly->q_blk) + s * q_step,
                                  static_cast<const __nv_bfloat16*>(ly->k_blk) + s * kv_step,
                                  static_cast<const __nv_bfloat16*>(ly->v_blk) + s * kv_step,
                                  ly->out + s * q_step, nullptr, p->ws_attn, p->ws_attn_bytes, s_main,
                                  planned ? reinterpret_cast<const int32_t*>(static_cast<const uint8_t*>(p->ws_attn) + ws_layer * l) : nullptr);
            if (rc) return rc;
        }
    }
    e = cudaStreamWaitEvent(s_main, ev_join, 0);
    if (e != cudaSuccess) return cuda_fail(e, "wait join");
    p->active = idle;
    return HERALD_OK;
}

#ifdef HERALD_ATTN_TRACE
int herald_debug_set_attn_trace(void* dev_buf) {
    g_attn_trace = static_cast<unsigned long long*>(dev_buf);
    return HERALD_OK;
}
#endif

int herald_pipeline_tune(herald_pipeline_t* p, int32_t reps, herald_schedule_t* table, int32_t table_cap, int32_t* n_table) {
    int rc = check_pipeline(p);
    if (rc) return rc;
    if (reps < 1 || reps > 1000) return fail(HERALD_ERR_INVALID_ARG, "herald_pipeline_tune: reps must be 1..1000");
    cudaStream_t s_main = static_cast<cudaStream_t>(p->main_stream), s_ret = static_cast<cudaStream_t>(p->retrieval_stream);
    cudaEvent_t a, b;
    cudaError_t e = cudaEventCreate(&a);
    if (e != cudaSuccess) return cuda_fail(e, "event create");
    e = cudaEventCreate(&b);
    if (e != cudaSuccess) { cudaEventDestroy(a); return cuda_fail(e, "event create"); }
    const int n_sm = sm_count(), spare = default_scan_ctas(&p->shape), start0 = p->start_after_step;
    int n = 0;
    float best_ms = 0.f;
    herald_schedule_t best{p->scan_ctas, p->start_after_step, p->scan_head_permille, 0.f};
    // a candidate is timed the way a serving loop runs it: the block step captured once into a CUDA graph and replayed (cross-stream
    // event waits cost several microseconds more between eagerly launched kernels than between graph nodes, which would
    // bias the choice against schedules with an extra dependency); the replays use the same pool parity, which changes nothing
    // in the work done.  If the capture fails (streams already capturing) the candidate is timed with eager steps.
    auto time_one = [&](int ctas, int start, int head) -> int {
        p->scan_ctas = ctas; p->start_after_step = start; p->scan_head_permille = head;
        int r = HERALD_OK;
        for (int i = 0; i < 2 && r == HERALD_OK; ++i) r = herald_pipeline_step(p);    // eager warm-up: one-time setup, both parities
        if (r) return r;
        cudaStreamSynchronize(s_main); cudaStreamSynchronize(s_ret);
        cudaGraph_t graph = nullptr;
        cudaGraphExec_t exec = nullptr;
        const int act0 = p->active;
        if (cudaStreamBeginCapture(s_main, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
            r = herald_pipeline_step(p);
            const cudaError_t ce = cudaStreamEndCapture(s_main, &graph);
            p->active = act0;                                   // the capture enqueued nothing
            if (r != HERALD_OK || ce != cudaSuccess || cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) exec = nullptr;
            if (r != HERALD_OK) { if (graph) cudaGraphDestroy(graph); return r; }
        }
        (void)cudaGetLastError();
        auto run = [&]() -> int {
            if (exec) return cudaGraphLaunch(exec, s_main) == cudaSuccess ? HERALD_OK : fail(HERALD_ERR_CUDA, "herald_pipeline_tune: graph launch failed");
            return herald_pipeline_step(p);
        };
        for (int i = 0; i < 2 && r == HERALD_OK; ++i) r = run();
        if (r == HERALD_OK) {
            cudaStreamSynchronize(s_main); cudaStreamSynchronize(s_ret);
            cudaEventRecord(a, s_main);
            for (int i = 0; i < reps && r == HERALD_OK; ++i) r = run();
            cudaEventRecord(b, s_main);
            const cudaError_t ee = cudaEventSynchronize(b);
            if (r == HERALD_OK && ee != cudaSuccess) r = cuda_fail(ee, "herald_pipeline_tune: step failed");
        }
        cudaStreamSynchronize(s_ret);
        if (exec) cudaGraphExecDestroy(exec);
        if (graph) cudaGraphDestroy(graph);
        if (r) return r;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, a, b);
        ms /= (float)reps;
        if (table && n < table_cap) table[n] = herald_schedule_t{ctas, start, head, ms};
        ++n;
        if (best_ms == 0.f || ms < best_ms) { best_ms = ms; best = herald_schedule_t{ctas, start, head, ms}; }
        return HERALD_OK;
    };
    // 1. the scan grid beside the denoising steps: around the SMs the attention grid leaves free; every SM; every SM after the last step
    // (a multi-wave attention grid has no hard number of free SMs: a few more for the scan can pay, C5 takes 56 rather than 40)
    const int grids[5] = {spare - 2, spare, n_sm / 8, spare + n_sm / 16, spare + n_sm / 8};
    for (int i = 0; i < 5 && rc == HERALD_OK; ++i) {
        bool dup = (grids[i] < 8 && grids[i] != spare) || grids[i] >= n_sm;
        for (int j = 0; j < i; ++j) dup = dup || grids[j] == grids[i];
        if (!dup && grids[i] >= 1) rc = time_one(grids[i], start0, 0);
    }
    if (rc == HERALD_OK) rc = time_one(n_sm, start0, 0);
    if (rc == HERALD_OK && start0 != p->n_steps && p->n_steps > 0) rc = time_one(n_sm, p->n_steps, 0);
    // 2. with the best overlapped grid: how much of the scan runs on every SM before the denoising steps start
    if (rc == HERALD_OK && best.scan_ctas < n_sm && p->shape.agg_mode == HERALD_AGG_MAX_LOGIT) {
        const int ctas = best.scan_ctas, start = best.start_after_step;
        const int heads[6] = {50, 100, 200, 300, 450, 600};
        for (int i = 0; i < 6 && rc == HERALD_OK; ++i) rc = time_one(ctas, start, heads[i]);
    }
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    p->scan_ctas = best.scan_ctas; p->start_after_step = best.start_after_step; p->scan_head_permille = best.scan_head_permille;
    if (n_table) *n_table = n < table_cap ? n : table_cap;
    return rc;
}

int herald_set_tuning(const herald_tuning_t* t) {
    if (!t) {
        g_tune = herald_tuning_t{0, 0, 0, 0, 0, 0, 0, 0};
        return HERALD_OK;
    }
    if (t->attn_splits < 0 || t->attn_splits > kTcMaxSplits || t->attn_m_tiles < 0 || t->attn_total_ctas < 0 || t->scan_ctas < 0 ||
        t->xq_path < HERALD_XQ_AUTO || t->xq_path > HERALD_XQ_TCGEN05 || t->attn_precision < HERALD_ATTN_AUTO ||
        t->attn_precision > HERALD_ATTN_FAST_FIRST)
        return fail(HERALD_ERR_INVALID_ARG, "herald_set_tuning: value out of range (attn_splits 0..%d, xq_path 0..2, the rest >= 0)", kTcMaxSplits);
    g_tune = *t;
    return HERALD_OK;
}

int herald_pipeline_set_debug_delay(uint32_t main_us, uint32_t retrieval_us) {
    if (main_us > 1000000u || retrieval_us > 1000000u) return fail(HERALD_ERR_INVALID_ARG, "debug delay above one second");
    g_delay_main_us = main_us;
    g_delay_retrieval_us = retrieval_us;
    return HERALD_OK;
}

int herald_pipeline_set_profile(const herald_profile_t* prof) {
    g_prof = prof;
    return HERALD_OK;
}

int herald_pipeline_step_host(herald_pipeline_t* p, const herald_host_io_t* io) {
    int rc = check_pipeline(p);
    if (rc) return rc;
    if (!io || !io->host_q_rep || !io->host_q_blk || !io->host_k_blk || !io->host_v_blk || !io->host_out)
        return fail(HERALD_ERR_INVALID_ARG, "pipeline_step_host: NULL host io");
    const bool out_alt = io->dev_out_alt != nullptr, in_alt = io->dev_q_blk_alt != nullptr;
    if ((out_alt || in_alt) && p->n_layers > 64) return fail(HERALD_ERR_INVALID_ARG, "pipeline_step_host: double buffering supports at most 64 layers");
    if (out_alt && (!io->ev_download[0] || !io->ev_download[1]))
        return fail(HERALD_ERR_INVALID_ARG, "pipeline_step_host: dev_out_alt needs both ev_download events");
    if (in_alt && (!io->dev_q_rep_alt || !io->dev_k_blk_alt || !io->dev_v_blk_alt || !io->upload_stream || !io->ev_upload[0] || !io->ev_upload[1] ||
                   !io->ev_compute[0] || !io->ev_compute[1]))
        return fail(HERALD_ERR_INVALID_ARG, "pipeline_step_host: the second input set needs all four dev_*_alt arrays, upload_stream, ev_upload[2] and ev_compute[2]");
    for (int l = 0; l < p->n_layers; ++l) {
        const bool dense = p->layers[l].dense != 0;
        if ((out_alt && !io->dev_out_alt[l]) || (!dense && !io->host_q_rep[l]) || !io->host_q_blk[l] || !io->host_k_blk[l] || !io->host_v_blk[l] || !io->host_out[l])
            return fail(HERALD_ERR_INVALID_ARG, "pipeline_step_host: layer %d has a NULL host pointer", l);
        if (in_alt && ((!dense && !io->dev_q_rep_alt[l]) || !io->dev_q_blk_alt[l] || !io->dev_k_blk_alt[l] || !io->dev_v_blk_alt[l]))
            return fail(HERALD_ERR_INVALID_ARG, "pipeline_step_host: layer %d has a NULL pointer in the second input set", l);
    }
    cudaStream_t s_main = static_cast<cudaStream_t>(p->main_stream);
    cudaStream_t s_ret = static_cast<cudaStream_t>(p->retrieval_stream);
    cudaEvent_t ev_fork = static_cast<cudaEvent_t>(p->ev_fork), ev_join = static_cast<cudaEvent_t>(p->ev_join);
    const herald_shape_t* sh = &p->shape;
    const size_t q_step = (size_t)sh->batch * sh->block_size * sh->n_q_heads * kHeadDim;
    const size_t kv_step = (size_t)sh->batch * sh->block_size * sh->n_kv_heads * kHeadDim;
    const size_t q_rep_bytes = (size_t)sh->batch * sh->n_q_heads * kHeadDim * 2;
    cudaError_t e = cudaSuccess;
    // Blocks alternate (by pipe->active) between the caller's device buffers and the optional second sets: with a second
    // OUTPUT set the attention of this block waits only for the download issued two calls ago, with a second INPUT set the
    // uploads of this block run on their own stream beside the previous block's attention -- the link is then busy in both
    // directions all the time and a block costs what its larger direction costs.
    const int parity = p->active;
    struct Saved { const void *q_rep, *q_blk, *k_blk, *v_blk; float* out; } saved[64];
    const bool swap_out = out_alt && parity == 1, swap_in = in_alt && parity == 1;
    if (swap_out || swap_in)
        for (int l = 0; l < p->n_layers; ++l) {
            herald_layer_t* ly = &p->layers[l];
            saved[l] = Saved{ly->q_rep, ly->q_blk, ly->k_blk, ly->v_blk, ly->out};
            if (swap_out) ly->out = static_cast<float*>(io->dev_out_alt[l]);
            if (swap_in) {
                ly->q_rep = io->dev_q_rep_alt[l];
                ly->q_blk = io->dev_q_blk_alt[l];
                ly->k_blk = io->dev_k_blk_alt[l];
                ly->v_blk = io->dev_v_blk_alt[l];
            }
        }
    auto restore = [&]() {
        if (swap_out || swap_in)
            for (int l = 0; l < p->n_layers; ++l) {
                herald_layer_t* ly = &p->layers[l];
                ly->q_rep = saved[l].q_rep; ly->q_blk = saved[l].q_blk; ly->k_blk = saved[l].k_blk; ly->v_blk = saved[l].v_blk; ly->out = saved[l].out;
            }
    };
    // uploads: on the main stream, or on the upload stream once the block that last read this input set has finished
    cudaStream_t s_up = in_alt ? static_cast<cudaStream_t>(io->upload_stream) : s_main;
    if (in_alt) e = cudaStreamWaitEvent(s_up, static_cast<cudaEvent_t>(io->ev_compute[parity]), 0);
    for (int l = 0; l < p->n_layers && e == cudaSuccess; ++l) {
        herald_layer_t* ly = &p->layers[l];
        if (!ly->dense)                       // a dense layer has no representative query (host_q_rep[l] may be NULL)
            e = cudaMemcpyAsync(const_cast<void*>(ly->q_rep), io->host_q_rep[l], q_rep_bytes, cudaMemcpyHostToDevice, s_up);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(const_cast<void*>(ly->q_blk), io->host_q_blk[l], q_step * p->n_steps * 2, cudaMemcpyHostToDevice, s_up);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(const_cast<void*>(ly->k_blk), io->host_k_blk[l], kv_step * p->n_steps * 2, cudaMemcpyHostToDevice, s_up);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(const_cast<void*>(ly->v_blk), io->host_v_blk[l], kv_step * p->n_steps * 2, cudaMemcpyHostToDevice, s_up);
    }
    if (e == cudaSuccess && in_alt) {
        e = cudaEventRecord(static_cast<cudaEvent_t>(io->ev_upload[parity]), s_up);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(s_main, static_cast<cudaEvent_t>(io->ev_upload[parity]), 0);
    }
    // this block's attention overwrites its output buffer: the download that last read that buffer must be done
    cudaEvent_t ev_done = out_alt ? static_cast<cudaEvent_t>(io->ev_download[parity]) : ev_join;
    if (e == cudaSuccess) e = cudaStreamWaitEvent(s_main, ev_done, 0);
    if (e != cudaSuccess) {
        restore();
        return cuda_fail(e, "H2D copy / ordering");
    }
    rc = herald_pipeline_step(p);
    if (rc == HERALD_OK) {
        // downloads go to the copy stream if there is one: on the retrieval stream the NEXT block's selection would queue behind them
        cudaStream_t s_copy = io->copy_stream ? static_cast<cudaStream_t>(io->copy_stream) : s_ret;
        e = cudaEventRecord(ev_fork, s_main);                    // this block is complete (the step joined the retrieval stream)
        if (e == cudaSuccess && in_alt) e = cudaEventRecord(static_cast<cudaEvent_t>(io->ev_compute[parity]), s_main);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(s_copy, ev_fork, 0);
        for (int l = 0; l < p->n_layers && e == cudaSuccess; ++l)
            e = cudaMemcpyAsync(io->host_out[l], p->layers[l].out, q_step * p->n_steps * sizeof(float), cudaMemcpyDeviceToHost, s_copy);
        if (e == cudaSuccess) e = cudaEventRecord(ev_done, s_copy);   // download done: a later call waits on it
        if (e != cudaSuccess) rc = cuda_fail(e, "D2H copy");
    }
    restore();
    return rc;
}

}  // extern "C"
