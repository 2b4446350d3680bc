"""Thin ctypes binding over the C-ABI library ``libherald.so`` (include/herald.h).

Argument marshalling only: every step of the hot path runs in the CUDA kernels of the library.
Importing this module loads the library and raises if it is missing -- there is no CPU fallback
and no other backend.  torch is used for device memory and streams only.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libherald.so")

if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} is missing: build it with `python -m paper_2606_21633_b200.build` "
        "(nvcc, sm_100a).  The HERALD hot path has no fallback implementation.")
_lib = C.CDLL(LIB_PATH)

OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_WORKSPACE_TOO_SMALL, ERR_CUDA = 0, -1, -2, -3, -4
AGG_MAX_LOGIT, AGG_SOFTMAX_SUM = 0, 1

EXPORTS = ("herald_last_error", "herald_set_tuning", "herald_budget_rows", "herald_select_workspace_bytes",
           "herald_attn_workspace_bytes", "herald_attn_grid_ctas", "herald_select", "herald_select_static",
           "herald_select_static_max_bytes", "herald_select_xq", "herald_gather", "herald_sparse_attn", "herald_sparse_attn_groups",
           "herald_dense_attn", "herald_rep_attn_workspace_bytes", "herald_rep_attn",
           "herald_select_rep_workspace_bytes", "herald_select_rep",
           "herald_cache_write_block", "herald_pool_append_block",
           "herald_pipeline_step", "herald_pipeline_tune", "herald_pipeline_step_host", "herald_pipeline_set_profile",
           "herald_pipeline_set_debug_delay")


class HeraldError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"herald error {code}: {msg}")
        self.code = code


class Shape(C.Structure):
    _fields_ = [("batch", C.c_int32), ("n_q_heads", C.c_int32), ("n_kv_heads", C.c_int32),
                ("head_dim", C.c_int32), ("page_size", C.c_int32), ("block_size", C.c_int32),
                ("max_seq_len", C.c_int32), ("max_pages_per_seq", C.c_int32),
                ("pool_capacity", C.c_int32), ("agg_mode", C.c_int32), ("sm_scale", C.c_float)]


class Cache(C.Structure):
    _fields_ = [("k_pages", C.c_void_p), ("v_pages", C.c_void_p), ("page_stride", C.c_int64),
                ("token_stride", C.c_int64), ("head_stride", C.c_int64),
                ("page_table", C.c_void_p), ("seq_lens", C.c_void_p)]


class Layer(C.Structure):
    _fields_ = [("cache", Cache), ("q_rep", C.c_void_p), ("k_per_seq", C.c_void_p),
                ("q_blk", C.c_void_p), ("k_blk", C.c_void_p), ("v_blk", C.c_void_p), ("out", C.c_void_p),
                ("pool_k", C.c_void_p * 2), ("pool_v", C.c_void_p * 2), ("pool_len", C.c_void_p * 2), ("dense", C.c_int32)]


class Pipeline(C.Structure):
    _fields_ = [("shape", Shape), ("n_layers", C.c_int32), ("n_steps", C.c_int32),
                ("start_after_step", C.c_int32), ("active", C.c_int32), ("scan_ctas", C.c_int32),
                ("scan_head_permille", C.c_int32), ("layers", C.POINTER(Layer)),
                ("sel_idx", C.c_void_p), ("ws_select", C.c_void_p), ("ws_select_bytes", C.c_size_t),
                ("ws_attn", C.c_void_p), ("ws_attn_bytes", C.c_size_t),
                ("main_stream", C.c_void_p), ("retrieval_stream", C.c_void_p),
                ("ev_fork", C.c_void_p), ("ev_join", C.c_void_p)]


class Schedule(C.Structure):
    _fields_ = [("scan_ctas", C.c_int32), ("start_after_step", C.c_int32), ("scan_head_permille", C.c_int32),
                ("ms_per_step", C.c_float)]


class HostIO(C.Structure):
    _fields_ = [("host_q_rep", C.POINTER(C.c_void_p)), ("host_q_blk", C.POINTER(C.c_void_p)),
                ("host_k_blk", C.POINTER(C.c_void_p)), ("host_v_blk", C.POINTER(C.c_void_p)),
                ("host_out", C.POINTER(C.c_void_p)), ("dev_out_alt", C.POINTER(C.c_void_p)), ("ev_download", C.c_void_p * 2), ("copy_stream", C.c_void_p),
                ("dev_q_rep_alt", C.POINTER(C.c_void_p)), ("dev_q_blk_alt", C.POINTER(C.c_void_p)),
                ("dev_k_blk_alt", C.POINTER(C.c_void_p)), ("dev_v_blk_alt", C.POINTER(C.c_void_p)),
                ("upload_stream", C.c_void_p), ("ev_upload", C.c_void_p * 2), ("ev_compute", C.c_void_p * 2)]


class Tuning(C.Structure):
    _fields_ = [("attn_splits", C.c_int32), ("attn_m_tiles", C.c_int32), ("attn_total_ctas", C.c_int32),
                ("attn_no_pdl", C.c_int32), ("scan_ctas", C.c_int32), ("scan_head_major", C.c_int32), ("xq_path", C.c_int32), ("attn_precision", C.c_int32)]


XQ_AUTO, XQ_MMA_SYNC, XQ_TCGEN05 = 0, 1, 2
ATTN_AUTO, ATTN_EXACT, ATTN_FAST_FIRST = 0, 1, 2


class Profile(C.Structure):
    _fields_ = [("scan_begin", C.c_void_p), ("scan_end", C.c_void_p), ("topk_end", C.c_void_p),
                ("gather_end", C.c_void_p)]


_lib.herald_last_error.restype = C.c_char_p
_lib.herald_last_error.argtypes = []
_lib.herald_budget_rows.restype = C.c_int32
_lib.herald_budget_rows.argtypes = [C.c_int32, C.c_int32]
_lib.herald_select_workspace_bytes.restype = C.c_size_t
_lib.herald_select_workspace_bytes.argtypes = [C.POINTER(Shape)]
_lib.herald_attn_workspace_bytes.restype = C.c_size_t
_lib.herald_attn_workspace_bytes.argtypes = [C.POINTER(Shape)]
_lib.herald_attn_grid_ctas.restype = C.c_int32
_lib.herald_attn_grid_ctas.argtypes = [C.POINTER(Shape)]
_lib.herald_select.restype = C.c_int
_lib.herald_select.argtypes = [C.POINTER(Shape), C.POINTER(Cache), C.c_void_p, C.c_void_p, C.c_void_p,
                               C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
_lib.herald_select_static_max_bytes.restype = C.c_size_t
_lib.herald_select_static_max_bytes.argtypes = []
_lib.herald_select_static.restype = C.c_int
_lib.herald_select_static.argtypes = [C.POINTER(Shape), C.POINTER(Cache), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.herald_select_xq.restype = C.c_int
_lib.herald_select_xq.argtypes = [C.POINTER(Shape), C.POINTER(Cache), C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p,
                                  C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
_lib.herald_gather.restype = C.c_int
_lib.herald_gather.argtypes = [C.POINTER(Shape), C.POINTER(Cache), C.c_void_p, C.c_void_p, C.c_void_p,
                               C.c_void_p, C.c_void_p]
_lib.herald_sparse_attn.restype = C.c_int
_lib.herald_sparse_attn.argtypes = [C.POINTER(Shape)] + [C.c_void_p] * 9 + [C.c_size_t, C.c_void_p]
_lib.herald_sparse_attn_groups.restype = C.c_int
_lib.herald_sparse_attn_groups.argtypes = [C.POINTER(Shape), C.c_int32] + [C.c_void_p] * 9 + [C.c_size_t, C.c_void_p]
_lib.herald_dense_attn.restype = C.c_int
_lib.herald_dense_attn.argtypes = [C.POINTER(Shape), C.POINTER(Cache)] + [C.c_void_p] * 6 + [C.c_size_t, C.c_void_p]
_lib.herald_rep_attn_workspace_bytes.restype = C.c_size_t
_lib.herald_rep_attn_workspace_bytes.argtypes = [C.POINTER(Shape)]
_lib.herald_rep_attn.restype = C.c_int
_lib.herald_rep_attn.argtypes = [C.POINTER(Shape), C.POINTER(Cache), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t,
                                 C.c_void_p]
_lib.herald_select_rep_workspace_bytes.restype = C.c_size_t
_lib.herald_select_rep_workspace_bytes.argtypes = [C.POINTER(Shape)]
_lib.herald_select_rep.restype = C.c_int
_lib.herald_select_rep.argtypes = [C.POINTER(Shape), C.POINTER(Cache)] + [C.c_void_p] * 8 + [C.c_size_t, C.c_void_p]
_lib.herald_cache_write_block.restype = C.c_int
_lib.herald_cache_write_block.argtypes = [C.POINTER(Shape), C.POINTER(Cache), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.herald_pool_append_block.restype = C.c_int
_lib.herald_pool_append_block.argtypes = [C.POINTER(Shape)] + [C.c_void_p] * 6
_lib.herald_pipeline_step.restype = C.c_int
_lib.herald_pipeline_step.argtypes = [C.POINTER(Pipeline)]
_lib.herald_pipeline_tune.restype = C.c_int
_lib.herald_pipeline_tune.argtypes = [C.POINTER(Pipeline), C.c_int32, C.POINTER(Schedule), C.c_int32, C.POINTER(C.c_int32)]
_lib.herald_pipeline_step_host.restype = C.c_int
_lib.herald_pipeline_step_host.argtypes = [C.POINTER(Pipeline), C.POINTER(HostIO)]


def _ptr(t):
    if t is None:
        return None
    if isinstance(t, int):
        return t
    return t.data_ptr()


def _stream(stream):
    if stream is None:
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def _ws(ws):
    """workspace: a torch uint8 tensor, or a (device_pointer, nbytes) tuple."""
    if ws is None:
        return None, 0
    if isinstance(ws, tuple):
        return int(ws[0]), int(ws[1])
    return ws.data_ptr(), ws.numel() * ws.element_size()


def _check(rc):
    if rc != 0:
        raise HeraldError(rc, _lib.herald_last_error().decode())


_lib.herald_set_tuning.restype = C.c_int
_lib.herald_set_tuning.argtypes = [C.POINTER(Tuning)]


def herald_set_tuning(**fields):
    """Launch-geometry overrides for the following calls of this thread; no arguments = the defaults."""
    if not fields:
        _check(_lib.herald_set_tuning(None))
    else:
        t = Tuning(**fields)
        _check(_lib.herald_set_tuning(C.byref(t)))


def herald_last_error() -> str:
    return _lib.herald_last_error().decode()


def herald_budget_rows(seq_len: int, permille: int) -> int:
    return int(_lib.herald_budget_rows(int(seq_len), int(permille)))


def make_shape(batch, n_q_heads, n_kv_heads, block_size, max_seq_len, max_pages_per_seq, pool_capacity,
               agg_mode=AGG_MAX_LOGIT, sm_scale=None, head_dim=128, page_size=16) -> Shape:
    if sm_scale is None:
        sm_scale = head_dim ** -0.5
    return Shape(batch, n_q_heads, n_kv_heads, head_dim, page_size, block_size, max_seq_len,
                 max_pages_per_seq, pool_capacity, agg_mode, sm_scale)


def make_cache(k_pages, v_pages, page_table, seq_lens) -> Cache:
    """k_pages / v_pages: bf16 [n_pages, page, H_kv, d] torch tensors (any strides with contiguous rows)."""
    assert k_pages.stride(3) == 1 and (v_pages is None or v_pages.stride() == k_pages.stride())
    return Cache(_ptr(k_pages), _ptr(v_pages), k_pages.stride(0), k_pages.stride(1), k_pages.stride(2),
                 _ptr(page_table), _ptr(seq_lens))


def herald_select_workspace_bytes(shape: Shape) -> int:
    return int(_lib.herald_select_workspace_bytes(C.byref(shape)))


def herald_attn_workspace_bytes(shape: Shape) -> int:
    return int(_lib.herald_attn_workspace_bytes(C.byref(shape)))


def herald_attn_grid_ctas(shape: Shape) -> int:
    return int(_lib.herald_attn_grid_ctas(C.byref(shape)))


def herald_select(shape, cache, q_rep, k_per_seq, sel_idx, sel_cnt, scores_out, ws, stream=None):
    ws_ptr, ws_bytes = _ws(ws)
    _check(_lib.herald_select(C.byref(shape), C.byref(cache), _ptr(q_rep), _ptr(k_per_seq), _ptr(sel_idx),
                              _ptr(sel_cnt), _ptr(scores_out), ws_ptr, ws_bytes, _stream(stream)))


def herald_select_static_max_bytes() -> int:
    return int(_lib.herald_select_static_max_bytes())


def herald_select_static(shape, cache, q_rep, k_per_seq, sel_idx, sel_cnt, stream=None):
    """herald_select with the workspace held inside the library (no allocation anywhere; include/herald.h)."""
    _check(_lib.herald_select_static(C.byref(shape), C.byref(cache), _ptr(q_rep), _ptr(k_per_seq), _ptr(sel_idx),
                                     _ptr(sel_cnt), _stream(stream)))


def herald_select_xq(shape, cache, q_x, x, k_per_seq, sel_idx, sel_cnt, scores_out, ws, stream=None):
    ws_ptr, ws_bytes = _ws(ws)
    _check(_lib.herald_select_xq(C.byref(shape), C.byref(cache), _ptr(q_x), int(x), _ptr(k_per_seq), _ptr(sel_idx),
                                 _ptr(sel_cnt), _ptr(scores_out), ws_ptr, ws_bytes, _stream(stream)))


def herald_gather(shape, cache, sel_idx, sel_cnt, pool_k, pool_v, stream=None):
    _check(_lib.herald_gather(C.byref(shape), C.byref(cache), _ptr(sel_idx), _ptr(sel_cnt), _ptr(pool_k),
                              _ptr(pool_v), _stream(stream)))


def herald_sparse_attn_groups(shape, n_groups, pool_k, pool_v, pool_len, q_blk, k_blk, v_blk, out, lse, ws, stream=None):
    ws_ptr, ws_bytes = _ws(ws)
    _check(_lib.herald_sparse_attn_groups(C.byref(shape), int(n_groups), _ptr(pool_k), _ptr(pool_v), _ptr(pool_len), _ptr(q_blk),
                                          _ptr(k_blk), _ptr(v_blk), _ptr(out), _ptr(lse), ws_ptr, ws_bytes, _stream(stream)))


def herald_sparse_attn(shape, pool_k, pool_v, pool_len, q_blk, k_blk, v_blk, out, lse, ws, stream=None):
    ws_ptr, ws_bytes = _ws(ws)
    _check(_lib.herald_sparse_attn(C.byref(shape), _ptr(pool_k), _ptr(pool_v), _ptr(pool_len), _ptr(q_blk),
                                   _ptr(k_blk), _ptr(v_blk), _ptr(out), _ptr(lse), ws_ptr, ws_bytes,
                                   _stream(stream)))


def herald_dense_attn(shape, cache, q_blk, k_blk, v_blk, out, lse, ws, stream=None):
    ws_ptr, ws_bytes = _ws(ws)
    _check(_lib.herald_dense_attn(C.byref(shape), C.byref(cache), _ptr(q_blk), _ptr(k_blk), _ptr(v_blk), _ptr(out),
                                  _ptr(lse), ws_ptr, ws_bytes, _stream(stream)))


def herald_select_rep_workspace_bytes(shape: Shape) -> int:
    return int(_lib.herald_select_rep_workspace_bytes(C.byref(shape)))


def herald_select_rep(shape, cache, q_rep, k_per_seq, sel_idx, sel_cnt, scores_out, rep_out, rep_lse, ws, stream=None):
    ws_ptr, ws_bytes = _ws(ws)
    _check(_lib.herald_select_rep(C.byref(shape), C.byref(cache), _ptr(q_rep), _ptr(k_per_seq), _ptr(sel_idx), _ptr(sel_cnt),
                                  _ptr(scores_out), _ptr(rep_out), _ptr(rep_lse), ws_ptr, ws_bytes, _stream(stream)))


def herald_rep_attn_workspace_bytes(shape: Shape) -> int:
    return int(_lib.herald_rep_attn_workspace_bytes(C.byref(shape)))


def herald_rep_attn(shape, cache, q_rep, out, lse, ws, stream=None):
    ws_ptr, ws_bytes = _ws(ws)
    _check(_lib.herald_rep_attn(C.byref(shape), C.byref(cache), _ptr(q_rep), _ptr(out), _ptr(lse), ws_ptr, ws_bytes,
                                _stream(stream)))


def herald_cache_write_block(shape, cache, write_pos, k_new, v_new, stream=None):
    _check(_lib.herald_cache_write_block(C.byref(shape), C.byref(cache), _ptr(write_pos), _ptr(k_new), _ptr(v_new), _stream(stream)))


def herald_pool_append_block(shape, pool_k, pool_v, pool_len, k_new, v_new, stream=None):
    _check(_lib.herald_pool_append_block(C.byref(shape), _ptr(pool_k), _ptr(pool_v), _ptr(pool_len), _ptr(k_new), _ptr(v_new),
                                         _stream(stream)))


def herald_pipeline_step(pipe: Pipeline):
    _check(_lib.herald_pipeline_step(C.byref(pipe)))


def herald_pipeline_step_host(pipe: Pipeline, io: HostIO):
    _check(_lib.herald_pipeline_step_host(C.byref(pipe), C.byref(io)))


_lib.herald_pipeline_set_profile.restype = C.c_int
_lib.herald_pipeline_set_profile.argtypes = [C.POINTER(Profile)]


def herald_pipeline_set_profile(prof):
    """prof: a Profile struct (kept alive by the caller) or None."""
    _check(_lib.herald_pipeline_set_profile(C.byref(prof) if prof is not None else None))


_lib.herald_pipeline_set_debug_delay.restype = C.c_int
_lib.herald_pipeline_set_debug_delay.argtypes = [C.c_uint32, C.c_uint32]


def herald_pipeline_set_debug_delay(main_us: int, retrieval_us: int):
    """Test hook: idle kernels on the main / retrieval stream inside the following pipeline steps (0, 0 = off)."""
    _check(_lib.herald_pipeline_set_debug_delay(int(main_us), int(retrieval_us)))


def alloc_workspace(nbytes: int, device) -> torch.Tensor:
    """256-byte aligned device scratch (torch's caching allocator aligns to 512 B)."""
    return torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=device)


class BlockPipeline:
    """Owns the device buffers of a dual-stream block pipeline (pools, workspaces, streams, events)
    and the ctypes structs that describe them.  Marshalling and memory ownership only."""

    def __init__(self, shape: Shape, layers, n_steps: int, start_after_step: int = 0, device="cuda", scan_ctas=None,
                 scan_head_permille: int = 0):
        """layers: list of dicts with torch tensors k_pages, v_pages, page_table, seq_lens, q_rep, k_per_seq,
        q_blk, k_blk, v_blk ([n_steps, ...]); optional "dense": True for a layer that keeps its full KV."""
        dev = torch.device(device)
        self.shape, self.n_steps, self.device = shape, n_steps, dev
        units, cap = shape.batch * shape.n_kv_heads, shape.pool_capacity
        self.keep = []
        self.layer_arr = (Layer * len(layers))()
        self.outs, self.pools_k, self.pools_v, self.pool_lens = [], [], [], []
        for i, ly in enumerate(layers):
            out = torch.empty((n_steps, shape.batch, shape.block_size, shape.n_q_heads, 128), dtype=torch.float32, device=dev)
            rows = 1 if ly.get("dense") else cap          # a dense layer has no pools: placeholders
            pk = [torch.zeros((shape.batch, shape.n_kv_heads, rows, 128), dtype=torch.bfloat16, device=dev) for _ in range(2)]
            pv = [torch.zeros((shape.batch, shape.n_kv_heads, rows, 128), dtype=torch.bfloat16, device=dev) for _ in range(2)]
            pl = [torch.zeros((shape.batch, shape.n_kv_heads), dtype=torch.int32, device=dev) for _ in range(2)]
            L = self.layer_arr[i]
            L.cache = make_cache(ly["k_pages"], ly["v_pages"], ly["page_table"], ly["seq_lens"])
            L.q_rep, L.k_per_seq = _ptr(ly["q_rep"]), _ptr(ly["k_per_seq"])
            L.q_blk, L.k_blk, L.v_blk, L.out = _ptr(ly["q_blk"]), _ptr(ly["k_blk"]), _ptr(ly["v_blk"]), _ptr(out)
            L.dense = 1 if ly.get("dense") else 0
            for j in range(2):
                L.pool_k[j], L.pool_v[j], L.pool_len[j] = _ptr(pk[j]), _ptr(pv[j]), _ptr(pl[j])
            self.outs.append(out)
            self.pools_k.append(pk)
            self.pools_v.append(pv)
            self.pool_lens.append(pl)
            self.keep.append(ly)
        self.sel_idx = torch.zeros((max(units, 1), max(cap, 1)), dtype=torch.int32, device=dev)
        self.ws_select = alloc_workspace(herald_select_workspace_bytes(shape), dev)
        self.ws_attn = alloc_workspace(herald_attn_workspace_bytes(shape) * max(len(layers), 1), dev)   # one slice per layer
        self.main_stream = torch.cuda.Stream(device=dev, priority=-1)
        self.retrieval_stream = torch.cuda.Stream(device=dev, priority=0)
        self.ev_fork, self.ev_join = torch.cuda.Event(), torch.cuda.Event()
        with torch.cuda.device(dev):
            self.ev_fork.record(self.main_stream)      # materialises the cudaEvent_t handles
            self.ev_join.record(self.retrieval_stream)
        p = Pipeline()
        p.shape, p.n_layers, p.n_steps, p.start_after_step, p.active = shape, len(layers), n_steps, start_after_step, 0
        if scan_ctas is None:
            scan_ctas = 0          # the library's default: the SMs the attention grid leaves free
        p.scan_ctas = int(scan_ctas)
        p.scan_head_permille = int(scan_head_permille)
        p.layers = C.cast(self.layer_arr, C.POINTER(Layer))
        p.sel_idx = _ptr(self.sel_idx)
        p.ws_select, p.ws_select_bytes = _ptr(self.ws_select), self.ws_select.numel()
        p.ws_attn, p.ws_attn_bytes = _ptr(self.ws_attn), self.ws_attn.numel()
        p.main_stream, p.retrieval_stream = self.main_stream.cuda_stream, self.retrieval_stream.cuda_stream
        p.ev_fork, p.ev_join = self.ev_fork.cuda_event, self.ev_join.cuda_event
        self.c = p

    @property
    def active(self) -> int:
        return int(self.c.active)

    def step(self):
        herald_pipeline_step(self.c)

    def make_host_io(self, host_layers, double_buffer=True) -> HostIO:
        """host_layers: list of dicts of PINNED host tensors q_rep, q_blk, k_blk, v_blk, out.  double_buffer: a second set of
        device output buffers, so that a block's attention runs beside the previous block's download."""
        n = len(host_layers)
        io = HostIO()
        self._io_arrays = []
        if double_buffer:
            self.outs_alt = [torch.empty_like(o) for o in self.outs]
            alt = (C.c_void_p * n)(*[o.data_ptr() for o in self.outs_alt])
            self._io_arrays.append(alt)
            io.dev_out_alt = C.cast(alt, C.POINTER(C.c_void_p))
            self._ev_download = [torch.cuda.Event(), torch.cuda.Event()]
            with torch.cuda.device(self.device):
                for i, e in enumerate(self._ev_download):
                    e.record(self.retrieval_stream)          # materialises the cudaEvent_t handles
                    io.ev_download[i] = e.cuda_event
            self.copy_stream = torch.cuda.Stream(device=self.device)
            io.copy_stream = self.copy_stream.cuda_stream
            # second set of device inputs + an upload stream: the uploads of a block run beside the previous block's attention
            self.ins_alt = {}
            for name in ("q_rep", "q_blk", "k_blk", "v_blk"):
                bufs = [torch.empty_like(ly[name]) if not (name == "q_rep" and ly.get("dense")) else None for ly in self.keep]
                self.ins_alt[name] = bufs
                arr = (C.c_void_p * n)(*[b.data_ptr() if b is not None else None for b in bufs])
                self._io_arrays.append(arr)
                setattr(io, f"dev_{name}_alt", C.cast(arr, C.POINTER(C.c_void_p)))
            self.upload_stream = torch.cuda.Stream(device=self.device)
            io.upload_stream = self.upload_stream.cuda_stream
            self._ev_io = [torch.cuda.Event() for _ in range(4)]
            with torch.cuda.device(self.device):
                for i, e in enumerate(self._ev_io):
                    e.record(self.main_stream)
                    (io.ev_upload if i < 2 else io.ev_compute)[i % 2] = e.cuda_event
        for name in ("q_rep", "q_blk", "k_blk", "v_blk", "out"):
            arr = (C.c_void_p * n)(*[h[name].data_ptr() for h in host_layers])
            self._io_arrays.append(arr)
            setattr(io, "host_" + name, C.cast(arr, C.POINTER(C.c_void_p)))
        self._host_layers = host_layers
        return io

    def step_host(self, io: HostIO):
        herald_pipeline_step_host(self.c, io)

    def tune_schedule(self, reps=4):
        """herald_pipeline_tune: times a handful of schedules (scan grid, start step, head start of the scan) with eager block
        steps outside any timed region and leaves the fastest one set.  Returns {"scan_ctas/start/head_permille": ms per step}."""
        table = (Schedule * 32)()
        n = C.c_int32(0)
        _check(_lib.herald_pipeline_tune(C.byref(self.c), int(reps), table, 32, C.byref(n)))
        return {f"{t.scan_ctas}/{t.start_after_step}/{t.scan_head_permille}": t.ms_per_step for t in table[:n.value]}

    # ---- CUDA graphs: one captured block step per pool parity (launch-bound inner loop, no per-launch host cost) ----
    def capture(self):
        """Capture herald_pipeline_step twice, once per value of ``active``, into two CUDA graphs whose root is the main
        stream; the retrieval stream joins the capture through the fork/join events.  Run at least one eager step first
        (function attributes and tensor maps are set up on first use).  herald_pipeline_step_host is eager-only: it orders
        itself after the previous call's download through an event recorded outside any capture."""
        graphs = {}
        start = self.active
        for _ in range(2):
            parity = self.active
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=self.main_stream, capture_error_mode="thread_local"):
                herald_pipeline_step(self.c)
            graphs[parity] = g                      # the capture flipped ->active exactly like an eager step
        assert self.active == start
        return graphs

    def replay(self, graphs):
        """Launch the captured step for the current parity on the main stream and flip ``active``."""
        with torch.cuda.stream(self.main_stream):
            graphs[self.active].replay()
        self.c.active = 1 - self.c.active
