"""CPU-side checks of the C-ABI boundary: the library builds/loads, exports every symbol that
include/herald.h declares, and its host-only logic (budget, workspace sizes, argument checks that
fail before any CUDA call) behaves as documented.  No GPU compute here."""
import ctypes as C
import os
import re

import pytest

from oracle import herald_oracle as O

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def H():
    from paper_2606_21633_b200 import build
    build.build()
    from paper_2606_21633_b200 import herald
    return herald


def declared_functions():
    text = open(os.path.join(ROOT, "include", "herald.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    text = re.sub(r"#ifdef HERALD_ATTN_TRACE.*?#endif", "", text, flags=re.S)      # debug builds only, not in the release ABI
    return sorted(set(re.findall(r"\b(herald_[a-z_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(H):
    names = declared_functions()
    assert len(names) >= 9
    lib = C.CDLL(H.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), f"{n} is declared in include/herald.h but not exported"
    assert set(names) == set(H.EXPORTS)


def test_budget_rows_matches_oracle_and_golden(H):
    for L in list(range(0, 70)) + [4096, 32768, 65536, 131072, 99999]:
        for pm in (0, 1, 25, 50, 100, 175, 500, 999, 1000):
            assert H.herald_budget_rows(L, pm) == O.budget_rows(L, pm)
    assert H.herald_budget_rows(4096, 50) == 205 and H.herald_budget_rows(32768, 50) == 1639
    assert H.herald_budget_rows(-1, 50) == -1 and H.herald_budget_rows(10, 1001) == -1


def test_workspace_sizes(H):
    s = H.make_shape(8, 28, 4, 32, 32768, 2048, 1639 + 32)
    sel, att = H.herald_select_workspace_bytes(s), H.herald_attn_workspace_bytes(s)
    assert sel >= 32 * 4096 * 4 + 32 * 32768 * 4      # level-1 histograms + score plane
    assert att >= 256
    s1 = H.make_shape(8, 28, 4, 32, 32768, 2048, 1639 + 32, agg_mode=1)
    assert H.herald_select_workspace_bytes(s1) >= sel + 32 * 7 * 32768 * 4   # raw per-head scores
    bad = H.make_shape(8, 28, 4, 32, 32768, 2048, 100, head_dim=64)
    assert H.herald_select_workspace_bytes(bad) == 0


@pytest.mark.parametrize("kw,code", [
    (dict(head_dim=64), -2), (dict(page_size=32), -2), (dict(n_q_heads=36), -2), (dict(n_q_heads=30), -1),
    (dict(block_size=128), -2), (dict(max_seq_len=1000), -1), (dict(agg_mode=3), -1), (dict(sm_scale=0.0), -1),
    (dict(max_pages_per_seq=1), -1),
])
def test_invalid_shapes_are_rejected_before_any_cuda_call(H, kw, code):
    base = dict(batch=2, n_q_heads=8, n_kv_heads=4, block_size=16, max_seq_len=1024, max_pages_per_seq=64, pool_capacity=64)
    base.update(kw)
    shape = H.make_shape(**base)
    cache = H.Cache(256, 256, 16 * 4 * 128, 4 * 128, 128, 256, 256)
    with pytest.raises(H.HeraldError) as ei:
        H.herald_select(shape, cache, 256, 256, 256, 256, None, (256, 1 << 30), stream=0)
    assert ei.value.code == code and H.herald_last_error() != ""


def test_null_and_misaligned_pointers_are_rejected(H):
    shape = H.make_shape(2, 8, 4, 16, 1024, 64, 64)
    cache = H.Cache(256, 256, 16 * 4 * 128, 4 * 128, 128, 256, 256)
    with pytest.raises(H.HeraldError) as ei:
        H.herald_select(shape, cache, None, 256, 256, 256, None, (256, 1 << 30), stream=0)
    assert ei.value.code == H.ERR_INVALID_ARG
    with pytest.raises(H.HeraldError) as ei:
        H.herald_gather(shape, cache, 256, 256, 264, 256, stream=0)       # pool_k not 16-byte aligned
    assert ei.value.code == H.ERR_INVALID_ARG
    bad_cache = H.Cache(256, 256, 16 * 4 * 128, 4 * 128 + 4, 128, 256, 256)
    with pytest.raises(H.HeraldError) as ei:
        H.herald_gather(shape, bad_cache, 256, 256, 256, 256, stream=0)
    assert ei.value.code == H.ERR_INVALID_ARG


def test_workspace_too_small_is_reported(H):
    shape = H.make_shape(2, 8, 4, 16, 1024, 64, 64)
    cache = H.Cache(256, 256, 16 * 4 * 128, 4 * 128, 128, 256, 256)
    with pytest.raises(H.HeraldError) as ei:       # the size check fails before any device access
        H.herald_select(shape, cache, 256, 256, 256, 256, None, (4096, 256), stream=0)
    assert ei.value.code == H.ERR_WORKSPACE_TOO_SMALL


def test_follow_up_entries_check_their_arguments_before_any_cuda_call(H):
    """herald_select_xq / herald_select_rep / herald_rep_attn / herald_sparse_attn_groups: NULL pointers, a query count out of
    range, a workspace that is too small and a bad group count are reported without touching the device."""
    shape = H.make_shape(2, 8, 4, 16, 1024, 64, 64)
    cache = H.Cache(256, 256, 16 * 4 * 128, 4 * 128, 128, 256, 256)
    big = (256, 1 << 30)
    cases = [
        (lambda: H.herald_select_xq(shape, cache, None, 2, 256, 256, 256, None, big, stream=0), H.ERR_INVALID_ARG),
        (lambda: H.herald_select_xq(shape, cache, 256, 0, 256, 256, 256, None, big, stream=0), H.ERR_INVALID_ARG),
        (lambda: H.herald_select_xq(shape, cache, 256, 129, 256, 256, 256, None, big, stream=0), H.ERR_INVALID_ARG),     # 129 x G=2 > 256 rows
        (lambda: H.herald_select_xq(shape, cache, 256, 2, 256, 256, 256, None, (256, 256), stream=0), H.ERR_WORKSPACE_TOO_SMALL),
        (lambda: H.herald_select_rep(shape, cache, 256, 256, 256, 256, None, None, None, big, stream=0), H.ERR_INVALID_ARG),   # rep_out NULL
        (lambda: H.herald_select_rep(shape, cache, 256, 256, 256, 256, None, 256, None, (256, 256), stream=0), H.ERR_WORKSPACE_TOO_SMALL),
        (lambda: H.herald_rep_attn(shape, cache, 256, None, None, big, stream=0), H.ERR_INVALID_ARG),
        (lambda: H.herald_rep_attn(shape, cache, 256, 256, None, (256, 256), stream=0), H.ERR_WORKSPACE_TOO_SMALL),
        (lambda: H.herald_sparse_attn_groups(shape, 0, 256, 256, 256, 256, 256, 256, 256, None, big, stream=0), H.ERR_INVALID_ARG),
        (lambda: H.herald_sparse_attn_groups(shape, 2, 256, 256, None, 256, 256, 256, 256, None, big, stream=0), H.ERR_INVALID_ARG),
    ]
    for i, (call, code) in enumerate(cases):
        with pytest.raises(H.HeraldError) as ei:
            call()
        assert ei.value.code == code, (i, ei.value.code, str(ei.value))
    # the fused entry needs both workspaces and a log-sum-exp plane
    assert H.herald_select_rep_workspace_bytes(shape) > H.herald_select_workspace_bytes(shape) + H.herald_rep_attn_workspace_bytes(shape) - 256
    shape1 = H.make_shape(2, 8, 4, 16, 1024, 64, 64, 1)
    with pytest.raises(H.HeraldError) as ei:          # x queries: the aggregation is only defined for max-logit (reading 25)
        H.herald_select_xq(shape1, cache, 256, 2, 256, 256, 256, None, big, stream=0)
    assert ei.value.code == H.ERR_INVALID_ARG


def test_tuning_struct_is_the_only_knob(H):
    """No environment variable is read by the library (no env-var magic); geometry overrides go
    through herald_set_tuning, are validated, and change the attention grid the size query reports."""
    src = open(os.path.join(ROOT, "paper_2606_21633_b200", "csrc", "herald_api.cu")).read()
    assert "getenv" not in src
    shape = H.make_shape(8, 28, 4, 32, 32768, 2048, 1639 + 32)
    try:
        base = H.herald_attn_grid_ctas(shape)
        assert base == 128                                   # 2 KV splits x 2 M tiles x 32 units on 148 SMs
        H.herald_set_tuning(attn_splits=1)
        assert H.herald_attn_grid_ctas(shape) == 64
        H.herald_set_tuning(attn_splits=4)
        assert H.herald_attn_grid_ctas(shape) == 256
        for bad in (dict(attn_splits=9), dict(attn_splits=-1), dict(xq_path=3), dict(scan_ctas=-2)):
            with pytest.raises(H.HeraldError) as ei:
                H.herald_set_tuning(**bad)
            assert ei.value.code == H.ERR_INVALID_ARG
        assert H.herald_attn_grid_ctas(shape) == 256         # a rejected call changes nothing
    finally:
        H.herald_set_tuning()
    assert H.herald_attn_grid_ctas(shape) == base


def test_too_many_units_is_unsupported(H):
    shape = H.make_shape(20000, 8, 4, 16, 1024, 64, 64)      # 80000 (sequence, KV head) units > 65535
    assert H.herald_select_workspace_bytes(shape) == 0
    cache = H.Cache(256, 256, 16 * 4 * 128, 4 * 128, 128, 256, 256)
    with pytest.raises(H.HeraldError) as ei:
        H.herald_gather(shape, cache, 256, 256, 256, 256, stream=0)
    assert ei.value.code == H.ERR_UNSUPPORTED


def test_pipeline_arguments_are_validated_before_anything_is_enqueued(H):
    shape = H.make_shape(2, 8, 4, 16, 1024, 64, 64)
    layers = (H.Layer * 1)()
    ly = layers[0]
    ly.cache = H.Cache(256, 256, 16 * 4 * 128, 4 * 128, 128, 256, 256)
    ly.q_rep = ly.k_per_seq = ly.q_blk = ly.k_blk = ly.v_blk = ly.out = 256
    for j in range(2):
        ly.pool_k[j] = ly.pool_v[j] = ly.pool_len[j] = 256
    p = H.Pipeline()
    p.shape, p.n_layers, p.n_steps, p.start_after_step, p.active, p.scan_ctas, p.scan_head_permille = shape, 1, 3, 0, 0, 0, 0
    p.layers = C.cast(layers, C.POINTER(H.Layer))
    p.sel_idx = p.ws_select = p.ws_attn = 256
    p.ws_select_bytes = p.ws_attn_bytes = 1 << 30
    p.main_stream, p.retrieval_stream, p.ev_fork, p.ev_join = 1, 2, 256, 256
    def expect(code):
        with pytest.raises(H.HeraldError) as ei:
            H.herald_pipeline_step(p)
        assert ei.value.code == code, str(ei.value)
        assert p.active == 0                                  # a rejected step does not swap the pools
    p.scan_head_permille = 1001
    expect(H.ERR_INVALID_ARG)
    p.scan_head_permille = 0
    p.start_after_step = 4
    expect(H.ERR_INVALID_ARG)
    p.start_after_step = 0
    ly.pool_v[1] = None                                       # a sparse layer needs both pool buffers ...
    expect(H.ERR_INVALID_ARG)
    ly.dense = 1                                              # ... a dense one does not, but still its block tensors
    ly.out = None
    expect(H.ERR_INVALID_ARG)
    p.retrieval_stream = 1
    expect(H.ERR_INVALID_ARG)


def test_host_io_double_buffering_is_validated(H):
    """herald_pipeline_step_host: the optional second buffer sets need their streams and events; nothing is enqueued otherwise."""
    shape = H.make_shape(2, 8, 4, 16, 1024, 64, 64)
    layers = (H.Layer * 1)()
    ly = layers[0]
    ly.cache = H.Cache(256, 256, 16 * 4 * 128, 4 * 128, 128, 256, 256)
    ly.q_rep = ly.k_per_seq = ly.q_blk = ly.k_blk = ly.v_blk = ly.out = 256
    for j in range(2):
        ly.pool_k[j] = ly.pool_v[j] = ly.pool_len[j] = 256
    p = H.Pipeline()
    p.shape, p.n_layers, p.n_steps, p.start_after_step, p.active = shape, 1, 3, 0, 0
    p.layers = C.cast(layers, C.POINTER(H.Layer))
    p.sel_idx = p.ws_select = p.ws_attn = 256
    p.ws_select_bytes = p.ws_attn_bytes = 1 << 30
    p.main_stream, p.retrieval_stream, p.ev_fork, p.ev_join = 1, 2, 256, 256
    one = (C.c_void_p * 1)(256)
    ptrs = C.cast(one, C.POINTER(C.c_void_p))
    io = H.HostIO()
    io.host_q_rep = io.host_q_blk = io.host_k_blk = io.host_v_blk = io.host_out = ptrs
    def expect_invalid():
        with pytest.raises(H.HeraldError) as ei:
            H.herald_pipeline_step_host(p, io)
        assert ei.value.code == H.ERR_INVALID_ARG, str(ei.value)
        assert p.active == 0
    io.dev_out_alt = ptrs                    # a second output set without its events
    expect_invalid()
    io.ev_download[0] = io.ev_download[1] = 256
    io.dev_q_blk_alt = ptrs                  # a second input set without the other arrays / the upload stream
    expect_invalid()
    io.dev_q_rep_alt = io.dev_k_blk_alt = io.dev_v_blk_alt = ptrs
    expect_invalid()                         # ... still no upload stream and events
    io.host_out = C.cast((C.c_void_p * 1)(None), C.POINTER(C.c_void_p))
    io.dev_out_alt = None
    io.dev_q_blk_alt = None
    expect_invalid()                         # a NULL host pointer for layer 0
