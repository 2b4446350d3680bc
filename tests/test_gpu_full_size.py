"""GPU parity at BASELINE.json's full sizes (oracle-coverage table) and the schedule-independence
of the block step.  The oracle sees exactly the bytes of the sampled units; everything else is checked through properties
(counts, canaries, bit equality of pools).  Run with -m gpu on a B200."""
import numpy as np
import pytest
import torch

from oracle import herald_oracle as O
from paper_2606_21633_b200 import synth
from parity_util import ATTN_TOL, check_selection

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def H():
    from paper_2606_21633_b200 import herald
    return herald


def _seed(name, layer=0):
    return 21633 + 1000 * int(name[1]) + 97 * layer


def _shape(H, w, inp, cap, agg_mode=0):
    return H.make_shape(w.batch, w.n_q_heads, w.n_kv_heads, w.block_size, (w.max_seq_len + 15) // 16 * 16,
                        inp["page_table"].shape[1], cap, agg_mode)


def _seq_view(inp, b, L, cuda):
    """The pages of sequence b re-indexed 0..n-1 (what the oracle gets): k pages, v pages, identity page table."""
    n_pages = (L + 15) // 16
    phys = inp["page_table"][b, :n_pages].long()
    return synth.to_u16(inp["k_pages"][phys]), synth.to_u16(inp["v_pages"][phys]), np.arange(n_pages, dtype=np.int32)[None, :]


def _layer(w, inp, ks, cuda):
    return dict(k_pages=inp["k_pages"], v_pages=inp["v_pages"], page_table=inp["page_table"], seq_lens=inp["seq_lens"],
                q_rep=inp["q_rep"], k_per_seq=torch.tensor(ks, dtype=torch.int32, device=cuda),
                q_blk=inp["q_blk"], k_blk=inp["k_blk"], v_blk=inp["v_blk"])


def _check_unit_pools(case, w, inp, b, ks, cap, pool_k, pool_v, pool_len, cuda, agg_mode=0):
    """Selection and pools of every KV head of sequence b against the oracle; returns (oracle pools, #units with in-band swaps)."""
    L, Hkv = w.seq_lens[b], w.n_kv_heads
    kp, vp, ident = _seq_view(inp, b, L, cuda)
    sel_o, sc_o = O.select(synth.to_u16(inp["q_rep"][b:b + 1]), kp, ident, np.array([L]), [ks[b]], Hkv, 128 ** -0.5, agg_mode)
    pk_o, pv_o, pl_o = O.gather(kp, vp, ident, sel_o, cap)
    assert np.array_equal(pool_len[b].cpu().numpy(), pl_o[0]), (case, b)
    pk_g, pv_g = synth.to_u16(pool_k[b]), synth.to_u16(pool_v[b])
    differing = 0
    for h in range(Hkv):
        n = ks[b]
        if np.array_equal(pk_g[h, :n], pk_o[0, h, :n]) and np.array_equal(pv_g[h, :n], pv_o[0, h, :n]):
            continue
        # the index sets differ: only keys inside the tolerance band may (north_star), and the pool must still be a
        # bit-exact gather of SOME ascending index set -- recover it by matching rows
        differing += 1
        rows = O.cached_rows(kp, ident, 0, L, h)
        key = {r.tobytes(): t for t, r in enumerate(rows)}
        got = np.array([key[r.tobytes()] for r in pk_g[h, :n]], dtype=np.int64)
        check_selection(got, n, sc_o[0][h], ks[b], L, f"{case} b{b} h{h}")
        assert np.array_equal(pv_g[h, :n], O.cached_rows(vp, ident, 0, L, h)[got])
    return pl_o, differing


def _check_attn(case, inp, b, s, pool_k, pool_v, pl_o, out_s):
    ref, _ = O.sparse_attn(synth.to_u16(inp["q_blk"][s, b:b + 1]), synth.to_u16(inp["k_blk"][s, b:b + 1]),
                           synth.to_u16(inp["v_blk"][s, b:b + 1]), synth.to_u16(pool_k[b:b + 1]), synth.to_u16(pool_v[b:b + 1]),
                           pl_o, 128 ** -0.5)
    err = np.abs(out_s[b:b + 1].cpu().numpy() - ref).max()
    assert err <= ATTN_TOL, (case, b, s, err)


# ---- C3 select on all 16 units; C4 at the three budgets, 8 sampled units each ------------------------------
SIZE_CASES = {
    # name: (config, sequences whose units the oracle checks, (sequence, attention step) pairs checked)
    "C3_all_units": ("C3", (0, 1, 2, 3), ((2, 0), (0, 14))),
    "C4@2.5": ("C4@2.5", (5,), ((5, 3),)),           # one sequence = 8 KV heads = 8 units
    "C4@10": ("C4@10", (11,), ((11, 0),)),
}


@pytest.mark.parametrize("case", list(SIZE_CASES))
def test_full_size_units_sampled(H, cuda, case):
    name, seqs, attn = SIZE_CASES[case]
    w = synth.config(name)
    inp = synth.make_inputs(w, seed=_seed(name), device=cuda)
    ks = [O.budget_rows(L, w.permille) for L in w.seq_lens]
    cap = max(ks) + w.block_size
    pipe = H.BlockPipeline(_shape(H, w, inp, cap), [_layer(w, inp, ks, cuda)], w.n_attn_steps, 0, cuda)
    pipe.step()                       # block 0 (eager): attention over the empty pool, selection for block 1
    graphs = pipe.capture()           # the configuration bench.py times: one CUDA graph per pool parity
    pipe.replay(graphs)               # block 1: attention over the selected pool
    torch.cuda.synchronize()
    differing, pl_os = 0, {}
    for b in seqs:
        pl_os[b], d = _check_unit_pools(case, w, inp, b, ks, cap, pipe.pools_k[0][1], pipe.pools_v[0][1], pipe.pool_lens[0][1], cuda)
        differing += d
    assert differing <= max(1, len(seqs) * w.n_kv_heads // 8), f"{differing} units with in-band index swaps"
    for b, s in attn:
        _check_attn(case, inp, b, s, pipe.pools_k[0][1], pipe.pools_v[0][1], pl_os[b], pipe.outs[0][s])


# ---- SURVEY 8(c) reading 1: the paper's softmax-sum aggregation at C2 size ------------------------------
def test_mode1_select_at_c2_size(H, cuda):
    w = synth.config("C2")
    inp = synth.make_inputs(w, seed=_seed("C2"), device=cuda)
    ks = [O.budget_rows(L, w.permille) for L in w.seq_lens]
    cap = max(ks) + w.block_size
    shape = _shape(H, w, inp, cap, agg_mode=H.AGG_SOFTMAX_SUM)
    cache = H.make_cache(inp["k_pages"], inp["v_pages"], inp["page_table"], inp["seq_lens"])
    k_per_seq = torch.tensor(ks, dtype=torch.int32, device=cuda)
    sel_idx = torch.full((w.batch, w.n_kv_heads, cap), -7, dtype=torch.int32, device=cuda)
    sel_cnt = torch.full((w.batch, w.n_kv_heads), -7, dtype=torch.int32, device=cuda)
    scores = torch.full((w.batch, w.n_kv_heads, shape.max_seq_len), float("nan"), dtype=torch.float32, device=cuda)
    ws = H.alloc_workspace(H.herald_select_workspace_bytes(shape), cuda)
    H.herald_select(shape, cache, inp["q_rep"], k_per_seq, sel_idx, sel_cnt, scores, ws)
    torch.cuda.synchronize()
    assert (sel_cnt.cpu().numpy() == np.array(ks)[:, None]).all()
    differing = 0
    for b in (1, 6):                  # two sampled sequences = 8 units
        L = w.seq_lens[b]
        kp, _, ident = _seq_view(inp, b, L, cuda)
        _, sc_o = O.select(synth.to_u16(inp["q_rep"][b:b + 1]), kp, ident, np.array([L]), [ks[b]], w.n_kv_heads, 128 ** -0.5, 1)
        for h in range(w.n_kv_heads):
            ref = sc_o[0][h]
            got = scores[b, h, :L].cpu().numpy()
            assert abs(ref.sum() - w.group) < 1e-6                    # G softmaxes, each sums to one
            assert np.abs(got - ref).max() <= 2e-3 * ref.max(), (b, h)
            differing += check_selection(sel_idx[b, h].cpu().numpy(), int(sel_cnt[b, h]), ref, ks[b], L, f"mode1 C2 b{b} h{h}")
            assert (sel_idx[b, h, ks[b]:] == -7).all()
    assert differing <= 2


# ---- C5 -- 16 sampled (layer, b, h) units over the layers of a cut-down stack + full pool equality on 2 layers ----
def test_c5_stack_sampled_layers(H, cuda):
    w = synth.config("C5x4")          # 4 layers of the ragged 28-layer stack (contexts 9574..128375, batch 32)
    inps = [synth.make_inputs(w, seed=_seed("C5", l), device=cuda) for l in range(w.n_layers)]
    ks = [O.budget_rows(L, w.permille) for L in w.seq_lens]
    cap = max(ks) + w.block_size
    pipe = H.BlockPipeline(_shape(H, w, inps[0], cap), [_layer(w, x, ks, cuda) for x in inps], w.n_attn_steps, 0, cuda)
    pipe.step()
    graphs = pipe.capture()
    pipe.replay(graphs)
    torch.cuda.synchronize()
    # one sequence per layer (4 KV heads each): 16 units, selection + pools + one attention step
    order = np.argsort(w.seq_lens)
    picks = [(0, int(order[0]), 2), (1, int(order[-1]), 14), (2, int(order[len(order) // 2]), 7), (3, int(order[3]), 0)]
    differing = 0
    for l, b, s in picks:
        pl_o, d = _check_unit_pools(f"C5 l{l}", w, inps[l], b, ks, cap, pipe.pools_k[l][1], pipe.pools_v[l][1], pipe.pool_lens[l][1], cuda)
        differing += d
        _check_attn(f"C5 l{l}", inps[l], b, s, pipe.pools_k[l][1], pipe.pools_v[l][1], pl_o, pipe.outs[l][s])
    assert differing <= 2
    # full pool equality on two layers: every (sequence, KV head) pool against the oracle's
    for l in (1, 3):
        bad = 0
        for b in range(w.batch):
            _, d = _check_unit_pools(f"C5 pools l{l}", w, inps[l], b, ks, cap, pipe.pools_k[l][1], pipe.pools_v[l][1], pipe.pool_lens[l][1], cuda)
            bad += d
        assert bad <= 4, f"layer {l}: {bad} of {w.batch * w.n_kv_heads} units with in-band index swaps"


# ---- the NEXT rows at the size bench.py times them ----------------------------------------------------------------------
def test_dense_attn_at_c2_size(H, cuda):
    """herald_dense_attn over the whole 8 x 32768 paged cache; the oracle checks one sampled sequence."""
    w = synth.config("C2")
    inp = synth.make_inputs(w, seed=_seed("C2"), device=cuda)
    shape = _shape(H, w, inp, 16)
    cache = H.make_cache(inp["k_pages"], inp["v_pages"], inp["page_table"], inp["seq_lens"])
    out = torch.full((w.batch, w.block_size, w.n_q_heads, 128), float("nan"), dtype=torch.float32, device=cuda)
    lse = torch.empty((w.batch, w.block_size, w.n_q_heads), dtype=torch.float32, device=cuda)
    ws = H.alloc_workspace(H.herald_attn_workspace_bytes(shape), cuda)
    H.herald_dense_attn(shape, cache, inp["q_blk"][3], inp["k_blk"][3], inp["v_blk"][3], out, lse, ws)
    torch.cuda.synchronize()
    assert torch.isfinite(out).all()
    b, L = 4, w.seq_lens[4]
    kp, vp, ident = _seq_view(inp, b, L, cuda)
    sel = [[np.arange(L, dtype=np.int32) for _ in range(w.n_kv_heads)]]
    pk, pv, pl = O.gather(kp, vp, ident, sel, L)
    ref, lse_ref = O.sparse_attn(synth.to_u16(inp["q_blk"][3, b:b + 1]), synth.to_u16(inp["k_blk"][3, b:b + 1]),
                                 synth.to_u16(inp["v_blk"][3, b:b + 1]), pk, pv, pl, 128 ** -0.5)
    assert np.abs(out[b:b + 1].cpu().numpy() - ref).max() <= ATTN_TOL
    assert np.abs(lse[b:b + 1].cpu().numpy() - lse_ref).max() <= 2e-3


def test_sparse_attn_groups_at_c2_size(H, cuda):
    """The 2B-token step over C2-sized pools: two query groups, one launch; the oracle checks one sequence per group."""
    w = synth.config("C2")
    ks = [O.budget_rows(L, w.permille) for L in w.seq_lens]
    cap = max(ks) + w.block_size
    g = torch.Generator(device=cuda)
    g.manual_seed(4711)
    rn = lambda *s: torch.randn(*s, generator=g, device=cuda, dtype=torch.float32).to(torch.bfloat16)
    pk, pv = rn(w.batch, w.n_kv_heads, cap, 128), rn(w.batch, w.n_kv_heads, cap, 128)
    pl = torch.tensor([[k, k - 1, k // 2, k] for k in ks], dtype=torch.int32, device=cuda)
    for b in range(w.batch):
        for h in range(w.n_kv_heads):
            pv[b, h, int(pl[b, h]):] = float("nan")          # rows past pool_len must be ignored
    q, kb, vb = rn(2, w.batch, w.block_size, w.n_q_heads, 128), rn(2, w.batch, w.block_size, w.n_kv_heads, 128), rn(2, w.batch, w.block_size, w.n_kv_heads, 128)
    shape = H.make_shape(w.batch, w.n_q_heads, w.n_kv_heads, w.block_size, 16, 1, cap)
    out = torch.full((2, w.batch, w.block_size, w.n_q_heads, 128), float("nan"), dtype=torch.float32, device=cuda)
    ws = H.alloc_workspace(2 * H.herald_attn_workspace_bytes(shape), cuda)
    H.herald_sparse_attn_groups(shape, 2, pk, pv, pl, q, kb, vb, out, None, ws)
    torch.cuda.synchronize()
    assert torch.isfinite(out).all()
    pv_clean = pv.clone()
    pv_clean[torch.isnan(pv_clean)] = 0
    for grp, b in ((0, 2), (1, 7)):
        ref, _ = O.sparse_attn(synth.to_u16(q[grp, b:b + 1]), synth.to_u16(kb[grp, b:b + 1]), synth.to_u16(vb[grp, b:b + 1]),
                               synth.to_u16(pk[b:b + 1]), synth.to_u16(pv_clean[b:b + 1]), pl[b:b + 1].cpu().numpy(), 128 ** -0.5)
        assert np.abs(out[grp, b:b + 1].cpu().numpy() - ref).max() <= ATTN_TOL, (grp, b)


# ---- PAPER.md:191 / :175: the schedule affects neither the outputs nor the pools ----------------------------------------
@pytest.mark.parametrize("start_after", [0, 2])
def test_pipeline_is_independent_of_stream_delays(H, cuda, start_after):
    """An idle kernel is put on the main stream (right after the fork) and on the retrieval stream in turn: attention
    outputs, pools and pool lengths of two consecutive block steps must be bit-identical to the undelayed run, and the
    idle (NaN-poisoned) pool must not be read by the delayed main stream."""
    w = synth.Workload("delay", 2, (6000, 2500), 28, 4, 32, 5, 50, "planted", 10)
    inp = synth.make_inputs(w, seed=611, device=cuda, spare_pages=1, hostile_tails=True)
    ks = [O.budget_rows(L, w.permille) for L in w.seq_lens]
    cap = max(ks) + w.block_size
    shape = _shape(H, w, inp, cap)

    def run(main_us, retrieval_us):
        pipe = H.BlockPipeline(shape, [_layer(w, inp, ks, cuda)], w.n_attn_steps, start_after, cuda)
        g = torch.Generator(device=cuda)
        g.manual_seed(5)
        pipe.pools_k[0][0].copy_(torch.randn(pipe.pools_k[0][0].shape, generator=g, device=cuda).to(torch.bfloat16))
        pipe.pools_v[0][0].copy_(torch.randn(pipe.pools_v[0][0].shape, generator=g, device=cuda).to(torch.bfloat16))
        pipe.pool_lens[0][0].copy_(torch.tensor([[cap, 10, 0, 77], [1, cap - 1, 64, 65]], dtype=torch.int32, device=cuda))
        pipe.pools_k[0][1].fill_(float("nan"))
        pipe.pools_v[0][1].fill_(float("nan"))
        pipe.pool_lens[0][1].fill_(-1)
        torch.cuda.synchronize()
        H.herald_pipeline_set_debug_delay(main_us, retrieval_us)
        try:
            snaps = []
            for _ in range(2):
                pipe.step()
                torch.cuda.synchronize()
                snaps.append([t.clone() for t in (pipe.outs[0], pipe.pools_k[0][0], pipe.pools_v[0][0], pipe.pools_k[0][1],
                                                  pipe.pools_v[0][1], pipe.pool_lens[0][0], pipe.pool_lens[0][1])])
        finally:
            H.herald_pipeline_set_debug_delay(0, 0)
        return snaps

    base = run(0, 0)
    assert torch.isfinite(base[0][0]).all() and torch.isfinite(base[1][0]).all()
    for main_us, retrieval_us in ((3000, 0), (0, 3000)):
        got = run(main_us, retrieval_us)
        for blk in range(2):
            for a, b in zip(base[blk], got[blk]):
                assert torch.equal(a.view(torch.uint8), b.view(torch.uint8)), (main_us, retrieval_us, blk)


def test_fused_retrieval_chained_in_one_graph(H, cuda):
    """herald_select_rep -> herald_gather -> attention, twice back to back with different representative queries, captured
    in ONE CUDA graph: the second selection reuses the workspace (histogram, score plane) of the first, so everything the
    first enqueued -- its top-k included -- must be complete when the entry's last kernel is (the graph orders the next
    node only behind that one).  Pools of both rounds against the oracle."""
    w = synth.Workload("chain", 2, (9000, 4100), 28, 4, 32, 3, 50, "planted", 12)
    inp = synth.make_inputs(w, seed=808, device=cuda, spare_pages=1, hostile_tails=True)
    ks = [O.budget_rows(L, w.permille) for L in w.seq_lens]
    cap = max(ks) + w.block_size
    shape = _shape(H, w, inp, cap)
    cache = H.make_cache(inp["k_pages"], inp["v_pages"], inp["page_table"], inp["seq_lens"])
    k_per_seq = torch.tensor(ks, dtype=torch.int32, device=cuda)
    g = torch.Generator(device=cuda)
    g.manual_seed(809)
    q_reps = [inp["q_rep"], torch.randn(inp["q_rep"].shape, generator=g, device=cuda).to(torch.bfloat16)]
    sel_idx = torch.zeros((w.batch, w.n_kv_heads, cap), dtype=torch.int32, device=cuda)
    sel_cnt = [torch.zeros((w.batch, w.n_kv_heads), dtype=torch.int32, device=cuda) for _ in range(2)]
    pools_k = [torch.zeros((w.batch, w.n_kv_heads, cap, 128), dtype=torch.bfloat16, device=cuda) for _ in range(2)]
    pools_v = [torch.zeros_like(pools_k[0]) for _ in range(2)]
    rep_out = torch.empty((w.batch, w.n_q_heads, 128), dtype=torch.float32, device=cuda)
    outs = [torch.empty((w.batch, w.block_size, w.n_q_heads, 128), dtype=torch.float32, device=cuda) for _ in range(2)]
    ws = H.alloc_workspace(H.herald_select_rep_workspace_bytes(shape), cuda)
    ws_att = H.alloc_workspace(H.herald_attn_workspace_bytes(shape), cuda)
    st = torch.cuda.Stream()

    def chain():
        for r in range(2):
            H.herald_select_rep(shape, cache, q_reps[r], k_per_seq, sel_idx, sel_cnt[r], None, rep_out, None, ws, st)
            H.herald_gather(shape, cache, sel_idx, sel_cnt[r], pools_k[r], pools_v[r], st)
            H.herald_sparse_attn(shape, pools_k[r], pools_v[r], sel_cnt[r], inp["q_blk"][r], inp["k_blk"][r], inp["v_blk"][r], outs[r], None, ws_att, st)

    with torch.cuda.stream(st):
        chain()                          # eager once: one-time setup
    torch.cuda.synchronize()
    gr = torch.cuda.CUDAGraph()
    with torch.cuda.graph(gr, stream=st, capture_error_mode="thread_local"):
        chain()
    for it in range(5):
        for t in pools_k + pools_v:
            t.zero_()
        torch.cuda.synchronize()
        with torch.cuda.stream(st):
            gr.replay()
        torch.cuda.synchronize()
        for r in range(2):
            for b in range(w.batch):
                L = w.seq_lens[b]
                kp, vp, ident = _seq_view(inp, b, L, cuda)
                sel_o, _ = O.select(synth.to_u16(q_reps[r][b:b + 1]), kp, ident, np.array([L]), [ks[b]], w.n_kv_heads, 128 ** -0.5)
                pk_o, pv_o, pl_o = O.gather(kp, vp, ident, sel_o, cap)
                assert np.array_equal(sel_cnt[r][b].cpu().numpy(), pl_o[0])
                n = ks[b]
                assert np.array_equal(synth.to_u16(pools_k[r][b])[:, :n], pk_o[0][:, :n]), (it, r, b)
                assert np.array_equal(synth.to_u16(pools_v[r][b])[:, :n], pv_o[0][:, :n]), (it, r, b)
                if it == 0:
                    _check_attn("chain", {k: v for k, v in inp.items()}, b, r, pools_k[r], pools_v[r], pl_o, outs[r])


def test_pipeline_tune_keeps_results_and_reports_its_table(H, cuda):
    """herald_pipeline_tune (C ABI): times a handful of schedules with complete block steps, leaves the fastest one set, and
    changes nothing in what the pipeline computes -- the block after the calibration attends over exactly the oracle's pool."""
    w = synth.Workload("tune", 4, (20000, 12345, 8000, 16384), 28, 4, 32, 6, 50, "planted", 16)
    inp = synth.make_inputs(w, seed=4242, device=cuda)
    ks = [O.budget_rows(L, w.permille) for L in w.seq_lens]
    cap = max(ks) + w.block_size
    pipe = H.BlockPipeline(_shape(H, w, inp, cap), [_layer(w, inp, ks, cuda)], w.n_attn_steps, 0, cuda)
    pipe.step()
    table = pipe.tune_schedule(reps=2)
    assert len(table) >= 4
    chosen = f"{pipe.c.scan_ctas}/{pipe.c.start_after_step}/{pipe.c.scan_head_permille}"
    assert chosen in table and table[chosen] == min(table.values())
    assert any(k.split("/")[2] != "0" for k in table), "the head start of the scan was not among the candidates"
    # a head start forced on: the scan runs in two launches, the histogram accumulates over both
    pipe.c.scan_ctas, pipe.c.start_after_step, pipe.c.scan_head_permille = 20, 0, 350
    pipe.step()
    act = pipe.active
    pipe.step()
    torch.cuda.synchronize()
    differing = 0
    for b in range(w.batch):
        pl_o, d = _check_unit_pools("tune", w, inp, b, ks, cap, pipe.pools_k[0][act], pipe.pools_v[0][act], pipe.pool_lens[0][act], cuda)
        differing += d
        _check_attn("tune", inp, b, 1, pipe.pools_k[0][act], pipe.pools_v[0][act], pl_o, pipe.outs[0][1])
    assert differing <= 2
